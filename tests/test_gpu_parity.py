"""GPU-vs-oracle parity of the Sim(3) GN step, through the C ABI (libsim3ba.so).

Bars (BASELINE.json north_star): bit-exact on edge/index bookkeeping and the gathered match set
(per-edge n_valid and checksum); <= 1e-4 relative Frobenius on per-edge blocks, H and g;
<= 1e-3 relative on the pose update tau.  Floors for converged iterations follow DESIGN.md
"Parity protocol": gradients (per edge and assembled) against max(||g||, FLOOR_G ||g_abs||) with
g_abs = sum |J^T| Omega |e| from the oracle and FLOOR_G = 2^-23 / 1e-4 (every term J^T Omega e is
evaluated in fp32, i.e. to ~2^-23 relative; worst case without any averaging), tau against
max(||tau||, 1e-6 sqrt(n)).
"""
import numpy as np
import pytest

from oracle import sim3_gn_oracle as orc
from sim3ba_inputs import CONFIGS, make_config, make_graph
from tests.gpu_common import (TOL_BLOCK, TOL_TAU, blocks35_from_oracle, free_idx, make_solver, oracle_params,
                              rel, set_poses, sym_from_lower)

pytestmark = pytest.mark.gpu

FLOOR_G = 2.0 ** -23 / TOL_BLOCK


def reduced(k):
    """Reduced variants: several 4096-pixel tiles per edge plus a ragged tail."""
    if k == 2:
        return CONFIGS[2].scaled(kf_per_agent=8, height=100, width=130, n_scene=20_000)
    if k == 3:
        return CONFIGS[3].scaled(kf_per_agent=10, height=72, width=100, n_scene=12_000, n_inter=4)
    if k == 4:
        return CONFIGS[4].scaled(kf_per_agent=8, height=48, width=96, n_scene=8_000, n_inter=8)
    if k == 5:
        return CONFIGS[5].scaled(kf_per_agent=60, height=50, width=90, n_scene=9_000, loop_every=20)
    raise KeyError(k)


def check_system(ba, g, poses, prm, tag=""):
    """One lock-step comparison at the given poses; returns (oracle system, oracle solution)."""
    set_poses(ba, poses)
    ba.build_system()
    ba.solve()
    sysm = orc.build_system(poses, g.points, g.conf, g.edges, g.match, prm)
    sol = orc.solve(sysm.H, sysm.g, g.fixed_kf, prm)
    nv, chk, cost_e = (t.cpu().numpy() for t in ba.edge_stats())
    assert np.array_equal(nv.astype(np.int64), sysm.n_valid), tag
    assert np.array_equal(chk.view(np.uint64), sysm.checksum), tag
    blk = ba.edge_blocks().cpu().numpy()
    ref = blocks35_from_oracle(sysm)
    for e in range(g.n_edges):
        if sysm.n_valid[e] == 0:
            assert np.all(blk[e] == 0.0)
            continue
        assert rel(blk[e, :28], ref[e, :28]) <= TOL_BLOCK, (tag, e)
        assert rel(blk[e, 28:], ref[e, 28:], FLOOR_G * np.linalg.norm(sysm.edge_b_abs[e])) <= TOL_BLOCK, (tag, e)
    assert rel(cost_e, sysm.edge_cost) <= TOL_BLOCK, tag
    Hl, gg = (t.cpu().numpy() for t in ba.system())
    fr = free_idx(g)
    Hs = sym_from_lower(Hl)
    assert rel(Hs[np.ix_(fr, fr)], sysm.H[np.ix_(fr, fr)]) <= TOL_BLOCK, tag
    g_floor = FLOOR_G * np.linalg.norm(sysm.g_abs[fr])
    assert rel(gg[fr], sysm.g[fr], g_floor) <= TOL_BLOCK, tag
    # gauge rows/cols: identity block, zero gradient
    for k in g.fixed_kf:
        s = slice(7 * k, 7 * k + 7)
        assert np.array_equal(Hs[s, s], np.eye(7)) and np.all(gg[s] == 0.0)
        Hs_off = Hs[s, :].copy()
        Hs_off[:, s] = 0.0
        assert np.all(Hs_off == 0.0)
    tau, attempts, eps, cost = ba.update()
    tau = tau.cpu().numpy()
    assert attempts == sol.attempts and (eps == sol.eps_used), tag
    tau_floor = 1e-6 * np.sqrt(tau.size)
    assert rel(tau, sol.tau, tau_floor) <= TOL_TAU, tag
    assert rel(np.array([cost]), np.array([sysm.cost])) <= TOL_BLOCK
    for k in g.fixed_kf:
        assert np.all(tau[7 * k:7 * k + 7] == 0.0)
    return sysm, sol


@pytest.mark.parametrize("preset", ["config", "paper"])
def test_config1_full(preset):
    g = make_config(1)
    prm = oracle_params(preset)
    ba = make_solver(g, prm)
    bk = ba.bookkeeping()
    ref = orc.bookkeeping(g.n_kf, g.edges)
    for key in ref:
        assert np.array_equal(bk[key], ref[key]), key
    check_system(ba, g, g.poses_init, prm, f"C1/{preset}")
    ba.close()


@pytest.mark.parametrize("k", [2, 3, 4, 5])
@pytest.mark.parametrize("preset", ["config", "paper"])
def test_reduced_configs_lockstep(k, preset):
    """Lock-step: at every iteration the GPU gets the ORACLE's poses (DESIGN.md parity protocol)."""
    g = make_graph(reduced(k))
    prm = oracle_params(preset)
    ba = make_solver(g, prm)
    bk, ref = ba.bookkeeping(), orc.bookkeeping(g.n_kf, g.edges)
    for key in ref:
        assert np.array_equal(bk[key], ref[key]), key
    poses = g.poses_init.copy()
    for it in range(4):
        sysm, sol = check_system(ba, g, poses, prm, f"C{k}r/{preset}/it{it}")
        poses = orc.retract(poses, sol.tau)
    ba.close()


@pytest.mark.parametrize("k", [1, 2, 3])
def test_free_running_matches_oracle(k):
    """sim3ba_step iterated on its own poses vs the oracle iterated on its own: accumulated update
    Log(T_final T_init^-1) agrees to 1e-3 relative over the whole graph."""
    g = make_config(1) if k == 1 else make_graph(reduced(k))
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    poses = g.poses_init.copy()
    n_it = max(1, min(g.spec.n_iters, 5))
    for _ in range(n_it):
        ba.step()
        poses, _, _ = orc.gn_step(poses, g.points, g.conf, g.edges, g.match, g.fixed_kf, prm)
    out = ba.get_poses().cpu().numpy()
    d_gpu = np.concatenate([orc.pose_delta_log(out[i], g.poses_init[i]) for i in range(g.n_kf)])
    d_orc = np.concatenate([orc.pose_delta_log(poses[i], g.poses_init[i]) for i in range(g.n_kf)])
    assert rel(d_gpu, d_orc) <= TOL_TAU
    assert np.allclose(np.linalg.norm(out[:, 3:7], axis=1), 1.0, atol=1e-14)
    assert np.array_equal(out[0], g.poses_init[0])
    ba.close()


def test_optimize_host_equals_stepping_and_odd_image_size():
    """sim3ba_optimize_host (host buffers in, poses out) runs the very same kernels as create + n x step; the image
    size 37 x 29 has HW % 4 != 0, so the match indices take the non-TMA staging path of kernel 1."""
    import torch
    from paper_2605_30488_b200 import optimize_host
    from tests.gpu_common import gpu_params
    for spec in (reduced(2), CONFIGS[2].scaled(kf_per_agent=6, height=37, width=29, n_scene=3_000)):
        g = make_graph(spec)
        prm = oracle_params("config")
        ba = make_solver(g, prm)
        check_system(ba, g, g.poses_init, prm, tag=f"hw={g.hw}")
        set_poses(ba, g.poses_init)
        costs = []
        for _ in range(3):
            ba.step()
            costs.append(ba.update()[3])
        ref = ba.get_poses().cpu().numpy()
        ba.close()
        h_out = torch.empty((g.n_kf, 8), dtype=torch.float64).pin_memory()
        h_cost = torch.empty((3,), dtype=torch.float64).pin_memory()
        optimize_host(torch.from_numpy(g.points).pin_memory(), torch.from_numpy(g.conf).pin_memory(),
                      torch.from_numpy(g.edges).contiguous(), torch.from_numpy(g.match).pin_memory(), g.fixed_kf,
                      gpu_params(prm), g.spec.height, g.spec.width, torch.from_numpy(g.poses_init.copy()), 3, h_out, h_cost,
                      torch.cuda.current_stream().cuda_stream)
        assert np.array_equal(h_out.numpy(), ref)
        assert np.array_equal(h_cost.numpy(), np.asarray(costs))


def test_step_equals_build_solve_retract_and_is_deterministic():
    g = make_graph(reduced(2))
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    ba.step()
    a = ba.get_poses().cpu().numpy()
    set_poses(ba, g.poses_init)
    ba.build_system()
    ba.solve()
    ba.retract()
    b = ba.get_poses().cpu().numpy()
    assert np.array_equal(a, b)          # same kernels, fixed reduction order: bitwise identical
    set_poses(ba, g.poses_init)
    ba.step()
    assert np.array_equal(a, ba.get_poses().cpu().numpy())
    # retraction alone vs the oracle's Exp-map retraction on the GPU's own tau
    set_poses(ba, g.poses_init)
    ba.build_system()
    ba.solve()
    tau = ba.update()[0].cpu().numpy()
    ref = orc.retract(g.poses_init, tau)
    assert np.allclose(a[:, :3], ref[:, :3], rtol=1e-12, atol=1e-12)
    assert np.allclose(a[:, 7], ref[:, 7], rtol=1e-13)
    sign = np.sign(np.sum(a[:, 3:7] * ref[:, 3:7], axis=1, keepdims=True))
    assert np.allclose(a[:, 3:7], sign * ref[:, 3:7], atol=1e-13)
    ba.close()


def test_solver_decomposition_oracle_system_to_gpu_solver():
    """Oracle (H, g) -> GPU blocked Cholesky: agrees with the oracle's LAPACK solve to ~1e-9."""
    import torch
    g = make_graph(reduced(5))      # 60 keyframes -> n = 420, several 64-blocks plus padding
    prm = oracle_params("config")
    sysm = orc.build_system(g.poses_init, g.points, g.conf, g.edges, g.match, prm)
    sol = orc.solve(sysm.H, sysm.g, g.fixed_kf, prm)
    ba = make_solver(g, prm)
    ba.load_system(torch.from_numpy(sysm.H).cuda(), torch.from_numpy(sysm.g).cuda())
    ba.solve()
    tau, attempts, eps, _ = ba.update()
    assert attempts == 1 and eps == prm.eps0
    assert rel(tau.cpu().numpy(), sol.tau) <= 1e-8
    ba.close()


def test_epsilon_escalation_and_zero_update_on_gpu():
    import torch
    g = make_config(1, height=8, width=8)
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    n = 7 * g.n_kf
    H = np.eye(n)
    H[30, 30] = -5e-3
    gg = np.ones(n)
    ba.load_system(torch.from_numpy(H).cuda(), torch.from_numpy(gg).cuda())
    ba.solve()
    tau, attempts, eps, _ = ba.update()
    ref = orc.solve(H, gg, g.fixed_kf, prm)
    assert attempts == ref.attempts == 3 and np.isclose(eps, 1e-2)
    assert rel(tau.cpu().numpy(), ref.tau) <= 1e-10
    H[30, 30] = -1e6
    ba.load_system(torch.from_numpy(H).cuda(), torch.from_numpy(gg).cuda())
    ba.solve()
    tau, attempts, eps, _ = ba.update()
    assert attempts == 6 and np.isnan(eps) and np.all(tau.cpu().numpy() == 0.0)
    before = ba.get_poses().cpu().numpy()
    ba.retract()
    assert np.array_equal(before, ba.get_poses().cpu().numpy())
    H[30, 30] = np.nan
    ba.load_system(torch.from_numpy(H).cuda(), torch.from_numpy(gg).cuda())
    ba.solve()
    assert ba.update()[1] == 6
    ba.close()


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_solver_modes_agree(k, monkeypatch):
    """a7 three ways -- band + border block Cholesky (mode 2, default), tile-sparse (0), dense tiles (1) -- on the same
    built system: same attempts / eps, tau within 1e-6 of each other (different elimination orders on cond ~ 1e8
    systems) and each within the north_star 1e-3 of the oracle.  Mode 2 also with short segments (separators)."""
    g = make_config(1) if k == 1 else make_graph(reduced(k))
    prm = oracle_params("config")
    sysm = orc.build_system(g.poses_init, g.points, g.conf, g.edges, g.match, prm)
    sol = orc.solve(sysm.H, sysm.g, g.fixed_kf, prm)
    tau_floor = 1e-6 * np.sqrt(sol.tau.size)
    taus = {}
    for tag, mode, lmax in (("bb", 2, None), ("bb-short", 2, "5"), ("tile", 0, None), ("dense", 1, None)):
        if lmax is None:
            monkeypatch.delenv("SIM3BA_BB_LMAX", raising=False)
        else:
            monkeypatch.setenv("SIM3BA_BB_LMAX", lmax)
        ba = make_solver(g, prm)
        info = ba.bb_info()
        assert info["valid"] == 1 and info["n_interior"] + info["n_border"] == g.n_kf - len(g.fixed_kf)
        if lmax is not None:
            assert info["max_segment"] <= 5
        ba.set_solver_mode(mode)
        set_poses(ba, g.poses_init)
        ba.build_system()
        ba.solve()
        tau, attempts, eps, _ = ba.update()
        taus[tag] = tau.cpu().numpy()
        assert attempts == sol.attempts and eps == sol.eps_used, tag
        assert rel(taus[tag], sol.tau, tau_floor) <= TOL_TAU, tag
        for kf in g.fixed_kf:
            assert np.all(taus[tag][7 * kf:7 * kf + 7] == 0.0)
        ba.close()
    for tag in ("bb-short", "tile", "dense"):
        assert rel(taus[tag], taus["bb"], tau_floor) <= 1e-6, tag


def test_band_border_zero_information_keyframe_and_all_attempts_fail():
    """A keyframe none of whose edges has a valid match has a zero diagonal block: with eps0 > 0 its update is 0 and the
    rest matches the oracle; with eps0 = 0 every attempt meets a zero pivot -> tau = 0, attempts = max."""
    g = make_config(1, height=40, width=60)
    lone = 3
    for e in range(g.n_edges):
        if lone in g.edges[e]:
            g.match[e, :] = -1
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    assert ba.bb_info()["valid"] == 1
    sysm, sol = check_system(ba, g, g.poses_init, prm, "lone keyframe")
    tau = ba.update()[0].cpu().numpy()
    assert np.all(tau[7 * lone:7 * lone + 7] == 0.0)
    ba.close()
    prm0 = oracle_params("config", eps0=0.0)
    ba = make_solver(g, prm0)
    set_poses(ba, g.poses_init)
    ba.build_system()
    ba.solve()
    tau, attempts, eps, _ = ba.update()
    ref = orc.solve(sysm.H, sysm.g, g.fixed_kf, prm0)
    assert attempts == ref.attempts == prm0.max_attempts and np.isnan(eps)
    assert np.all(tau.cpu().numpy() == 0.0) and np.all(ref.tau == 0.0)
    before = ba.get_poses().cpu().numpy()
    ba.step()
    assert np.array_equal(before, ba.get_poses().cpu().numpy())
    ba.close()


def test_edge_cases_validity_confmin_multiple_gauges():
    g = make_config(1, height=40, width=60)
    g.match[3, :] = -1                       # an edge without any valid match
    g.match[4, ::7] = g.hw + 5               # out-of-range targets are "no match"
    g.conf[2, ::5] = 0.0                     # zero-confidence pixels
    prm = oracle_params("config", conf_min=0.3)
    ba = make_solver(g, prm, fixed=[0, 5])
    g.fixed_kf = np.array([0, 5], dtype=np.int32)
    check_system(ba, g, g.poses_init, prm, "edge-cases")
    ba.close()


def test_create_rejects_bad_arguments():
    import torch
    from paper_2605_30488_b200 import Sim3BA, Sim3BAError, make_params
    g = make_config(1, height=8, width=8)
    dev = torch.device("cuda:0")
    pts, cf, mt = (torch.from_numpy(x).to(dev) for x in (g.points, g.conf, g.match))
    bad = g.edges.copy()
    bad[2] = (3, 3)
    with pytest.raises(Sim3BAError):
        Sim3BA(pts, cf, torch.from_numpy(bad).to(dev), mt, [0], make_params(), 8, 8)
    bad[2] = (3, 99)
    with pytest.raises(Sim3BAError):
        Sim3BA(pts, cf, torch.from_numpy(bad).to(dev), mt, [0], make_params(), 8, 8)
    with pytest.raises(Sim3BAError):
        Sim3BA(pts, cf, torch.from_numpy(g.edges).to(dev), mt, [42], make_params(), 8, 8)
    with pytest.raises(Sim3BAError):
        Sim3BA(pts, cf, torch.from_numpy(g.edges).to(dev), mt, [0], make_params(sigma_ray=0.0), 8, 8)
    ba = Sim3BA(pts, cf, torch.from_numpy(g.edges).to(dev), mt, [0], make_params(), 8, 8)
    with pytest.raises(Sim3BAError):
        ba.solve()                           # BAD_STATE: no system built yet
    ba.close()


def test_config2_full_size_sampled_edges():
    """BASELINE configs[1] at full size (the bench workload): every edge's match set bit-exact,
    a sample of per-edge blocks against the oracle, and H, g, tau from the oracle run on all edges."""
    g = make_config(2)
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    check_system(ba, g, g.poses_init, prm, "C2-full")
    ba.close()


def test_config4_full_size_sampled_edges_and_solver_property():
    """BASELINE configs[3] at full size (1000 keyframes, 3036 edges, 7000 x 7000 system, the launch configuration bench.py
    times): the match set of EVERY edge bit-exact against the validity rule written out in NumPy, the 7x7 blocks of a sample of
    edges (first, last, every inter-agent tenth, a stride through the chains) against the oracle, and the update tau against
    SciPy's dense Cholesky of the system assembled in NumPy from the GPU's own per-edge blocks (decomposition: a1-a5 vs the
    oracle on samples, a6-a7 vs a library solve on the whole system)."""
    import scipy.linalg
    g = make_config(4)
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    ba.build_system()
    ba.solve()
    nv, chk, _ = (t.cpu().numpy() for t in ba.edge_stats())
    blk = ba.edge_blocks().cpu().numpy()
    tau, attempts, eps, _ = ba.update()
    tau = tau.cpu().numpy()
    HW = g.hw
    for e in range(g.n_edges):                                 # R12, typed out: 0 <= n < HW, c_i[m] > c_min, c_j[n] > c_min
        i, j = g.edges[e]
        n = g.match[e].astype(np.int64)
        m = np.flatnonzero((n >= 0) & (n < HW))
        m = m[(g.conf[i, m] > prm.conf_min) & (g.conf[j, n[m]] > prm.conf_min)]
        assert nv[e] == m.size, e
        with np.errstate(over="ignore"):
            ref = np.sum(m.astype(np.uint64) * np.uint64(HW) + n[m].astype(np.uint64), dtype=np.uint64)
        assert chk.view(np.uint64)[e] == ref, e
    inter = np.flatnonzero(g.edge_kind == 2)
    sample = sorted(set([0, g.n_edges - 1] + list(inter[::10]) + list(range(5, g.n_edges, 211))))
    sysm = orc.build_system(g.poses_init, g.points, g.conf, g.edges, g.match, prm, edge_subset=sample)
    ref = blocks35_from_oracle(sysm)
    for e in sample:
        assert rel(blk[e, :28], ref[e, :28]) <= TOL_BLOCK, e
        assert rel(blk[e, 28:], ref[e, 28:], FLOOR_G * np.linalg.norm(sysm.edge_b_abs[e])) <= TOL_BLOCK, e
    # a6 + a7 on the whole system: assemble H, g from the GPU's blocks (two diagonal, one off-diagonal block per edge,
    # PAPER.md:118), delete the gauge rows, eps_0 on the diagonal (Eq. (7)), library Cholesky
    n = 7 * g.n_kf
    H, gg = np.zeros((n, n)), np.zeros(n)
    iu = np.triu_indices(7)
    for e in range(g.n_edges):
        i, j = (int(v) for v in g.edges[e])
        A = np.zeros((7, 7))
        A[iu] = blk[e, :28]
        A = A + A.T - np.diag(np.diag(A))
        si, sj = slice(7 * i, 7 * i + 7), slice(7 * j, 7 * j + 7)
        H[si, si] += A
        H[sj, sj] += A
        H[si, sj] -= A
        H[sj, si] -= A
        gg[sj] += blk[e, 28:]
        gg[si] -= blk[e, 28:]
    fr = free_idx(g)
    Hf = H[np.ix_(fr, fr)] + prm.eps0 * np.eye(fr.size)
    ref_tau = np.zeros(n)
    ref_tau[fr] = -scipy.linalg.cho_solve(scipy.linalg.cho_factor(Hf, lower=True), gg[fr])
    assert attempts == 1 and eps == prm.eps0
    assert rel(tau, ref_tau) <= 1e-6
    assert ba.bb_info()["valid"] == 1
    ba.close()
