"""GPU-vs-oracle parity of the Sim(3) GN step, through the C ABI (libsim3ba.so).

Bars (BASELINE.json north_star): bit-exact on edge/index bookkeeping and the gathered match set
(per-edge n_valid and checksum); <= 1e-4 relative Frobenius on per-edge blocks, H and g;
<= 1e-3 relative on the pose update tau.  Floors for converged iterations follow DESIGN.md
"Parity protocol": gradients (per edge and assembled) against
max(||g||, FLOOR_G ||g_abs||) with g_abs = sum |J^T| Omega |e| from the oracle and FLOOR_G = 1e-6, tau against
max(||tau||, 1e-6 sqrt(n)).  Every check_system call appends its measured errors, ||g|| / ||g_abs|| and whether a floor
was the active bound to $SIM3BA_PARITY_LOG (the table in DESIGN.md).
"""
import numpy as np
import pytest

from oracle import sim3_gn_oracle as orc
from oracle.edge_pool import build_system_parallel
from sim3ba_inputs import CONFIG_PARAMS, CONFIGS, make_config, make_graph
from tests.gpu_common import (TOL_BLOCK, TOL_TAU, blocks35_from_oracle, free_idx, make_solver, oracle_params,
                              parity_log, rel, set_poses, start_poses, sym_from_lower)

pytestmark = pytest.mark.gpu

FLOOR_G = 1e-6


def reduced(k):
    """Reduced variants: several 512-pixel slices per edge plus a ragged tail."""
    if k == 2:
        return CONFIGS[2].scaled(kf_per_agent=8, height=100, width=130, n_scene=20_000)
    if k == 3:
        return CONFIGS[3].scaled(kf_per_agent=10, height=72, width=100, n_scene=12_000, n_inter=4)
    if k == 4:
        return CONFIGS[4].scaled(kf_per_agent=8, height=48, width=96, n_scene=8_000, n_inter=8)
    if k == 5:
        return CONFIGS[5].scaled(kf_per_agent=60, height=50, width=90, n_scene=9_000, loop_every=20)
    raise KeyError(k)


def check_system(ba, g, poses, prm, tag="", pool=False):  # noqa: C901
    """One lock-step comparison at the given poses; returns (oracle system, oracle solution).  ``pool``: the unchanged
    oracle runs edge-parallel on every host core (oracle/edge_pool.py) -- the full-size configs."""
    set_poses(ba, poses)
    ba.build_system()
    ba.solve()
    if pool:
        sysm = build_system_parallel(poses, g.points, g.conf, g.edges, g.match, prm)
    else:
        sysm = orc.build_system(poses, g.points, g.conf, g.edges, g.match, prm)
    sol = orc.solve(sysm.H, sysm.g, g.fixed_kf, prm)
    nv, chk, cost_e = (t.cpu().numpy() for t in ba.edge_stats())
    assert np.array_equal(nv.astype(np.int64), sysm.n_valid), tag
    assert np.array_equal(chk.view(np.uint64), sysm.checksum), tag
    blk = ba.edge_blocks().cpu().numpy()
    ref = blocks35_from_oracle(sysm)
    err_A, err_b = 0.0, 0.0
    for e in range(g.n_edges):
        if sysm.n_valid[e] == 0:
            assert np.all(blk[e] == 0.0)
            continue
        err_A = max(err_A, rel(blk[e, :28], ref[e, :28]))
        err_b = max(err_b, rel(blk[e, 28:], ref[e, 28:], FLOOR_G * np.linalg.norm(sysm.edge_b_abs[e])))
        assert rel(blk[e, :28], ref[e, :28]) <= TOL_BLOCK, (tag, e)
        assert rel(blk[e, 28:], ref[e, 28:], FLOOR_G * np.linalg.norm(sysm.edge_b_abs[e])) <= TOL_BLOCK, (tag, e)
    assert rel(cost_e, sysm.edge_cost) <= TOL_BLOCK, tag
    Hl, gg = (t.cpu().numpy() for t in ba.system())
    fr = free_idx(g)
    Hs = sym_from_lower(Hl)
    del Hl
    err_H = rel(Hs[np.ix_(fr, fr)], sysm.H[np.ix_(fr, fr)])
    g_norm, g_abs_norm = np.linalg.norm(sysm.g[fr]), np.linalg.norm(sysm.g_abs[fr])
    g_floor = FLOOR_G * g_abs_norm
    err_g = rel(gg[fr], sysm.g[fr], g_floor)
    tau, attempts, eps, cost = ba.update()
    tau = tau.cpu().numpy()
    tau_floor = 1e-6 * np.sqrt(tau.size)
    err_tau = rel(tau, sol.tau, tau_floor)
    parity_log(tag=tag, n_kf=g.n_kf, n_edges=g.n_edges, hw=g.hw, n_valid=int(sysm.n_valid.sum()), err_edge_A_max=err_A,
               err_edge_b_max=err_b, err_H=err_H, err_g=err_g, err_tau=err_tau, g_over_g_abs=g_norm / max(g_abs_norm, 1e-300),
               g_err_over_g_abs=float(np.linalg.norm(gg[fr] - sysm.g[fr]) / max(g_abs_norm, 1e-300)),
               g_floor_active=bool(g_norm < g_floor), tau_norm=float(np.linalg.norm(sol.tau)),
               tau_floor_active=bool(np.linalg.norm(sol.tau) < tau_floor), attempts=int(attempts))
    assert err_H <= TOL_BLOCK, tag
    assert err_g <= TOL_BLOCK, tag
    # gauge rows/cols: identity block, zero gradient
    for k in g.fixed_kf:
        s = slice(7 * k, 7 * k + 7)
        assert np.array_equal(Hs[s, s], np.eye(7)) and np.all(gg[s] == 0.0)
        Hs_off = Hs[s, :].copy()
        Hs_off[:, s] = 0.0
        assert np.all(Hs_off == 0.0)
    assert attempts == sol.attempts and (eps == sol.eps_used), tag
    assert err_tau <= TOL_TAU, tag
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
    poses = start_poses(g, prm)
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
    p0 = start_poses(g, prm)
    set_poses(ba, p0)
    poses = p0.copy()
    n_it = max(1, min(g.spec.n_iters, 5))
    for _ in range(n_it):
        ba.step()
        poses, _, _ = orc.gn_step(poses, g.points, g.conf, g.edges, g.match, g.fixed_kf, prm)
    out = ba.get_poses().cpu().numpy()
    d_gpu = np.concatenate([orc.pose_delta_log(out[i], p0[i]) for i in range(g.n_kf)])
    d_orc = np.concatenate([orc.pose_delta_log(poses[i], p0[i]) for i in range(g.n_kf)])
    assert rel(d_gpu, d_orc) <= TOL_TAU
    assert np.allclose(np.linalg.norm(out[:, 3:7], axis=1), 1.0, atol=1e-14)
    assert np.array_equal(out[0], p0[0])
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
    p0 = start_poses(g, prm)
    sysm = orc.build_system(p0, g.points, g.conf, g.edges, g.match, prm)
    sol = orc.solve(sysm.H, sysm.g, g.fixed_kf, prm)
    tau_floor = 1e-6 * np.sqrt(sol.tau.size)
    taus = {}
    for tag, mode, lmax, max_ctas in (("bb", 2, None, None), ("bb-short", 2, "5", None), ("tile", 0, None, None), ("dense", 1, None, None),
                                      ("bb-short-2ctas", 2, "5", "2"), ("tile-1cta", 0, None, "1"), ("dense-2ctas", 1, None, "2"),
                                      ("bb-1level", 2, None, None), ("bb-short-1level", 2, "5", None),
                                      ("bb-2level", 2, None, None), ("bb-short-2level", 2, "5", None), ("bb-short-2level-2ctas", 2, "5", "2")):
        if tag.endswith("1level"):                        # without the second level of the plan (separator groups out of S)
            monkeypatch.setenv("SIM3BA_BB_LEVELS", "1")
        elif "2level" in tag:                             # ... and with it wherever a group can be eliminated (by default: where it pays)
            monkeypatch.setenv("SIM3BA_BB_LEVELS", "2")
        else:
            monkeypatch.delenv("SIM3BA_BB_LEVELS", raising=False)
        if lmax is None:
            monkeypatch.delenv("SIM3BA_BB_LMAX", raising=False)
        else:
            monkeypatch.setenv("SIM3BA_BB_LMAX", lmax)
        if max_ctas is None:                              # a capped grid: several segments, tiles and update tasks per CTA
            monkeypatch.delenv("SIM3BA_SOLVE_MAX_CTAS", raising=False)
        else:
            monkeypatch.setenv("SIM3BA_SOLVE_MAX_CTAS", max_ctas)
        ba = make_solver(g, prm)
        info = ba.bb_info()
        assert info["valid"] == 1 and info["n_interior"] + info["n_border"] == g.n_kf - len(g.fixed_kf)
        if lmax is not None:
            assert info["max_segment"] <= 5
        if tag.endswith("1level"):
            assert info["n_groups_level2"] == 0 and info["n_border_dense"] == info["n_border"]
        elif "2level" in tag and k >= 4 + (lmax is None):  # reduced C4 / C5 with short segments, reduced C5 as it is: groups to eliminate
            assert info["n_groups_level2"] > 0 and info["n_border_dense"] < info["n_border"]
        ba.set_solver_mode(mode)
        set_poses(ba, p0)
        ba.build_system()
        ba.solve()
        tau, attempts, eps, _ = ba.update()
        taus[tag] = tau.cpu().numpy()
        assert attempts == sol.attempts and eps == sol.eps_used, tag
        assert rel(taus[tag], sol.tau, tau_floor) <= TOL_TAU, tag
        for kf in g.fixed_kf:
            assert np.all(taus[tag][7 * kf:7 * kf + 7] == 0.0)
        ba.close()
    for tag in taus:
        assert rel(taus[tag], taus["bb"], tau_floor) <= 1e-6, tag
    for tag, same in (("bb-short-2ctas", "bb-short"), ("tile-1cta", "tile"), ("dense-2ctas", "dense"), ("bb-short-2level-2ctas", "bb-short-2level")):
        assert np.array_equal(taus[tag], taus[same]), tag          # the grid size does not change the order of any sum


def test_band_border_plan_on_a_very_long_chain():
    """12000 keyframes in one chain (tiny images): at the default segment length the cuts would put more than 292 keyframes on
    the border; the plan then takes longer segments instead of giving up on the band + border solve, further levels take the
    separator groups out again, and Gauss-Newton steps on it run in one attempt with a falling cost."""
    spec = CONFIGS[5].scaled(name="chain12000", kf_per_agent=12000, height=6, width=8, n_scene=4_000, loop_every=0, p_out=0.05)
    g = make_graph(spec)
    prm = oracle_params("config", lm_lambda=1e-3)
    ba = make_solver(g, prm)
    info = ba.bb_info()
    assert info["valid"] == 1 and 7 * info["n_border"] <= 2048
    assert info["max_segment"] > int(0.9 * np.sqrt(g.n_kf - 1) + 0.5)            # the segments were lengthened
    assert info["n_groups_level2"] > 0 and info["n_border_dense"] < info["n_border"]
    set_poses(ba, g.poses_init)
    costs = []
    for _ in range(3):
        ba.build_system()
        ba.solve()
        tau, attempts, _, cost = ba.update()
        assert attempts == 1 and bool(np.isfinite(tau.cpu().numpy()).all())
        costs.append(cost)
        ba.retract()
    assert costs[2] < costs[1] < costs[0], costs
    ba.close()


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


@pytest.mark.parametrize("seed", range(48))
def test_random_topologies_lockstep(seed):
    """Arbitrary connected topologies instead of the configs' chains: 2..12 (a dozen seeds: 30..60) keyframes of 30x20 pixels (one full 512-pixel
    slice and a ragged one), a random spanning tree plus random extra edges with duplicate and reversed pairs, every third
    seed with a hub keyframe that half of the extra edges leave (many edges share one staged X_i slice), one or two gauge
    keyframes anywhere, both presets, with and without the Eq. (7) damping, all three solver plans (the band + border plan
    is valid for some of these graphs only; the library falls back to the tile plan by itself)."""
    rng = np.random.default_rng(1000 + seed)
    n_kf = int(rng.integers(2, 13)) if seed < 36 else int(rng.integers(30, 61))      # the last dozen: several 64-row tile columns
    spec = CONFIGS[1].scaled(name=f"fuzz{seed}", seed=100 + seed, n_agents=1, kf_per_agent=n_kf, height=20, width=30, n_inter=0)
    order = rng.permutation(n_kf)
    edges = [(int(order[k]), int(order[rng.integers(0, k)])) for k in range(1, n_kf)]            # spanning tree
    hub = int(rng.integers(0, n_kf)) if seed % 3 == 0 else -1
    for _ in range(int(rng.integers(0, 2 * n_kf))):
        i = hub if (hub >= 0 and rng.random() < 0.5) else int(rng.integers(0, n_kf))
        j = int(rng.integers(0, n_kf - 1))
        j += j >= i
        edges.append((i, j))
    if len(edges) > 1:
        edges.append(edges[0])                               # the same pair twice
        edges.append((edges[1][1], edges[1][0]))             # and one pair in both directions
    edges = [edges[k] for k in rng.permutation(len(edges))]
    g = make_graph(spec, edges=np.asarray(edges, dtype=np.int32), valid_frac=float(rng.uniform(0.3, 0.95)))
    fixed = sorted(set(int(k) for k in rng.choice(n_kf, size=min(n_kf - 1, int(rng.integers(1, 3))), replace=False)))
    g.fixed_kf = np.asarray(fixed, dtype=np.int32)
    prm = oracle_params(["config", "paper"][seed % 2], lm_lambda=[0.0, 1e-3][(seed // 2) % 2])
    ba = make_solver(g, prm)
    bk, ref = ba.bookkeeping(), orc.bookkeeping(g.n_kf, g.edges)
    for key in ref:
        assert np.array_equal(bk[key], ref[key]), key
    ba.set_solver_mode([2, 0, 1][seed % 3])
    poses = g.poses_init
    for it in range(2):
        _, sol = check_system(ba, g, poses, prm, f"fuzz{seed}/it{it}")
        poses = orc.retract(poses, sol.tau)
    ba.close()


def test_matches_mapped_next_to_the_camera_centre():
    """Matches whose transformed point x = T_ij X_j lands within |X_i| / 32 ... |X_i| / 1e5 of camera i's centre: X_i + delta
    cancels there and the 1 / |x|^2 terms of the Jacobian make such a match dominate its edge's block.  The device defers them
    to an FP64 evaluation (k_deferred); the blocks must still meet the 1e-4 bar -- and the match set stays bit-exact."""
    g = make_config(1, height=40, width=60)
    prm = oracle_params("paper")
    rng = np.random.default_rng(5)
    for e in range(0, g.n_edges, 2):
        i, j = (int(v) for v in g.edges[e])
        Ti, Tj = orc.pose_to_srt(g.poses_init[i]), orc.pose_to_srt(g.poses_init[j])
        s, R, t = orc.sim3_mul(orc.sim3_inv(*Ti), Tj)                       # T_ij at the start poses
        ms = rng.choice(np.flatnonzero(g.match[e] >= 0), size=12, replace=False)
        for q, m in enumerate(ms):
            n = int(g.match[e, m])
            scale = np.linalg.norm(g.points[i, m]) * 10.0 ** (-1.6 - 0.3 * q)   # |x| = |X_i| / 40 ... / 8e4
            x = scale * rng.normal(size=3) / np.sqrt(3.0)
            g.points[j, n] = (R.T @ (x - t) / s).astype(np.float32)             # X_j = T_ij^-1 x
    ba = make_solver(g, prm)
    check_system(ba, g, g.poses_init, prm, "near-centre/paper")
    # the same graph twice: the deferred path is part of the fixed reduction order
    blk_a = ba.edge_blocks().cpu().numpy()
    set_poses(ba, g.poses_init)
    ba.build_system()
    assert np.array_equal(blk_a, ba.edge_blocks().cpu().numpy())
    ba.close()


def test_empty_graphs():
    """No edges at all (every keyframe is then held only by eps_r: tau = 0, the poses do not move) and a graph that consists
    of the gauge keyframe alone."""
    import torch
    from paper_2605_30488_b200 import Sim3BA
    from tests.gpu_common import gpu_params
    g = make_config(1, height=8, width=8)
    prm = oracle_params("config")
    dev = torch.device("cuda:0")
    empty_e = torch.zeros((0, 2), dtype=torch.int32, device=dev)
    empty_m = torch.zeros((0, g.hw), dtype=torch.int32, device=dev)
    for n_kf in (g.n_kf, 1):
        pts, cf = torch.from_numpy(g.points[:n_kf]).to(dev), torch.from_numpy(g.conf[:n_kf]).to(dev)
        ba = Sim3BA(pts, cf, empty_e, empty_m, [0], gpu_params(prm), 8, 8)
        p0 = torch.from_numpy(g.poses_init[:n_kf].copy()).to(dev)
        ba.set_poses(p0)
        ba.build_system()
        ba.solve()
        tau, attempts, eps, cost = ba.update()
        ref = orc.solve(np.zeros((7 * n_kf, 7 * n_kf)), np.zeros(7 * n_kf), [0], prm)
        assert attempts == ref.attempts == 1 and eps == prm.eps0 and cost == 0.0
        assert np.all(tau.cpu().numpy() == 0.0) and np.all(ref.tau == 0.0)
        ba.set_poses(p0)
        ba.step()
        assert np.array_equal(ba.get_poses().cpu().numpy(), g.poses_init[:n_kf])
        assert ba.edge_stats()[0].numel() == 0
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


def test_config2_full_size_all_edges():
    """BASELINE configs[1] at full size: every edge's match set bit-exact, every per-edge block, H, g and tau against the
    oracle run on all edges."""
    g = make_config(2)
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    check_system(ba, g, g.poses_init, prm, "C2-full/config/it0", pool=True)
    ba.close()


@pytest.mark.parametrize("k,preset", [(3, "config"), (3, "paper"), (4, "config"), (4, "paper"), (5, "config"), (5, "bench")])
def test_full_size_vs_oracle(k, preset):
    """BASELINE configs[2..4] at FULL size, in the launch configuration bench.py times (C3: 200 keyframes 512x384, 608
    edges; C4: 1000 keyframes 256x192, 3036 edges, n = 7000; C5: 2000 keyframes 512x384, 6003 edges, 1.18e9 candidate
    matches, n = 14000), iteration 0 from the seeded start: every edge's n_valid / checksum bit-exact, ALL per-edge blocks,
    the assembled H and g on the free blocks (<= 1e-4) and tau against orc.solve of the ORACLE's own H, g (<= 1e-3; this
    is where cond(H) ~ 1e8-1e10 amplifies the fp32 per-match arithmetic).  The unchanged NumPy
    oracle runs edge-parallel on the host cores (oracle/edge_pool.py).  C3 starts from the independent per-agent gauges
    brought together by the oracle's gauge synchronisation; the device's own sim3ba_gauge_sync on the same
    raw start must land on the same poses.  (5, "bench"): config 5 with the parameters bench.py runs it with
    (sim3ba_inputs.config_params: the Eq. (7) damping lambda = 1e-4), followed by the five iterations of the config on the
    device: one factorisation attempt each and a cost that falls every iteration -- undamped, this chain leaves the basin."""
    g = make_config(k)
    prm = oracle_params("config", **CONFIG_PARAMS.get(k, {})) if preset == "bench" else oracle_params(preset)
    ba = make_solver(g, prm)
    bk, ref = ba.bookkeeping(), orc.bookkeeping(g.n_kf, g.edges)
    for key in ref:
        assert np.array_equal(bk[key], ref[key]), key
    p0 = start_poses(g, prm)
    if g.meta.get("gauge_sync_plan"):
        set_poses(ba, g.poses_init)
        for e, moving, moving_is_i in g.meta["gauge_sync_plan"]:
            ba.gauge_sync(e, moving, moving_is_i)
        dev = ba.get_poses().cpu().numpy()
        sgn = np.sign(np.sum(dev[:, 3:7] * p0[:, 3:7], axis=1, keepdims=True))
        assert np.allclose(dev[:, :3], p0[:, :3], rtol=0, atol=1e-9 * max(1.0, np.abs(p0[:, :3]).max()))
        assert np.allclose(dev[:, 3:7], sgn * p0[:, 3:7], rtol=0, atol=1e-9) and np.allclose(dev[:, 7], p0[:, 7], rtol=1e-9)
    check_system(ba, g, p0, prm, f"C{k}-full/{preset}/it0", pool=True)
    assert ba.bb_info()["valid"] == 1
    if preset == "bench":
        set_poses(ba, p0)
        costs = []
        for _ in range(g.spec.n_iters):
            ba.build_system()
            ba.solve()
            _, attempts, _, cost = ba.update()
            assert attempts == 1
            costs.append(cost)
            ba.retract()
        assert all(b < a for a, b in zip(costs, costs[1:])), costs
    ba.close()
