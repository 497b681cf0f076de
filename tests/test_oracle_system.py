"""Pins of the oracle's normal-equation assembly, solve (Eq. (7))
and iteration against things other than itself: a brute-force finite-difference
Gauss-Newton matrix built with scipy.linalg.expm, numpy.linalg.lstsq for kappa -> inf, structural
invariants, numpy.linalg.solve, forced epsilon escalation, and convergence to ground truth."""
import numpy as np
import pytest
import scipy.linalg

from oracle import sim3_gn_oracle as orc
from sim3ba_inputs import CONFIGS, make_graph
from tests.test_oracle_lie import gen4
from tests.test_oracle_residual_jacobian import _srt_from_4x4


def tiny_clean_graph(seed=0, n_kf=4, n_pts=12, noise=0.0, fp32=False):
    """All keyframes see the same n_pts scene points in the same pixel order (match = identity)."""
    rng = np.random.default_rng(seed)
    scene = rng.normal(0, 3, (n_pts, 3)) + np.array([0, 0, 8.0])
    poses = np.empty((n_kf, 8))
    X = np.empty((n_kf, n_pts, 3))
    for k in range(n_kf):
        q = rng.normal(size=4) * 0.2 + np.array([0, 0, 0, 1.0])
        q /= np.linalg.norm(q)
        poses[k] = np.concatenate([rng.normal(0, 0.5, 3), q, [np.exp(rng.normal(0, 0.2))]])
        s, R, t = orc.pose_to_srt(poses[k])
        X[k] = (scene - t) @ R / s + rng.normal(0, noise, (n_pts, 3)) if noise else (scene - t) @ R / s
    conf = rng.beta(5, 2, (n_kf, n_pts))
    edges = np.array([(a, b) for a in range(n_kf) for b in range(n_kf) if a != b and (b - a) % n_kf in (1, 2)],
                     dtype=np.int32)
    match = np.tile(np.arange(n_pts, dtype=np.int32), (edges.shape[0], 1))
    if fp32:
        X, conf = X.astype(np.float32), conf.astype(np.float32)
    return poses, X, conf, edges, match


def perturbed(poses, rng, mag=0.05):
    out = poses.copy()
    for k in range(1, poses.shape[0]):
        T4 = scipy.linalg.expm(gen4(rng.normal(0, mag, 7))) @ orc.sim3_matrix(*orc.pose_to_srt(poses[k]))
        out[k] = orc.srt_to_pose(*_srt_from_4x4(T4))
    return out


def brute_force_system(poses, X, conf, edges, match, prm, h=1e-6):
    """Pure-Python loops: for every match, the whitened residual as a function of all 7N tangent
    coordinates is differenced numerically (perturbations through expm), and J^T W J / J^T W e are
    summed term by term.  Shares only the residual definition (hand-pinned) with the oracle."""
    N = poses.shape[0]
    T4 = [orc.sim3_matrix(*orc.pose_to_srt(p)) for p in poses]
    H = np.zeros((7 * N, 7 * N))
    g = np.zeros(7 * N)
    sig = np.array([prm.sigma_ray] * 3 + [prm.sigma_dist])
    for e in range(edges.shape[0]):
        i, j = int(edges[e, 0]), int(edges[e, 1])
        for m in range(match.shape[1]):
            n = int(match[e, m])
            if n < 0 or n >= match.shape[1] or not (conf[i, m] > prm.conf_min and conf[j, n] > prm.conf_min):
                continue
            xi = np.asarray(X[i, m], float)[None]
            xj = np.asarray(X[j, n], float)[None]

            def res(di, dj):
                Ti = scipy.linalg.expm(gen4(di)) @ T4[i]
                Tj = scipy.linalg.expm(gen4(dj)) @ T4[j]
                return orc.residual(_srt_from_4x4(np.linalg.inv(Ti) @ Tj), xi, xj)[0]

            z = np.zeros(7)
            e0 = res(z, z)
            q = np.sqrt(float(conf[i, m]) * float(conf[j, n]))
            r = np.sqrt(q) * e0 / sig
            w = np.array([1.0 if abs(rc) <= prm.huber_k else prm.huber_k / abs(rc) for rc in r])
            om = q * w / sig ** 2
            J = np.zeros((4, 7 * N))
            for k in range(7):
                d = np.zeros(7)
                d[k] = h
                J[:, 7 * i + k] = (res(d, z) - res(-d, z)) / (2 * h)
                J[:, 7 * j + k] = (res(z, d) - res(z, -d)) / (2 * h)
            for c in range(4):
                H += om[c] * np.outer(J[c], J[c])
                g += om[c] * J[c] * e0[c]
    return H, g


@pytest.mark.parametrize("preset", [dict(sigma_ray=1.0, sigma_dist=1.0, huber_k=0.05),
                                    dict(sigma_ray=0.003, sigma_dist=10.0, huber_k=1.345)])
def test_system_vs_brute_force_fd(preset):
    rng = np.random.default_rng(3)
    poses_gt, X, conf, edges, match = tiny_clean_graph(seed=3, n_kf=3, n_pts=5, noise=0.02)
    match[0, 1] = -1            # one invalid, one out-of-range, one low-confidence match
    match[1, 2] = 99
    conf[0, 3] = 0.0
    poses = perturbed(poses_gt, rng, 0.03)
    prm = orc.Params(conf_min=0.05, **preset)
    sysm = orc.build_system(poses, X, conf, edges, match, prm)
    Hb, gb = brute_force_system(poses, X, conf, edges, match, prm)
    assert np.linalg.norm(sysm.H - Hb) <= 2e-6 * np.linalg.norm(Hb)
    assert np.linalg.norm(sysm.g - gb) <= 2e-6 * np.linalg.norm(gb)
    assert sysm.n_valid.sum() == edges.shape[0] * 5 - 2 - sum(
        1 for e in range(edges.shape[0]) for m in range(5)
        if 0 <= match[e, m] < 5 and (edges[e, 0] == 0 and m == 3 or edges[e, 1] == 0 and match[e, m] == 3))


def test_structure_invariants():
    g = make_graph(CONFIGS[1].scaled(height=6, width=8))
    prm = orc.Params(sigma_ray=1.0, sigma_dist=1.0, huber_k=0.05)
    sysm = orc.build_system(g.poses_init, g.points, g.conf, g.edges, g.match, prm)
    H, N = sysm.H, g.n_kf
    assert np.allclose(H, H.T, rtol=0, atol=1e-12 * np.abs(H).max())
    ev = np.linalg.eigvalsh(0.5 * (H + H.T))
    assert ev.min() >= -1e-9 * ev.max()
    # 7-dimensional null space (common world-frame twist): every block row sums to zero
    rows = H.reshape(N, 7, N, 7).sum(axis=2)
    assert np.abs(rows).max() <= 1e-10 * np.abs(H).max()
    assert np.abs(sysm.g.reshape(N, 7).sum(axis=0)).max() <= 1e-10 * np.abs(sysm.g).max()
    assert np.sum(ev < 1e-9 * ev.max()) == 7
    # sparsity: block (a,b) non-zero only if an edge joins a and b
    adj = np.eye(N, dtype=bool)
    for i, j in g.edges:
        adj[i, j] = adj[j, i] = True
    blocks = np.abs(H.reshape(N, 7, N, 7)).max(axis=(1, 3))
    assert np.all((blocks > 0) <= adj)
    # per-edge checksum / count by direct loops
    for e in range(g.n_edges):
        i, j = g.edges[e]
        cnt, chk = 0, 0
        for m in range(g.hw):
            n = int(g.match[e, m])
            if 0 <= n < g.hw and g.conf[i, m] > 0 and g.conf[j, n] > 0:
                cnt += 1
                chk = (chk + m * g.hw + n) % (1 << 64)
        assert cnt == sysm.n_valid[e] and chk == int(sysm.checksum[e])


def test_single_edge_blocks():
    poses, X, conf, edges, match = tiny_clean_graph(seed=5, n_kf=2, n_pts=9, noise=0.05)
    edges = np.array([[0, 1]], dtype=np.int32)
    match = match[:1]
    sysm = orc.build_system(poses, X, conf, edges, match, orc.Params())
    Hii, Hij, Hji, Hjj = sysm.H[:7, :7], sysm.H[:7, 7:], sysm.H[7:, :7], sysm.H[7:, 7:]
    assert np.allclose(Hii, Hjj, atol=1e-9 * np.abs(Hii).max())
    assert np.allclose(Hij, -Hii, atol=1e-9 * np.abs(Hii).max())
    assert np.allclose(Hji, -Hii, atol=1e-9 * np.abs(Hii).max())
    assert np.allclose(sysm.g[:7], -sysm.g[7:], atol=1e-9 * np.abs(sysm.g).max())
    assert np.allclose(sysm.edge_A[0], Hjj) and np.allclose(sysm.edge_b[0], sysm.g[7:])


def test_zero_residual_and_gradient_at_ground_truth():
    poses, X, conf, edges, match = tiny_clean_graph(seed=7, n_kf=4, n_pts=20)
    sysm = orc.build_system(poses, X, conf, edges, match, orc.Params())
    scale = np.abs(sysm.g_abs).max() + np.abs(sysm.H).max()
    assert sysm.cost <= 1e-18
    assert np.abs(sysm.g).max() <= 1e-12 * scale


def test_kappa_inf_step_equals_lstsq():
    """With kappa -> inf, one GN step (lambda = 0, eps0 = 0) is the linear least-squares solution
    of the stacked whitened finite-difference Jacobian (numpy.linalg.lstsq)."""
    rng = np.random.default_rng(9)
    poses_gt, X, conf, edges, match = tiny_clean_graph(seed=9, n_kf=3, n_pts=8, noise=0.03)
    poses = perturbed(poses_gt, rng, 0.04)
    prm = orc.Params(sigma_ray=0.7, sigma_dist=1.3, huber_k=1e30, eps0=0.0)
    sysm = orc.build_system(poses, X, conf, edges, match, prm)
    sol = orc.solve(sysm.H, sysm.g, [0], prm)
    assert sol.ok and sol.attempts == 1
    N = 3
    T4 = [orc.sim3_matrix(*orc.pose_to_srt(p)) for p in poses]
    sig = np.array([0.7, 0.7, 0.7, 1.3])
    rows, rhs = [], []
    h = 1e-6
    for e in range(edges.shape[0]):
        i, j = edges[e]
        for m in range(8):
            n = match[e, m]
            sq = (conf[i, m] * conf[j, n]) ** 0.25

            def res(di, dj):
                Ti = scipy.linalg.expm(gen4(di)) @ T4[i]
                Tj = scipy.linalg.expm(gen4(dj)) @ T4[j]
                return sq * orc.residual(_srt_from_4x4(np.linalg.inv(Ti) @ Tj), X[i, m][None], X[j, n][None])[0] / sig

            z = np.zeros(7)
            J = np.zeros((4, 7 * N))
            for k in range(7):
                d = np.zeros(7)
                d[k] = h
                J[:, 7 * i + k] = (res(d, z) - res(-d, z)) / (2 * h)
                J[:, 7 * j + k] = (res(z, d) - res(z, -d)) / (2 * h)
            rows.append(J)
            rhs.append(-res(z, z))
    A = np.concatenate(rows)[:, 7:]
    b = np.concatenate(rhs)
    ref = np.linalg.lstsq(A, b, rcond=None)[0]
    assert np.allclose(sol.tau[:7], 0.0)
    assert np.linalg.norm(sol.tau[7:] - ref) <= 1e-6 * np.linalg.norm(ref)


def test_solve_matches_numpy_and_fixes_gauge():
    rng = np.random.default_rng(10)
    n = 28
    A = rng.normal(size=(n + 5, n))
    H = A.T @ A
    g = rng.normal(size=n)
    prm = orc.Params(lm_lambda=0.1, eps0=1e-6)
    sol = orc.solve(H, g, [1], prm)
    fr = np.r_[0:7, 14:28]
    Hr = H[np.ix_(fr, fr)]
    ref = np.linalg.solve(Hr + 0.1 * np.diag(np.diag(Hr)) + 1e-6 * np.eye(21), -g[fr])
    assert sol.ok and sol.attempts == 1 and sol.eps_used == 1e-6
    assert np.allclose(sol.tau[fr], ref, rtol=1e-10, atol=1e-12)
    assert np.array_equal(sol.tau[7:14], np.zeros(7))


def test_epsilon_escalation_and_zero_update():
    n = 14
    H = np.eye(n)
    H[9, 9] = -5e-3                      # indefinite: needs eps > 5e-3 -> r = 2 (eps = 1e-2)
    g = np.ones(n)
    sol = orc.solve(H, g, [0], orc.Params())
    assert sol.ok and sol.attempts == 3 and np.isclose(sol.eps_used, 1e-2)
    assert np.isclose(sol.tau[9], -1.0 / (1e-2 - 5e-3))
    H[9, 9] = -1e6                       # beyond eps_5 = 1e4: all six attempts fail -> zero update
    sol = orc.solve(H, g, [0], orc.Params())
    assert (not sol.ok) and sol.attempts == 6 and np.array_equal(sol.tau, np.zeros(n))
    H[9, 9] = np.nan
    sol = orc.solve(H, g, [0], orc.Params())
    assert (not sol.ok) and np.array_equal(sol.tau, np.zeros(n))


def test_convergence_to_ground_truth_clean_data():
    rng = np.random.default_rng(12)
    poses_gt, X, conf, edges, match = tiny_clean_graph(seed=12, n_kf=5, n_pts=30)
    poses = perturbed(poses_gt, rng, 0.05)
    prm = orc.Params(sigma_ray=1.0, sigma_dist=1.0, huber_k=0.05, eps0=1e-12)
    costs = [orc.total_cost(poses, X, conf, edges, match, prm)]
    for _ in range(12):
        poses, sysm, sol = orc.gn_step(poses, X, conf, edges, match, [0], prm)
        assert sol.ok
        costs.append(orc.total_cost(poses, X, conf, edges, match, prm))
    assert all(b <= a * (1 + 1e-12) + 1e-24 for a, b in zip(costs, costs[1:])), costs
    assert np.array_equal(poses[0], poses_gt[0])
    for k in range(1, 5):
        assert np.linalg.norm(orc.pose_delta_log(poses[k], poses_gt[k])) < 1e-9


def test_total_cost_equals_system_cost():
    g = make_graph(CONFIGS[1].scaled(height=6, width=8))
    prm = orc.Params(sigma_ray=1.0, sigma_dist=1.0, huber_k=0.05)
    sysm = orc.build_system(g.poses_init, g.points, g.conf, g.edges, g.match, prm)
    assert np.isclose(sysm.cost, orc.total_cost(g.poses_init, g.points, g.conf, g.edges, g.match, prm), rtol=1e-13)
    assert np.isclose(sysm.cost, sysm.edge_cost.sum(), rtol=1e-13)


def test_bookkeeping_bruteforce():
    edges = np.array([[0, 1], [1, 2], [2, 1], [0, 2], [1, 0], [3, 1]], dtype=np.int32)
    bk = orc.bookkeeping(4, edges)
    assert bk["kf_ptr"].tolist() == [0, 3, 8, 11, 12]
    assert bk["kf_edge"].tolist() == [0, 3, 4, 0, 1, 2, 4, 5, 1, 2, 3, 5]
    assert bk["pair_kf"].tolist() == [[1, 0], [2, 0], [2, 1], [3, 1]]
    assert bk["pair_ptr"].tolist() == [0, 2, 3, 5, 6]
    assert bk["pair_edge"].tolist() == [0, 4, 3, 1, 2, 5]


def test_edge_pool_is_bit_identical_to_the_serial_oracle():
    """oracle/edge_pool.py runs the unchanged oracle one edge per call in worker processes and adds the 14 x 14 corners in
    edge order: every output equals the serial build_system bit for bit (duplicate and reversed edges included)."""
    from oracle.edge_pool import build_system_parallel
    g = make_graph(CONFIGS[3].scaled(kf_per_agent=5, height=20, width=30, n_scene=2_000, n_inter=3))
    edges = np.concatenate([g.edges, g.edges[:2, ::-1], g.edges[3:4]]).astype(np.int32)      # (j, i) and a duplicate
    match = np.concatenate([g.match, g.match[:2], g.match[3:4]])
    prm = orc.Params(sigma_ray=1.0, sigma_dist=1.0, huber_k=0.05, conf_min=0.2)
    ref = orc.build_system(g.poses_init, g.points, g.conf, edges, match, prm)
    for nw in (1, 3):
        par = build_system_parallel(g.poses_init, g.points, g.conf, edges, match, prm, n_workers=nw)
        for name in ("H", "g", "g_abs", "n_valid", "checksum", "edge_A", "edge_b", "edge_cost", "edge_b_abs"):
            assert np.array_equal(getattr(par, name), getattr(ref, name)), (nw, name)
        assert par.cost == ref.cost
    sub = [1, 4, 7]
    par = build_system_parallel(g.poses_init, g.points, g.conf, edges, match, prm, edge_subset=sub, n_workers=2, dense=False)
    ref = orc.build_system(g.poses_init, g.points, g.conf, edges, match, prm, edge_subset=sub)
    assert par.H is None and np.array_equal(par.g, ref.g) and np.array_equal(par.edge_A, ref.edge_A)
