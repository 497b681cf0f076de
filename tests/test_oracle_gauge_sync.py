"""Pins of oracle/gauge_sync_oracle.py (Eq. (3)-(4)) against things other than itself: exact recovery
of a known similarity, the reflection case, stationarity of the Eq. (3) objective, SciPy's Kabsch rotation, invariance of
the relative poses inside the moving component, the endpoint fallback."""
import numpy as np
from scipy.spatial.transform import Rotation

from oracle import gauge_sync_oracle as gs
from oracle import sim3_gn_oracle as orc
from sim3ba_inputs import CONFIGS, make_graph


def rand_sim3(rng):
    return float(np.exp(rng.uniform(np.log(0.3), np.log(3.0)))), Rotation.random(random_state=rng).as_matrix(), rng.normal(0, 2, 3)


def cost3(s, R, t, x, y):
    return float(np.sum((x - (s * y @ R.T + t)) ** 2))   # Eq. (3)


def test_exact_recovery_on_clean_points():
    rng = np.random.default_rng(3)
    for n in (3, 4, 64, 1000):
        s0, R0, t0 = rand_sim3(rng)
        y = rng.normal(0, 3, (n, 3))
        x = s0 * y @ R0.T + t0
        s, R, t = gs.umeyama(x, y)
        assert abs(s - s0) <= 1e-12 * s0 and np.allclose(R, R0, atol=1e-12) and np.allclose(t, t0, atol=1e-11)
        assert abs(np.linalg.det(R) - 1.0) <= 1e-12


def test_reflection_case_gives_a_proper_rotation_that_no_nearby_rotation_beats():
    rng = np.random.default_rng(5)
    y = rng.normal(0, 1, (200, 3)) * np.array([3.0, 2.0, 0.05])     # nearly planar cloud
    x = y * np.array([1.0, 1.0, -1.0]) + rng.normal(0, 0.01, y.shape)   # mirrored through the plane
    s, R, t = gs.umeyama(x, y)
    assert abs(np.linalg.det(R) - 1.0) <= 1e-12 and np.allclose(R @ R.T, np.eye(3), atol=1e-12)
    c0 = cost3(s, R, t, x, y)
    for _ in range(200):
        dR = orc.so3_exp(rng.normal(0, 0.05, 3))
        assert cost3(s, dR @ R, t, x, y) >= c0 - 1e-9
        assert cost3(s * np.exp(rng.normal(0, 0.05)), R, t + rng.normal(0, 0.05, 3), x, y) >= c0 - 1e-9


def test_stationary_point_of_eq3_and_kabsch_rotation():
    rng = np.random.default_rng(7)
    s0, R0, t0 = rand_sim3(rng)
    y = rng.normal(0, 2, (500, 3))
    x = s0 * y @ R0.T + t0 + rng.normal(0, 0.05, y.shape)
    s, R, t = gs.umeyama(x, y)
    h = 1e-6
    c0 = cost3(s, R, t, x, y)
    for k in range(7):                                    # central differences along the Sim(3) tangent directions
        tau = np.zeros(7)
        tau[k] = h
        cp = cost3(*orc.sim3_mul(orc.sim3_exp(tau), (s, R, t)), x, y)
        cm = cost3(*orc.sim3_mul(orc.sim3_exp(-tau), (s, R, t)), x, y)
        assert abs(cp - cm) / (2 * h) <= 1e-5 * max(c0, 1.0)
    # the optimal rotation of centred clouds does not depend on the scale: SciPy's Kabsch solution
    Rk, _ = Rotation.align_vectors(x - x.mean(0), y - y.mean(0))
    assert np.allclose(Rk.as_matrix(), R, atol=1e-9)
    # closed forms of Eq. (4) typed out again from the paper
    yt = y - y.mean(0)
    xt = x - x.mean(0)
    lam = np.linalg.svd(xt.T @ yt / len(x), compute_uv=False)
    assert np.isclose(s, lam.sum() / np.mean(np.sum(yt * yt, axis=1)))   # det(U V^T) = +1 here
    assert np.allclose(t, x.mean(0) - s * R @ y.mean(0))


def _two_agent_graph():
    spec = CONFIGS[3].scaled(kf_per_agent=5, height=24, width=32, n_scene=3_000, n_inter=2, sigma_n=0.0, p_out=0.0)
    g = make_graph(spec)
    e = int(np.flatnonzero(g.edge_kind == 2)[0])
    return g, e


def test_gauge_sync_moves_the_component_rigidly_and_closes_the_link():
    g, e = _two_agent_graph()
    i, j = (int(v) for v in g.edges[e])
    moving = [k for k in range(g.n_kf) if g.agent[k] == g.agent[j]]
    poses = g.poses_init_raw
    out, T, n_c = gs.gauge_sync(poses, g.points, g.conf, g.edges[e], g.match[e], moving)
    assert n_c >= gs.N_C_MIN
    for a in moving:                                     # relative poses inside the moving component are preserved
        for b in moving:
            before = orc.sim3_mul(orc.sim3_inv(*orc.pose_to_srt(poses[a])), orc.pose_to_srt(poses[b]))
            after = orc.sim3_mul(orc.sim3_inv(*orc.pose_to_srt(out[a])), orc.pose_to_srt(out[b]))
            assert np.allclose(orc.sim3_matrix(*before), orc.sim3_matrix(*after), atol=1e-10)
    for k in range(g.n_kf):
        if k not in moving:
            assert np.array_equal(out[k], poses[k])
    x0, y0 = gs.link_points(poses, g.points, g.conf, g.edges[e], g.match[e], 0.0)
    x1, y1 = gs.link_points(out, g.points, g.conf, g.edges[e], g.match[e], 0.0)
    assert np.sum((x1 - y1) ** 2) < 1e-3 * np.sum((x0 - y0) ** 2)   # the initial poses are perturbed: not exactly 0
    # the other direction: the component of i moves instead
    moving_i = [k for k in range(g.n_kf) if g.agent[k] == g.agent[i]]
    out_i, _, _ = gs.gauge_sync(poses, g.points, g.conf, g.edges[e], g.match[e], moving_i, moving_is_i=True)
    x2, y2 = gs.link_points(out_i, g.points, g.conf, g.edges[e], g.match[e], 0.0)
    assert np.isclose(np.sum((x2 - y2) ** 2) / orc.pose_to_srt(out_i[i])[0] ** 2, np.sum((x1 - y1) ** 2) / orc.pose_to_srt(out[i])[0] ** 2,
                      rtol=0.5)


def test_endpoint_fallback_below_64_correspondences():
    g, e = _two_agent_graph()
    i, j = (int(v) for v in g.edges[e])
    match = g.match[e].copy()
    keep = np.flatnonzero(match >= 0)[:63]
    sparse = np.full_like(match, -1)
    sparse[keep] = match[keep]
    moving = [k for k in range(g.n_kf) if g.agent[k] == g.agent[j]]
    out, T, n_c = gs.gauge_sync(g.poses_init_raw, g.points, g.conf, g.edges[e], sparse, moving)
    assert n_c == 63
    assert np.allclose(orc.sim3_matrix(*orc.pose_to_srt(out[j])), orc.sim3_matrix(*orc.pose_to_srt(g.poses_init_raw[i])), atol=1e-10)
    sparse[np.flatnonzero(match >= 0)[63]] = match[np.flatnonzero(match >= 0)[63]]
    _, _, n_c = gs.gauge_sync(g.poses_init_raw, g.points, g.conf, g.edges[e], sparse, moving)
    assert n_c == 64
