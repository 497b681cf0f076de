"""Pins of oracle/depth_oracle.py (Eq. (8)-(10)) against things other than itself: central differences of
the objective for the gradient, the second difference at a zero-residual point for the Jacobi diagonal, fixed point at
eta = 0 on clean data, recovery of a known per-segment scale error, monotone descent, anchors and clip."""
import numpy as np

from oracle import depth_oracle as dp
from sim3ba_inputs import CONFIGS, clean_variant, make_depth_inputs, make_graph


def small(clean=False, seed_spec=5):
    spec = CONFIGS[seed_spec].scaled(kf_per_agent=5, height=24, width=32, n_scene=2_000, loop_every=3)
    if clean:
        spec = clean_variant(spec)
    g = make_graph(spec)
    return g, make_depth_inputs(g, grid=(2, 4), drop_frac=0.05)


def objective(g, d, poses, eta, prm):
    return dp.depth_terms(poses, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta, d.pairs, d.delta, prm)[2]


def test_gradient_is_the_derivative_of_the_objective():
    g, d = small()
    rng = np.random.default_rng(2)
    for prm in (dp.DepthParams(), dp.DepthParams(huber_k=1e9), dp.DepthParams(sigma_point=1.0, huber_k=0.05)):
        eta = rng.normal(0, 0.05, g.n_kf * d.n_seg)
        grad, H, _ = dp.depth_terms(g.poses_init, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta, d.pairs, d.delta, prm)
        assert np.all(H >= prm.lambda_prior)
        h = 1e-6
        for a in rng.choice(eta.size, 12, replace=False):
            ep, em = eta.copy(), eta.copy()
            ep[a] += h
            em[a] -= h
            fd = (objective(g, d, g.poses_init, ep, prm) - objective(g, d, g.poses_init, em, prm)) / (2 * h)
            assert abs(fd - grad[a]) <= 1e-5 * max(1.0, abs(grad[a])), (a, fd, grad[a])


def test_jacobi_diagonal_is_the_second_derivative_at_zero_residual():
    g, d = small(clean=True)
    prm = dp.DepthParams(huber_k=1e9)
    eta = np.zeros(g.n_kf * d.n_seg)
    no_bnd = (np.zeros((0, 2), np.int32), np.zeros(0))
    grad, H, c0 = dp.depth_terms(g.poses_gt, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta, *no_bnd, prm)
    assert c0 <= 1e-6 and np.all(np.abs(grad) <= 1e-5 * H)          # fp32 pointmaps: residuals ~ 1e-6 m, |J| ~ 10 m
    h = 1e-4
    for a in range(0, eta.size, 5):
        ep, em = eta.copy(), eta.copy()
        ep[a] += h
        em[a] -= h
        cp = dp.depth_terms(g.poses_gt, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, ep, *no_bnd, prm)[2]
        cm = dp.depth_terms(g.poses_gt, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, em, *no_bnd, prm)[2]
        fd2 = (cp - 2 * c0 + cm) / (h * h)
        assert abs(fd2 - H[a]) <= 2e-3 * H[a] + 1e-6, (a, fd2, H[a])
    # boundary and prior alone: exact diagonal of a quadratic
    z = np.zeros_like(g.match)
    z[:] = -1
    _, Hb, _ = dp.depth_terms(g.poses_gt, g.points, g.conf, g.edges, z, d.labels, d.n_seg, eta, d.pairs, d.delta, prm)
    deg = np.bincount(d.pairs.reshape(-1), minlength=eta.size)
    assert np.allclose(Hb, prm.lambda_prior + prm.lambda_smooth * deg)


def test_fixed_point_recovery_descent_anchor_clip():
    g, d = small(clean=True)
    prm = dp.DepthParams()
    M = g.n_kf * d.n_seg
    zero_delta = np.zeros_like(d.delta)
    # eta = 0 stays put on clean data at the true poses (planar patches: Delta_gh of the data itself is not 0, so no boundary)
    eta, costs = dp.depth_refine(g.poses_gt, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, np.zeros(M),
                                 np.zeros((0, 2), np.int32), np.zeros(0), d.anchor_kf, prm, 3)
    assert np.max(np.abs(eta)) <= 1e-4
    # a known scale error on some segments of non-anchor keyframes is pulled back (prior shrinks it slightly: compare signs / size)
    pts = g.points.copy()
    bad = {(2, 3): 0.08, (3, 1): -0.06, (4, 6): 0.05}
    for (k, lab), a in bad.items():
        pts[k, d.labels[k] == lab] *= np.float32(np.exp(a))
    eta, costs = dp.depth_refine(g.poses_gt, pts, g.conf, g.edges, g.match, d.labels, d.n_seg, np.zeros(M),
                                 np.zeros((0, 2), np.int32), np.zeros(0), d.anchor_kf, prm, 10)
    assert np.all(np.diff(costs) <= 1e-9 * costs[0])
    for (k, lab), a in bad.items():
        assert abs(eta[k * d.n_seg + lab] + a) <= 0.2 * abs(a), (k, lab, eta[k * d.n_seg + lab], a)
    for k in d.anchor_kf:
        assert np.all(eta[k * d.n_seg:(k + 1) * d.n_seg] == 0.0)
    # clip
    pts2 = g.points.copy()
    pts2[2] *= np.float32(np.exp(2.0))
    eta1, _ = dp.depth_step(g.poses_gt, pts2, g.conf, g.edges, g.match, d.labels, d.n_seg, np.zeros(M), d.pairs, zero_delta,
                            d.anchor_kf, prm)
    assert np.max(np.abs(eta1)) <= prm.eta_max + 1e-15 and np.any(np.abs(eta1) == prm.eta_max)
