"""GPU-vs-oracle parity of sim3ba_gauge_sync (NEXT-2; Eq. (3)-(4)) through the C ABI: the similarity T*,
the number of correspondences (bit-exact: the GN step's match set), the transported poses, both directions, the endpoint
fallback below 64 correspondences, and the solve that follows on the raw (independent-gauge) start."""
import numpy as np
import pytest

from oracle import gauge_sync_oracle as gs
from oracle import sim3_gn_oracle as orc
from sim3ba_inputs import CONFIGS, make_graph
from tests.gpu_common import make_solver, oracle_params, rel, set_poses

pytestmark = pytest.mark.gpu


def pose_close(a, b, tol):
    sgn = np.sign(np.sum(a[..., 3:7] * b[..., 3:7], axis=-1, keepdims=True))
    bb = b.copy()
    bb[..., 3:7] *= sgn                       # q and -q are the same rotation
    return np.allclose(a, bb, rtol=0, atol=tol * max(1.0, float(np.abs(b).max())))


@pytest.mark.parametrize("moving_is_i", [False, True])
def test_gauge_sync_matches_oracle(moving_is_i):
    spec = CONFIGS[3].scaled(kf_per_agent=6, height=60, width=77, n_scene=9_000, n_inter=3)   # HW % 4 != 0 too
    g = make_graph(spec)
    prm = oracle_params("config", conf_min=0.25)
    ba = make_solver(g, prm)
    for e in np.flatnonzero(g.edge_kind == 2):
        i, j = (int(v) for v in g.edges[e])
        side = i if moving_is_i else j
        moving = [k for k in range(g.n_kf) if g.agent[k] == g.agent[side]]
        set_poses(ba, g.poses_init_raw)
        T, n_c, fb = ba.gauge_sync(int(e), moving, moving_is_i)
        ref, Tref, n_ref = gs.gauge_sync(g.poses_init_raw, g.points, g.conf, g.edges[e], g.match[e], moving, prm.conf_min, moving_is_i)
        assert n_c == n_ref and not fb
        assert pose_close(T[None], orc.srt_to_pose(*Tref)[None], 1e-9)
        assert pose_close(ba.get_poses().cpu().numpy(), ref, 1e-9)
        assert abs(np.linalg.norm(T[3:7]) - 1.0) <= 1e-14
    ba.close()


def test_gauge_sync_fallback_and_then_the_gn_step_runs():
    spec = CONFIGS[3].scaled(kf_per_agent=6, height=48, width=64, n_scene=6_000, n_inter=2)
    g = make_graph(spec)
    e = int(np.flatnonzero(g.edge_kind == 2)[0])
    i, j = (int(v) for v in g.edges[e])
    moving = [k for k in range(g.n_kf) if g.agent[k] == g.agent[j]]
    prm = oracle_params("config")
    # (a) 63 correspondences on the link: endpoint transform T_WCi T_WCj^-1
    sparse = g.match.copy()
    keep = np.flatnonzero(g.match[e] >= 0)[:63]
    sparse[e, :] = -1
    sparse[e, keep] = g.match[e, keep]
    g2 = make_graph(spec)
    g2.match[:] = sparse
    ba = make_solver(g2, prm)
    set_poses(ba, g.poses_init_raw)
    T, n_c, fb = ba.gauge_sync(e, moving)
    ref, Tref, n_ref = gs.gauge_sync(g.poses_init_raw, g.points, g.conf, g.edges[e], sparse[e], moving)
    assert n_c == n_ref == 63 and fb
    assert pose_close(ba.get_poses().cpu().numpy(), ref, 1e-12)
    ba.close()
    # (b) full link: synchronise on the device, then one GN step agrees with the oracle stepping from the oracle's sync
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init_raw)
    ba.gauge_sync(e, moving)
    ref, _, _ = gs.gauge_sync(g.poses_init_raw, g.points, g.conf, g.edges[e], g.match[e], moving)
    ba.step()
    tau = ba.update()[0].cpu().numpy()
    _, _, sol = orc.gn_step(ref, g.points, g.conf, g.edges, g.match, g.fixed_kf, prm)
    assert rel(tau, sol.tau, 1e-6 * np.sqrt(tau.size)) <= 1e-3
    ba.close()
    with pytest.raises(Exception):
        ba2 = make_solver(g, prm)
        try:
            ba2.gauge_sync(g.n_edges + 3, moving)
        finally:
            ba2.close()
