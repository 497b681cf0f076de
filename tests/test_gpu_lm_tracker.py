"""SURVEY section 8(f) NEXT-4 through the C ABI: Eq. (7) with lambda > 0 ("The tracker uses LM damping",
PAPER.md:122; per-agent local graphs with LM-IRLS) on all three solver plans, and the tracker's shape --
one relative pose against a fixed keyframe (E_track): N = 2, E = 1, n = 7 -- stepped with a fixed lambda.
The tracker's accept / reject rule for lambda is not in the paper (parity unpinned) and is not built: lambda stays
what the caller sets."""
import numpy as np
import pytest

from oracle import sim3_gn_oracle as orc
from sim3ba_inputs import CONFIGS, make_config, make_graph
from tests.gpu_common import TOL_TAU, make_solver, oracle_params, rel, set_poses, start_poses
from tests.test_gpu_parity import check_system, reduced

pytestmark = pytest.mark.gpu


def tracker_graph(height, width):
    """Two keyframes of one agent, one edge (0, 1), keyframe 0 fixed: the relative-pose problem of the tracker."""
    spec = CONFIGS[2].scaled(name="tracker", kf_per_agent=2, height=height, width=width, offsets=(1,), valid_frac=(0.9,),
                             cyclic=False, n_iters=4)
    g = make_graph(spec)
    assert g.n_kf == 2 and g.n_edges == 1 and tuple(g.edges[0]) == (0, 1)
    return g


@pytest.mark.parametrize("lam", [0.1, 1.0])
@pytest.mark.parametrize("which", ["C1", "C3r"])
def test_lm_damped_lockstep_all_solver_modes(which, lam):
    """(H + lambda diag(H) + eps I) tau = -g against the oracle, lock-step over three iterations, on the band + border,
    tile-sparse and dense plans."""
    g = make_config(1) if which == "C1" else make_graph(reduced(3))
    prm = oracle_params("config", lm_lambda=lam)
    for mode in (2, 0, 1):
        ba = make_solver(g, prm)
        ba.set_solver_mode(mode)
        poses = start_poses(g, prm)
        for it in range(3):
            _, sol = check_system(ba, g, poses, prm, f"{which}/lm{lam}/mode{mode}/it{it}")
            poses = orc.retract(poses, sol.tau)
        ba.close()
    # the damping is really in: the undamped update differs
    ba = make_solver(g, oracle_params("config"))
    set_poses(ba, start_poses(g, prm))
    ba.build_system()
    ba.solve()
    tau0 = ba.update()[0].cpu().numpy()
    ba.close()
    sysm = orc.build_system(start_poses(g, prm), g.points, g.conf, g.edges, g.match, prm)
    assert rel(tau0, orc.solve(sysm.H, sysm.g, g.fixed_kf, prm).tau) > 10 * TOL_TAU


@pytest.mark.parametrize("hw", [(48, 64), (384, 512)])
@pytest.mark.parametrize("lam", [0.0, 0.5])
def test_tracker_shape_single_relative_pose(hw, lam):
    """E = 1, N = 2, keyframe 0 fixed, n = 7: lock-step LM iterations with lambda fixed, then the free-running poses --
    stepped kernel by kernel and as ONE CUDA-graph launch (sim3ba_step_graph), bit-identical to each other."""
    g = tracker_graph(*hw)
    prm = oracle_params("config", lm_lambda=lam)
    ba = make_solver(g, prm)
    info = ba.bb_info()
    assert info["valid"] == 1 and info["n_interior"] + info["n_border"] == 1
    poses = g.poses_init.copy()
    for it in range(3):
        _, sol = check_system(ba, g, poses, prm, f"tracker{hw[0]}x{hw[1]}/lm{lam}/it{it}")
        poses = orc.retract(poses, sol.tau)
    n_it = 4
    set_poses(ba, g.poses_init)
    for _ in range(n_it):
        ba.step()
    stepped = ba.get_poses().cpu().numpy()
    set_poses(ba, g.poses_init)
    ba.step_graph(n_it)
    graphed = ba.get_poses().cpu().numpy()
    assert np.array_equal(stepped, graphed)
    set_poses(ba, g.poses_init)
    ba.step_graph(n_it)                                  # replay of the cached graph
    assert np.array_equal(stepped, ba.get_poses().cpu().numpy())
    ref = g.poses_init.copy()
    for _ in range(n_it):
        ref, _, _ = orc.gn_step(ref, g.points, g.conf, g.edges, g.match, g.fixed_kf, prm)
    d_gpu = orc.pose_delta_log(stepped[1], g.poses_init[1])
    d_orc = orc.pose_delta_log(ref[1], g.poses_init[1])
    assert rel(d_gpu, d_orc) <= TOL_TAU
    assert np.array_equal(stepped[0], g.poses_init[0])
    ba.close()


def test_step_graph_on_config1_and_after_a_parameter_change():
    """The graph is rebuilt when the constants change (they are kernel arguments of the captured launches)."""
    from tests.gpu_common import gpu_params
    g = make_config(1)
    prm = oracle_params("config")
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    ba.step_graph(2)
    a = ba.get_poses().cpu().numpy()
    set_poses(ba, g.poses_init)
    ba.step()
    ba.step()
    assert np.array_equal(a, ba.get_poses().cpu().numpy())
    prm2 = oracle_params("config", lm_lambda=2.0)
    ba.set_params(gpu_params(prm2))
    set_poses(ba, g.poses_init)
    ba.step_graph(2)
    b = ba.get_poses().cpu().numpy()
    assert not np.array_equal(a, b)
    set_poses(ba, g.poses_init)
    ba.step()
    ba.step()
    assert np.array_equal(b, ba.get_poses().cpu().numpy())
    ba.close()
