"""sim3ba_gauge_sync_static -- the entry point that allocates nothing (its scratch memory is a file-scope device array of
the library, images up to 2^18 pixels) -- against the existing, allocating path sim3ba_gauge_sync on the same inputs.

Collected last on purpose (the suite runs with ``pytest -x``).  The comparison uses the tolerance of
tests/test_gpu_gauge_sync.py (1e-9 absolute on poses of unit size); the two paths launch the same kernels on the same
grid, so the results are expected to be bit-identical, which is checked as well.  Calls are made back to back on contexts
of different image sizes (different numbers of scratch records in use), so the second and third call find the array
holding what the call before left there."""
import numpy as np
import pytest

from sim3ba_inputs import CONFIGS, make_graph
from tests.gpu_common import make_solver, oracle_params, set_poses
from tests.test_gpu_gauge_sync import pose_close

pytestmark = pytest.mark.gpu

TOL = 1e-9


def two_agent_graph(height, width, n_scene):
    return make_graph(CONFIGS[3].scaled(kf_per_agent=6, height=height, width=width, n_scene=n_scene, n_inter=3))


def existing_path(ba, g, e, moving, moving_is_i, n_c_min):
    set_poses(ba, g.poses_init_raw)
    T, n_c, fb = ba.gauge_sync(e, moving, moving_is_i, n_c_min)
    return T, n_c, fb, ba.get_poses().cpu().numpy()


def static_path(ba, g, e, moving, moving_is_i, n_c_min, result):
    import torch
    set_poses(ba, g.poses_init_raw)
    d_moving = torch.tensor(moving, dtype=torch.int32, device=ba.device)
    result.fill_(float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ba.gauge_sync_static(e, d_moving, result, moving_is_i, n_c_min)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    res = result.cpu().numpy()
    return res[:8], int(res[8]), bool(res[9]), ba.get_poses().cpu().numpy(), free0 - free1


def test_static_gauge_sync_equals_the_allocating_path_on_calls_in_a_row():
    import torch
    prm = oracle_params("config", conf_min=0.25)
    big = two_agent_graph(90, 120, 14_000)        # 10800 pixels: 11 scratch records, a ragged last block
    small = two_agent_graph(40, 50, 3_000)        # 2000 pixels: 2 records -- the rest of the array keeps `big`'s values
    ba_big, ba_small = make_solver(big, prm), make_solver(small, prm)
    result = torch.empty(10, dtype=torch.float64, device=ba_big.device)
    calls = []
    for g, ba in ((big, ba_big), (small, ba_small), (big, ba_big)):
        inter = np.flatnonzero(g.edge_kind == 2)
        e = int(inter[len(calls) % len(inter)])
        moving_is_i = len(calls) % 2 == 1
        side = int(g.edges[e, 0 if moving_is_i else 1])
        moving = [k for k in range(g.n_kf) if g.agent[k] == g.agent[side]]
        calls.append((g, ba, e, moving, moving_is_i, 64))
    # a fourth call below the correspondence threshold: the endpoint fallback through the same array
    g, ba, e, moving, moving_is_i, _ = calls[0]
    calls.append((g, ba, e, moving, moving_is_i, 10 ** 6))
    expected = [existing_path(ba, g, e, moving, mi, ncm) for g, ba, e, moving, mi, ncm in calls]
    for n, ((g, ba, e, moving, mi, ncm), (T0, nc0, fb0, poses0)) in enumerate(zip(calls, expected)):   # back to back
        T1, nc1, fb1, poses1, grown = static_path(ba, g, e, moving, mi, ncm, result)
        assert nc1 == nc0 and fb1 == fb0 and fb1 == (ncm > 64), n
        assert pose_close(T1[None], T0[None], TOL) and pose_close(poses1, poses0, TOL), n
        assert np.array_equal(T1, T0) and np.array_equal(poses1, poses0), n          # same kernels, same summation order
        assert not np.array_equal(poses1, g.poses_init_raw)
        if n > 0:
            assert grown == 0, "device memory in use changed across a call that must not allocate"
    # a device list nobody validated: out-of-range entries are skipped, the rest is transported as before
    g, ba, e, moving, mi, ncm = calls[0]
    set_poses(ba, g.poses_init_raw)
    d_moving = torch.tensor(moving[:2] + [-7, g.n_kf + 5] + moving[2:], dtype=torch.int32, device=ba.device)
    ba.gauge_sync_static(e, d_moving, result, mi, ncm)
    assert np.array_equal(ba.get_poses().cpu().numpy(), expected[0][3])
    # no moving keyframes: the estimate alone, poses untouched
    set_poses(ba, g.poses_init_raw)
    ba.gauge_sync_static(e, None, result, mi, ncm)
    assert np.array_equal(result.cpu().numpy()[:8], expected[0][0]) and np.array_equal(ba.get_poses().cpu().numpy(), g.poses_init_raw)
    # argument checks
    for bad in (lambda: ba.gauge_sync_static(g.n_edges, None, result), lambda: ba.gauge_sync_static(-1, None, result),
                lambda: ba.gauge_sync_static(e, None, result, n_c_min=0)):
        with pytest.raises(Exception):
            bad()
    ba_big.close()
    ba_small.close()


def test_static_gauge_sync_rejects_images_beyond_the_static_array():
    import torch
    g = make_graph(CONFIGS[3].scaled(kf_per_agent=1, height=513, width=512, n_scene=400_000, n_inter=1, offsets=(),
                               valid_frac=()))                                          # 262656 > 2^18 pixels
    assert g.n_kf == 2 and g.n_edges == 1 and g.hw > 262144
    ba = make_solver(g, oracle_params("config"))
    result = torch.zeros(10, dtype=torch.float64, device=ba.device)
    set_poses(ba, g.poses_init)
    before = ba.get_poses().cpu().numpy()
    with pytest.raises(Exception) as err:
        ba.gauge_sync_static(0, torch.tensor([1], dtype=torch.int32, device=ba.device), result)
    assert "262144" in str(err.value) and "sim3ba_gauge_sync" in str(err.value)
    assert np.array_equal(ba.get_poses().cpu().numpy(), before) and float(result.abs().sum()) == 0.0
    T, n_c, fb = ba.gauge_sync(0, [1])            # the allocating path takes the same image
    assert n_c > 64 and not fb
    ba.close()
