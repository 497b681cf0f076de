"""GPU-vs-oracle parity of sim3ba_depth_refine / sim3ba_apply_depth (NEXT-1; Eq. (8)-(10)) through the C
ABI: eta after 1 and after 10 iterations, the objective per iteration, anchors, excluded pixels, run-to-run bit
reproducibility, and one round of the pose-depth alternation."""
import numpy as np
import pytest

from oracle import depth_oracle as dp
from oracle import sim3_gn_oracle as orc
from sim3ba_inputs import CONFIGS, make_depth_inputs, make_graph
from tests.gpu_common import make_solver, oracle_params, rel, set_poses

pytestmark = pytest.mark.gpu


def graph(irregular=0, big=False):
    spec = CONFIGS[5].scaled(kf_per_agent=14, height=50, width=90, n_scene=9_000, loop_every=5)
    if big:       # several 512-pixel CTA iterations per tile, odd width (HW % 4 != 0, ragged last pair)
        spec = CONFIGS[5].scaled(kf_per_agent=10, height=111, width=163, n_scene=30_000, loop_every=4)
    g = make_graph(spec)
    # default: 4 x 8 = 32 segments per keyframe; irregular: ~M jittered superpixels (the paper's M_k ~ 200); 2 % excluded pixels
    return g, make_depth_inputs(g, irregular=irregular)


@pytest.mark.parametrize("preset,irregular,big", [("paper", 0, False), ("wide", 0, False), ("paper", 200, True), ("wide", 500, True)])
def test_depth_refine_matches_oracle(preset, irregular, big):
    import torch
    from paper_2605_30488_b200 import DepthParams
    g, d = graph(irregular, big)
    assert irregular == 0 or d.n_seg >= irregular
    prm = oracle_params("config", conf_min=0.2)
    dprm = dp.DepthParams(conf_min=prm.conf_min) if preset == "paper" else dp.DepthParams(sigma_point=0.5, huber_k=0.3, lambda_smooth=0.5,
                                                                                       lambda_prior=2.0, lambda_lm=0.2, eta_max=0.05,
                                                                                       conf_min=prm.conf_min)
    gp = DepthParams(dprm.sigma_point, dprm.huber_k, dprm.lambda_smooth, dprm.lambda_prior, dprm.lambda_lm, dprm.eta_max)
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    labels = torch.from_numpy(d.labels).cuda()
    M = g.n_kf * d.n_seg
    rng = np.random.default_rng(1)
    eta0 = rng.normal(0, 0.02, M)
    for k in d.anchor_kf:
        eta0[k * d.n_seg:(k + 1) * d.n_seg] = 0.0
    for n_it in (1, 10):
        eta = torch.from_numpy(eta0.copy()).cuda()
        cost = ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta, n_it, gp)
        ref, ref_cost = dp.depth_refine(g.poses_init, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta0, d.pairs, d.delta,
                                        d.anchor_kf, dprm, n_it)
        out = eta.cpu().numpy()
        assert rel(out - eta0, ref - eta0) <= 1e-6, (preset, n_it)      # the update itself (FP64 both sides; fp32 inputs)
        assert rel(cost, ref_cost) <= 1e-7                              # q from the packed fp32 w = c^(1/4): 1e-7 per match
        for k in d.anchor_kf:
            assert np.array_equal(out[k * d.n_seg:(k + 1) * d.n_seg], eta0[k * d.n_seg:(k + 1) * d.n_seg])
        eta_b = torch.from_numpy(eta0.copy()).cuda()
        ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta_b, n_it, gp)
        assert np.array_equal(out, eta_b.cpu().numpy())                 # fixed reduction order: bitwise reproducible
    ba.close()


def test_depth_refine_full_size_config2_paper_segment_count():
    """BASELINE configs[1] at full size (32 keyframes 512x384, 96 edges, 1.9e7 candidate matches -- the tile / patch / ring
    configuration the bench times) with ~200 irregular segments per keyframe, the paper's M_k: eta after two
    iterations and the objective against the oracle."""
    import torch
    from sim3ba_inputs import make_config
    g = make_config(2)
    d = make_depth_inputs(g, irregular=200)
    prm = oracle_params("config")
    dprm = dp.DepthParams()
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    M = g.n_kf * d.n_seg
    eta0 = np.random.default_rng(3).normal(0, 0.02, M)
    for k in d.anchor_kf:
        eta0[k * d.n_seg:(k + 1) * d.n_seg] = 0.0
    eta = torch.from_numpy(eta0.copy()).cuda()
    cost = ba.depth_refine(torch.from_numpy(d.labels).cuda(), d.n_seg, d.pairs, d.delta, d.anchor_kf, eta, 2)
    ref, ref_cost = dp.depth_refine(g.poses_init, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta0, d.pairs, d.delta, d.anchor_kf,
                                    dprm, 2)
    assert rel(eta.cpu().numpy() - eta0, ref - eta0) <= 1e-6
    assert rel(cost, ref_cost) <= 1e-7
    ba.close()


def scaled_points(g, d, eta):
    """X(eta) = exp(eta_g) X_init (Eq. (8)) as the fp32 pointmaps the next pose pass sees, in NumPy float64."""
    scale = np.ones((g.n_kf, g.hw))
    for k in range(g.n_kf):
        ok = d.labels[k] >= 0
        scale[k, ok] = np.exp(eta[k * d.n_seg + d.labels[k, ok]])
    return (g.points.astype(np.float64) * scale[:, :, None]).astype(np.float32)


@pytest.mark.parametrize("irregular", [0, 200])
def test_two_alternation_rounds_lockstep_and_free_running(irregular):
    """The pose-depth alternation of PAPER.md:143,177 over TWO rounds with eta carried across them (eta is the absolute
    log-scale of Eq. (8): the second structure pass must see the pristine X_init, not the pointmaps sim3ba_apply_depth
    has rescaled).  Lock-step: in every round the device starts from the ORACLE's poses and eta, so the bars hold as
    stated -- eta update <= 1e-6, tau <= 1e-3.  Then free-running, each side on its own numbers: <= 1e-3 on both."""
    import torch
    g, d = graph(irregular)
    prm = oracle_params("config")
    dprm = dp.DepthParams()
    n_dit, M = 3, g.n_kf * d.n_seg
    labels = torch.from_numpy(d.labels).cuda()
    pts, cf = torch.from_numpy(g.points).cuda(), torch.from_numpy(g.conf).cuda()
    ba = make_solver(g, prm)
    poses, eta = g.poses_init.copy(), np.zeros(M)
    for rnd in range(2):
        set_poses(ba, poses)
        eta_dev = torch.from_numpy(eta.copy()).cuda()
        ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta_dev, n_dit)
        eta_ref, _ = dp.depth_refine(poses, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta, d.pairs, d.delta, d.anchor_kf, dprm,
                                     n_dit)
        assert rel(eta_dev.cpu().numpy() - eta, eta_ref - eta) <= 1e-6, rnd
        eta = eta_ref
        ba.apply_depth(pts, cf, labels, d.n_seg, torch.from_numpy(eta).cuda())
        ba.build_system()
        ba.solve()
        tau = ba.update()[0].cpu().numpy()
        pts_ref = scaled_points(g, d, eta)
        sysm = orc.build_system(poses, pts_ref, g.conf, g.edges, g.match, prm)
        sol = orc.solve(sysm.H, sysm.g, g.fixed_kf, prm)
        assert rel(tau, sol.tau, 1e-6 * np.sqrt(tau.size)) <= 1e-3, rnd
        poses = orc.retract(poses, sol.tau)
    ba.close()
    # free-running: two rounds of {n_dit depth iterations, apply, 2 GN steps} on each side's own numbers
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    eta_dev = torch.zeros(M, dtype=torch.float64, device="cuda")
    poses, eta = g.poses_init.copy(), np.zeros(M)
    for rnd in range(2):
        ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta_dev, n_dit)
        ba.apply_depth(pts, cf, labels, d.n_seg, eta_dev)
        eta, _ = dp.depth_refine(poses, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta, d.pairs, d.delta, d.anchor_kf, dprm, n_dit)
        pts_ref = scaled_points(g, d, eta)
        for _ in range(2):
            ba.step()
            poses, _, _ = orc.gn_step(poses, pts_ref, g.conf, g.edges, g.match, g.fixed_kf, prm)
    assert rel(eta_dev.cpu().numpy(), eta) <= 1e-3
    out = ba.get_poses().cpu().numpy()
    d_gpu = np.concatenate([orc.pose_delta_log(out[i], g.poses_init[i]) for i in range(g.n_kf)])
    d_orc = np.concatenate([orc.pose_delta_log(poses[i], g.poses_init[i]) for i in range(g.n_kf)])
    assert rel(d_gpu, d_orc) <= 1e-3
    ba.close()


def test_refine_host_one_call_equals_the_manual_rounds_and_the_chained_oracles():
    """sim3ba_refine_host (host buffers in, poses and eta out) runs the very same kernels as the manual sequence
    depth_refine -> apply_depth -> n x step per round: bit-identical poses, eta and cost traces; and it agrees with the two
    oracles chained on their own numbers to 1e-3 (free-running)."""
    import torch
    from paper_2605_30488_b200 import refine_host
    from tests.gpu_common import gpu_params
    g, d = graph(irregular=200)
    prm = oracle_params("config")
    dprm = dp.DepthParams()
    n_rounds, n_dit, n_pit = 2, 3, 2
    M = g.n_kf * d.n_seg
    labels = torch.from_numpy(d.labels).cuda()
    pts, cf = torch.from_numpy(g.points).cuda(), torch.from_numpy(g.conf).cuda()
    ba = make_solver(g, prm)
    set_poses(ba, g.poses_init)
    eta_dev = torch.zeros(M, dtype=torch.float64, device="cuda")
    pose_cost, depth_cost = [], []
    for _ in range(n_rounds):
        depth_cost += list(ba.depth_refine(labels, d.n_seg, d.pairs, d.delta, d.anchor_kf, eta_dev, n_dit))
        ba.apply_depth(pts, cf, labels, d.n_seg, eta_dev)
        for _ in range(n_pit):
            ba.step()
            pose_cost.append(ba.update()[3])
    ref_poses, ref_eta = ba.get_poses().cpu().numpy(), eta_dev.cpu().numpy()
    ba.close()
    h_out = torch.empty((g.n_kf, 8), dtype=torch.float64).pin_memory()
    h_eta = torch.zeros(M, dtype=torch.float64).pin_memory()
    h_pc = torch.empty(n_rounds * n_pit, dtype=torch.float64).pin_memory()
    h_dc = torch.empty(n_rounds * n_dit, dtype=torch.float64).pin_memory()
    refine_host(torch.from_numpy(g.points).pin_memory(), torch.from_numpy(g.conf).pin_memory(), torch.from_numpy(g.edges).contiguous(),
                torch.from_numpy(g.match).pin_memory(), g.fixed_kf, gpu_params(prm), g.spec.height, g.spec.width,
                torch.from_numpy(d.labels).pin_memory(), d.n_seg, d.pairs, d.delta, None, n_rounds, n_dit, n_pit,
                torch.from_numpy(g.poses_init.copy()), h_out, h_eta, h_pc, h_dc, torch.cuda.current_stream().cuda_stream)
    assert np.array_equal(h_out.numpy(), ref_poses) and np.array_equal(h_eta.numpy(), ref_eta)
    assert np.array_equal(h_pc.numpy(), np.asarray(pose_cost)) and np.array_equal(h_dc.numpy(), np.asarray(depth_cost))
    poses, eta = g.poses_init.copy(), np.zeros(M)
    for _ in range(n_rounds):
        eta, _ = dp.depth_refine(poses, g.points, g.conf, g.edges, g.match, d.labels, d.n_seg, eta, d.pairs, d.delta, d.anchor_kf, dprm, n_dit)
        pts_ref = scaled_points(g, d, eta)
        for _ in range(n_pit):
            poses, _, _ = orc.gn_step(poses, pts_ref, g.conf, g.edges, g.match, g.fixed_kf, prm)
    assert rel(h_eta.numpy(), eta) <= 1e-3
    d_gpu = np.concatenate([orc.pose_delta_log(h_out.numpy()[i], g.poses_init[i]) for i in range(g.n_kf)])
    d_orc = np.concatenate([orc.pose_delta_log(poses[i], g.poses_init[i]) for i in range(g.n_kf)])
    assert rel(d_gpu, d_orc) <= 1e-3


def test_argument_checks():
    import torch
    from paper_2605_30488_b200 import Sim3BAError
    g, d = graph()
    ba = make_solver(g, oracle_params("config"))
    labels = torch.from_numpy(d.labels).cuda()
    M = g.n_kf * d.n_seg
    eta = torch.zeros(M, dtype=torch.float64, device="cuda")
    with pytest.raises(Sim3BAError):
        ba.depth_refine(labels, 513, d.pairs, d.delta, d.anchor_kf, torch.zeros(g.n_kf * 513, dtype=torch.float64, device="cuda"), 1)
    bad = d.pairs.copy()
    bad[0, 0] = M + 7
    with pytest.raises(Sim3BAError):
        ba.depth_refine(labels, d.n_seg, bad, d.delta, d.anchor_kf, eta, 1)
    ba.close()
