"""Shared helpers of the GPU parity tests: move a seeded graph to the device, wrap oracle outputs
in the layouts of the C ABI, relative-error norms.  No arithmetic of the method lives here."""
import json
import os

import numpy as np

from oracle import gauge_sync_oracle as gs
from oracle import sim3_gn_oracle as orc
from sim3ba_inputs import PRESETS

TOL_BLOCK = 1e-4   # relative Frobenius, assembled Hessian / gradient / per-edge blocks (north_star)
TOL_TAU = 1e-3     # relative 2-norm, pose update (north_star)


def oracle_params(preset="config", **kw):
    d = dict(PRESETS[preset])
    d.update(kw)
    return orc.Params(**d)


def gpu_params(p: orc.Params):
    from paper_2605_30488_b200 import make_params
    return make_params(p.sigma_ray, p.sigma_dist, p.huber_k, p.conf_min, p.lm_lambda, p.eps0, p.max_attempts)


def make_solver(g, prm: orc.Params, fixed=None):
    import torch
    from paper_2605_30488_b200 import Sim3BA
    dev = torch.device("cuda:0")
    ba = Sim3BA(torch.from_numpy(g.points).to(dev), torch.from_numpy(g.conf).to(dev),
                torch.from_numpy(g.edges).to(dev).contiguous(), torch.from_numpy(g.match).to(dev),
                g.fixed_kf if fixed is None else fixed, gpu_params(prm), g.spec.height, g.spec.width)
    return ba


def set_poses(ba, poses: np.ndarray):
    import torch
    ba.set_poses(torch.from_numpy(np.ascontiguousarray(poses)).to(ba.device))


def blocks35_from_oracle(sysm) -> np.ndarray:
    iu = np.triu_indices(7)
    return np.concatenate([sysm.edge_A[:, iu[0], iu[1]], sysm.edge_b], axis=1)


def sym_from_lower(Hl: np.ndarray) -> np.ndarray:
    return np.tril(Hl) + np.tril(Hl, -1).T


def rel(a: np.ndarray, b: np.ndarray, floor: float = 0.0) -> float:
    """||a - b|| / max(||b||, floor) (Frobenius / 2-norm)."""
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), floor, 1e-300))


def free_idx(g, fixed=None):
    return orc.free_index(g.n_kf, g.fixed_kf if fixed is None else fixed)


def start_poses(g, prm: orc.Params) -> np.ndarray:
    """The seeded start of a graph.  Config 3 hands out independent per-agent gauges plus the plan to synchronise them
    (PAPER.md:92-104); here the ORACLE's gauge synchronisation executes the plan, so no oracle input ever comes from the
    CUDA path (sim3ba_gauge_sync itself is compared with it in tests/test_gpu_gauge_sync.py)."""
    poses = g.poses_init.copy()
    for e, moving, moving_is_i in g.meta.get("gauge_sync_plan", []):
        poses, _, _ = gs.gauge_sync(poses, g.points, g.conf, g.edges[e], g.match[e], moving, prm.conf_min, moving_is_i)
    return poses


def parity_log(**rec):
    """Appends one record of measured parity errors to $SIM3BA_PARITY_LOG (JSON lines) -- the table of DESIGN.md
    "Parity protocol" is made from these; without the variable nothing is written."""
    path = os.environ.get("SIM3BA_PARITY_LOG")
    if not path:
        return
    with open(path, "a") as f:
        f.write(json.dumps({k: (float(v) if isinstance(v, (np.floating, float)) else v) for k, v in rec.items()}) + "\n")
