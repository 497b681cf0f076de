"""Seeded synthetic graphs for the Sim(3) Gauss-Newton step.

They stand in for the paper's Tanks-and-Temples / Waymo / Oxford-Spires workloads
(PAPER.md:149,242-244), which are not available: shapes, sizes, outlier fractions and overlap
fractions follow BASELINE.json's five configs.  No item of any of those datasets is reproduced.

Pose layout everywhere in this repository: ``pose[8] = (tx, ty, tz, qx, qy, qz, qw, s)`` for
``T_WC : X -> s * R(q) * X + t``.

All random draws come from ``numpy.random.Generator(PCG64)`` seeded with
``SeedSequence(seed, spawn_key=(kind, index))`` so that every keyframe and every edge has its own
stream and generation is order independent.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Tuple

import numpy as np

# ----------------------------------------------------------------------------------------------
# robust-kernel presets (reading #6): "config" = raw-residual Huber delta of config 1,
# "paper" = the constants of PAPER.md:76,177.
PRESETS: Dict[str, Dict[str, float]] = {
    "config": dict(sigma_ray=1.0, sigma_dist=1.0, huber_k=0.05),
    "paper": dict(sigma_ray=0.003, sigma_dist=10.0, huber_k=1.345),
}

# Parameters a config runs with on top of its preset.  Config 5 (2000 keyframes in one open chain, 20 % uniform-random
# outlier matches): every outlier pulls with the constant Huber influence kappa, the pull does not average out on an edge,
# and the per-edge bias of the relative pose adds up along 2000 sequential edges -- the minimiser of Eq. (5) lies tens of
# units (translation) and several e-folds (scale) away from the seeded start, in the weakest modes of H (smallest
# eigenvalue 2e-3 against 6e7).  The undamped step (lambda = 0) takes that whole distance at once and leaves the basin
# (cost 3.09e7, 3.01e7, 7.2e7, 2.5e8, ... with a failed factorisation on the way); with the diagonal damping of Eq. (7)
# the cost falls monotonically (3.09e7, 2.894e7, 2.881e7, 2.876e7, 2.873e7).  Configs 1-4 converge
# undamped and keep lambda = 0.  Measured on the device, DESIGN.md section 11.
CONFIG_PARAMS: Dict[int, Dict[str, float]] = {5: dict(lm_lambda=1e-4)}


def config_params(k: int, preset: str = "config") -> Dict[str, float]:
    """Keyword arguments of the parameter struct (oracle Params / make_params) config k is run with."""
    d = dict(PRESETS[preset])
    d.update(CONFIG_PARAMS.get(int(k), {}))
    return d


_K_SCENE, _K_POSE, _K_KF, _K_EDGE, _K_INIT, _K_GAUGE = range(6)


def _rng(seed: int, kind: int, index: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence(seed, spawn_key=(kind, index))))


# ----------------------------------------------------------------------------------------------
# plain rigid/similarity plumbing (composition only; the method's Exp/Log live elsewhere)
def _quat_to_mat(q: np.ndarray) -> np.ndarray:
    x, y, z, w = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


def _quat_mul(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    ax, ay, az, aw = a
    bx, by, bz, bw = b
    return np.array([
        aw * bx + ax * bw + ay * bz - az * by,
        aw * by - ax * bz + ay * bw + az * bx,
        aw * bz + ax * by - ay * bx + az * bw,
        aw * bw - ax * bx - ay * by - az * bz,
    ])


def _quat_from_rotvec(r: np.ndarray) -> np.ndarray:
    th = float(np.linalg.norm(r))
    if th < 1e-12:
        q = np.array([0.5 * r[0], 0.5 * r[1], 0.5 * r[2], 1.0])
    else:
        q = np.concatenate([np.sin(0.5 * th) * r / th, [np.cos(0.5 * th)]])
    return q / np.linalg.norm(q)


def _compose(a: np.ndarray, b: np.ndarray) -> np.ndarray:
    """pose a after pose b (a o b), both in the 8-vector layout."""
    Ra = _quat_to_mat(a[3:7])
    t = a[7] * Ra @ b[0:3] + a[0:3]
    q = _quat_mul(a[3:7], b[3:7])
    q = q / np.linalg.norm(q)
    return np.concatenate([t, q, [a[7] * b[7]]])


def _random_unit(rng: np.random.Generator, n: Optional[int] = None) -> np.ndarray:
    v = rng.normal(size=(3,) if n is None else (n, 3))
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _haar_quat(rng: np.random.Generator) -> np.ndarray:
    q = rng.normal(size=4)
    return q / np.linalg.norm(q)


def _n_threads() -> int:
    try:
        n = len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        n = os.cpu_count() or 1
    return max(1, min(32, n))


# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class GraphSpec:
    name: str
    seed: int
    n_agents: int
    kf_per_agent: int
    height: int
    width: int
    n_scene: int
    n_planes: int
    plane_side: float
    offsets: Tuple[int, ...]          # intra-agent edges (k, k+d) for d in offsets
    cyclic: bool                      # offsets taken modulo kf_per_agent (closed loop)
    n_inter: int                      # inter-agent edges
    loop_every: int                   # loop closures (k, k-loop_every), 0 = none
    valid_frac: Tuple[float, ...]     # per offset
    valid_frac_loop: float
    valid_frac_inter: float
    p_out: float                      # outlier fraction of the valid matches
    sigma_n: float                    # pointmap noise (std per coordinate)
    pose_mode: str                    # "iid" (config 1) or "walk"
    agent_gauge: bool                 # config 3: independent per-agent gauges on the initial poses
    n_iters: int
    n_segments: Tuple[int, int] = (0, 0)   # config 5: rectangular segment grid (rows, cols)

    @property
    def n_kf(self) -> int:
        return self.n_agents * self.kf_per_agent

    @property
    def hw(self) -> int:
        return self.height * self.width

    def scaled(self, **kw) -> "GraphSpec":
        """A reduced variant (smaller image / fewer keyframes) for tests; everything else kept."""
        return replace(self, **kw)


CONFIGS: Dict[int, GraphSpec] = {
    1: GraphSpec("C1-tiny", 0, 2, 4, 48, 64, 2000, 3, 10.0, (1, 2), False, 2, 0,
                 (0.9, 0.8), 0.5, 0.3, 0.10, 0.01, "iid", False, 1),
    2: GraphSpec("C2-single32", 1, 1, 32, 384, 512, 200_000, 20, 40.0, (1, 2, 3), True, 0, 0,
                 (0.9, 0.8, 0.7), 0.5, 0.3, 0.15, 0.02, "walk", False, 10),
    3: GraphSpec("C3-2x100", 2, 2, 100, 384, 512, 200_000, 20, 40.0, (1, 2, 3), False, 20, 0,
                 (0.9, 0.8, 0.7), 0.5, 0.3, 0.20, 0.02, "walk", True, 10),
    4: GraphSpec("C4-4x250", 3, 4, 250, 192, 256, 200_000, 20, 40.0, (1, 2, 3), False, 60, 0,
                 (0.9, 0.8, 0.7), 0.5, 0.3, 0.20, 0.02, "walk", False, 10),
    5: GraphSpec("C5-long2000", 4, 1, 2000, 384, 512, 200_000, 20, 40.0, (1, 2, 3), False, 0, 200,
                 (0.9, 0.8, 0.7), 0.5, 0.3, 0.20, 0.02, "walk", False, 5, (4, 8)),
}


@dataclass
class Graph:
    spec: GraphSpec
    points: np.ndarray        # [N, HW, 3] float32, keyframe's own camera frame
    conf: np.ndarray          # [N, HW] float32
    edges: np.ndarray         # [E, 2] int32, (i, j): X_j is mapped into camera i
    match: np.ndarray         # [E, HW] int32, pixel m of i -> pixel n of j, < 0 invalid
    edge_kind: np.ndarray     # [E] int8: 0 intra-sequential, 1 loop closure, 2 inter-agent
    agent: np.ndarray         # [N] int32, a(i)
    fixed_kf: np.ndarray      # int32 list of gauge keyframes
    poses_gt: np.ndarray      # [N, 8] float64
    poses_init: np.ndarray    # [N, 8] float64 (config 3: the raw start below; synchronise with meta['gauge_sync_plan'])
    poses_init_raw: Optional[np.ndarray] = None   # config 3 only: independent per-agent gauges
    segments: Optional[np.ndarray] = None         # [HW] int32 segment label grid (config 5)
    meta: Dict[str, object] = field(default_factory=dict)

    @property
    def n_kf(self) -> int:
        return self.points.shape[0]

    @property
    def hw(self) -> int:
        return self.points.shape[1]

    @property
    def n_edges(self) -> int:
        return self.edges.shape[0]


# ----------------------------------------------------------------------------------------------
def _make_scene(spec: GraphSpec) -> np.ndarray:
    rng = _rng(spec.seed, _K_SCENE)
    S, P = spec.n_scene, spec.n_planes
    pts = np.empty((S, 3))
    bounds = np.linspace(0, S, P + 1).astype(np.int64)
    for p in range(P):
        nrm = _random_unit(rng)
        off = rng.normal(0.0, 3.0)
        a = np.cross(nrm, [1.0, 0.0, 0.0] if abs(nrm[0]) < 0.9 else [0.0, 1.0, 0.0])
        a /= np.linalg.norm(a)
        b = np.cross(nrm, a)
        cnt = int(bounds[p + 1] - bounds[p])
        uv = rng.uniform(-0.5 * spec.plane_side, 0.5 * spec.plane_side, size=(cnt, 2))
        # order the ids of one plane along a raster so that consecutive ids are neighbours
        order = np.lexsort((uv[:, 0], np.floor(uv[:, 1] / (spec.plane_side / 64.0))))
        uv = uv[order]
        pts[bounds[p]:bounds[p + 1]] = off * nrm + uv[:, :1] * a + uv[:, 1:] * b
    return pts


def _make_gt_poses(spec: GraphSpec) -> np.ndarray:
    N = spec.n_kf
    poses = np.empty((N, 8))
    for a in range(spec.n_agents):
        rng = _rng(spec.seed, _K_POSE, a)
        if spec.pose_mode == "iid":
            for k in range(spec.kf_per_agent):
                poses[a * spec.kf_per_agent + k] = np.concatenate(
                    [rng.normal(0.0, 1.0, 3), _haar_quat(rng), [np.exp(rng.normal(0.0, 0.3))]])
        else:
            t = rng.normal(0.0, 1.0, 3)
            q = _haar_quat(rng)
            ls = rng.normal(0.0, 0.3)
            for k in range(spec.kf_per_agent):
                poses[a * spec.kf_per_agent + k] = np.concatenate([t, q, [np.exp(ls)]])
                t = t + 0.5 * _random_unit(rng)
                dq = _quat_from_rotvec(np.deg2rad(10.0) * _random_unit(rng))
                q = _quat_mul(dq, q)
                q /= np.linalg.norm(q)
                ls = ls + rng.normal(0.0, 0.05)
    return poses


def _scene_offsets(spec: GraphSpec) -> np.ndarray:
    """o_k: pixel m of keyframe k sees scene id (o_k + m) mod S."""
    adv = max(1, spec.hw // 16)
    o = np.empty(spec.n_kf, dtype=np.int64)
    agent_shift = min(spec.n_scene // 7, spec.hw // 4)
    for a in range(spec.n_agents):
        for k in range(spec.kf_per_agent):
            o[a * spec.kf_per_agent + k] = (a * agent_shift + k * adv) % spec.n_scene
    return o


def _make_keyframe(spec: GraphSpec, k: int, scene: np.ndarray, pose_gt: np.ndarray, o_k: int):
    rng = _rng(spec.seed, _K_KF, k)
    sid = (o_k + np.arange(spec.hw, dtype=np.int64)) % spec.n_scene
    R = _quat_to_mat(pose_gt[3:7])
    X = (scene[sid] - pose_gt[0:3]) @ R / pose_gt[7]          # R^T (p - t) / s
    X = X + rng.normal(0.0, spec.sigma_n, size=X.shape)
    c = rng.beta(5.0, 2.0, size=spec.hw)
    return X.astype(np.float32), c.astype(np.float32)


def _make_edges(spec: GraphSpec):
    edges: List[Tuple[int, int]] = []
    kind: List[int] = []
    frac: List[float] = []
    K = spec.kf_per_agent
    for a in range(spec.n_agents):
        base = a * K
        for d, vf in zip(spec.offsets, spec.valid_frac):
            for k in range(K if spec.cyclic else K - d):
                edges.append((base + k, base + (k + d) % K))
                kind.append(0)
                frac.append(vf)
    if spec.loop_every > 0:
        for k in range(spec.loop_every, spec.n_kf - spec.loop_every + 1, spec.loop_every):
            edges.append((k, k - spec.loop_every))
            kind.append(1)
            frac.append(spec.valid_frac_loop)
    if spec.n_inter > 0:
        pairs = [(a, (a + 1) % spec.n_agents) for a in range(spec.n_agents if spec.n_agents > 2 else 1)]
        per = spec.n_inter // len(pairs)
        rem = spec.n_inter - per * len(pairs)
        for pi, (a, b) in enumerate(pairs):
            cnt = per + (1 if pi < rem else 0)
            ks = np.linspace(0, K - 1, cnt + 2)[1:-1].round().astype(int)
            for k in ks:
                edges.append((a * K + int(k), b * K + int(k)))
                kind.append(2)
                frac.append(spec.valid_frac_inter)
    return (np.asarray(edges, dtype=np.int32).reshape(-1, 2), np.asarray(kind, dtype=np.int8),
            np.asarray(frac))


def _make_match(spec: GraphSpec, e: int, o_i: int, o_j: int, vf: float) -> np.ndarray:
    rng = _rng(spec.seed, _K_EDGE, e)
    HW, S = spec.hw, spec.n_scene
    m = np.arange(HW, dtype=np.int64)
    n = (o_i + m - o_j) % S                      # same scene id seen from j
    match = np.where(n < HW, n, -1).astype(np.int32)
    valid_idx = np.flatnonzero(match >= 0)
    target = int(round(vf * HW))
    if valid_idx.size > target:                  # invalidate one contiguous band of valid entries
        drop = valid_idx.size - target
        start = int(rng.integers(0, valid_idx.size - drop + 1))
        match[valid_idx[start:start + drop]] = -1
        valid_idx = np.flatnonzero(match >= 0)
    n_out = int(round(spec.p_out * valid_idx.size))
    if n_out > 0:                                # outliers: uniform random target pixels
        pick = rng.choice(valid_idx, size=n_out, replace=False)
        match[pick] = rng.integers(0, HW, size=n_out, dtype=np.int32)
    return match


def _perturb(pose: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    d = np.concatenate([rng.normal(0.0, 0.05, 3), _quat_from_rotvec(rng.normal(0.0, 0.03, 3)),
                        [np.exp(rng.normal(0.0, 0.02))]])
    return _compose(d, pose)


def make_graph(spec: GraphSpec, edges: Optional[np.ndarray] = None, valid_frac: float = 0.8) -> Graph:
    """The graph of a spec.  ``edges`` ([E, 2] keyframe pairs) replaces the spec's own edge list by an arbitrary topology
    (tests: hubs, duplicate and reversed pairs, isolated keyframes); those edges all get ``valid_frac``."""
    scene = _make_scene(spec)
    poses_gt = _make_gt_poses(spec)
    o = _scene_offsets(spec)
    N, HW = spec.n_kf, spec.hw
    points = np.empty((N, HW, 3), dtype=np.float32)
    conf = np.empty((N, HW), dtype=np.float32)
    if edges is None:
        edges, kind, frac = _make_edges(spec)
    else:
        edges = np.ascontiguousarray(edges, dtype=np.int32).reshape(-1, 2)
        assert edges.size == 0 or (edges.min() >= 0 and edges.max() < N)
        kind, frac = np.zeros(edges.shape[0], dtype=np.int8), np.full(edges.shape[0], float(valid_frac))
    E = edges.shape[0]
    match = np.empty((E, HW), dtype=np.int32)

    def fill_keyframe(k: int) -> None:
        points[k], conf[k] = _make_keyframe(spec, k, scene, poses_gt[k], int(o[k]))

    def fill_match(e: int) -> None:
        match[e] = _make_match(spec, e, int(o[edges[e, 0]]), int(o[edges[e, 1]]), float(frac[e]))

    # every keyframe / edge draws from its own stream, so the order (and the thread) does not matter; NumPy's
    # generators and gathers release the GIL
    with ThreadPoolExecutor(max_workers=_n_threads()) as pool:
        list(pool.map(fill_keyframe, range(N)))
        list(pool.map(fill_match, range(E)))
    agent = np.repeat(np.arange(spec.n_agents, dtype=np.int32), spec.kf_per_agent)

    poses_init = poses_gt.copy()
    for k in range(1, N):
        poses_init[k] = _perturb(poses_gt[k], _rng(spec.seed, _K_INIT, k))
    poses_raw = None
    sync_plan: List[Tuple[int, List[int], bool]] = []    # (linking edge, moving keyframes, moving component is i's)
    if spec.agent_gauge and spec.n_agents > 1:
        poses_raw = poses_init.copy()
        for a in range(1, spec.n_agents):
            rng = _rng(spec.seed, _K_GAUGE, a)
            G = np.concatenate([rng.normal(0.0, 2.0, 3), _haar_quat(rng),
                                [np.exp(rng.uniform(np.log(0.3), np.log(3.0)))]])
            for k in range(a * spec.kf_per_agent, (a + 1) * spec.kf_per_agent):
                poses_raw[k] = _compose(G, poses_init[k])
        # The start handed out is the RAW one: the components are brought into one gauge by the method itself
        # (sim3ba_gauge_sync on the device, oracle/gauge_sync_oracle.py in the tests), on the first
        # inter-agent edge of each moving agent, in this order.  The plan below is bookkeeping only.
        poses_init = poses_raw
        for a in range(1, spec.n_agents):
            es = [e for e in range(E) if kind[e] == 2 and
                  {int(agent[edges[e, 0]]), int(agent[edges[e, 1]])} == {a - 1, a}]
            e = es[0]
            moving = list(range(a * spec.kf_per_agent, (a + 1) * spec.kf_per_agent))
            sync_plan.append((int(e), moving, bool(agent[edges[e, 0]] == a)))

    segments = None
    if spec.n_segments[0] > 0:
        r, c = spec.n_segments
        rr = (np.arange(spec.height) * r // spec.height)[:, None]
        cc = (np.arange(spec.width) * c // spec.width)[None, :]
        segments = (rr * c + cc).astype(np.int32).reshape(-1)

    return Graph(spec=spec, points=points, conf=conf, edges=edges, match=match, edge_kind=kind,
                 agent=agent, fixed_kf=np.array([0], dtype=np.int32), poses_gt=poses_gt,
                 poses_init=poses_init, poses_init_raw=poses_raw, segments=segments,
                 meta=dict(valid_frac_target=frac, gauge_sync_plan=sync_plan))


def make_config(k: int, **scaled) -> Graph:
    """Config k of BASELINE.json (1..5); keyword overrides give a reduced variant for tests."""
    spec = CONFIGS[k]
    if scaled:
        spec = spec.scaled(**scaled)
    return make_graph(spec)


@dataclass
class DepthInputs:
    """Inputs of the segment-level structure refinement: labels, 4-adjacent pairs, Delta_gh."""
    labels: np.ndarray        # [N, HW] int32, segment label of a pixel inside its keyframe, < 0 = excluded
    n_seg: int                # segments per keyframe (segment id = k * n_seg + label)
    pairs: np.ndarray         # [P, 2] int32, unordered 4-adjacent segment pairs (g, h) of every keyframe, as segment ids
    delta: np.ndarray         # [P] float64, reference log-range difference averaged at the shared boundary
    anchor_kf: np.ndarray     # keyframes whose segments stay fixed


def _jittered_labels(H: int, W: int, rows: int, cols: int, rng: np.random.Generator) -> np.ndarray:
    """An irregular segmentation standing in for SLIC superpixels: rows x cols centres on a lattice, each jittered by up to
    +-40 % of a cell, every pixel labelled by the nearest of the 3 x 3 centres around its own cell."""
    ch, cw = H / rows, W / cols
    cy = (np.arange(rows)[:, None] + 0.5 + rng.uniform(-0.4, 0.4, (rows, cols))) * ch
    cx = (np.arange(cols)[None, :] + 0.5 + rng.uniform(-0.4, 0.4, (rows, cols))) * cw
    yy, xx = np.meshgrid(np.arange(H) + 0.5, np.arange(W) + 0.5, indexing="ij")
    r0 = np.minimum((yy / ch).astype(np.int64), rows - 1)
    c0 = np.minimum((xx / cw).astype(np.int64), cols - 1)
    best = np.full((H, W), np.inf)
    lab = np.zeros((H, W), dtype=np.int32)
    for dr in (-1, 0, 1):
        for dc in (-1, 0, 1):
            r, c = np.clip(r0 + dr, 0, rows - 1), np.clip(c0 + dc, 0, cols - 1)
            d = (yy - cy[r, c]) ** 2 + (xx - cx[r, c]) ** 2
            take = d < best
            best[take] = d[take]
            lab[take] = (r * cols + c)[take].astype(np.int32)
    return lab


def _boundary_pairs(lab: np.ndarray, logd: np.ndarray, base: int):
    """4-adjacent segment pairs (g < h, as segment ids base + label) of one keyframe and Delta_gh = mean over the pixel
    pairs straddling the shared boundary of log|X_p| - log|X_p'| (p in g, p' in h); excluded pixels (label < 0) never count."""
    keys, vals = [], []
    for a, b, da, db in ((lab[:, :-1], lab[:, 1:], logd[:, :-1], logd[:, 1:]), (lab[:-1, :], lab[1:, :], logd[:-1, :], logd[1:, :])):
        sel = (a != b) & (a >= 0) & (b >= 0)
        la, lb, d = a[sel].astype(np.int64), b[sel].astype(np.int64), (da - db)[sel]
        swap = la > lb
        lo, hi = np.where(swap, lb, la), np.where(swap, la, lb)
        keys.append(lo * (1 << 20) + hi)
        vals.append(np.where(swap, -d, d))
    keys, vals = np.concatenate(keys), np.concatenate(vals)
    uniq, inv = np.unique(keys, return_inverse=True)
    mean = np.bincount(inv, weights=vals) / np.maximum(np.bincount(inv), 1)
    pairs = np.stack([base + uniq // (1 << 20), base + uniq % (1 << 20)], axis=1).astype(np.int32)
    return pairs, mean


def make_depth_inputs(g: Graph, grid=None, drop_frac: float = 0.02, irregular: int = 0) -> DepthInputs:
    """Stands in for the SLIC segmentation of PAPER.md:126.  Default: a rows x cols grid of rectangular segments per
    keyframe (config 5: 4 x 8 = 32).  ``irregular = M`` (the paper: M_k ~ 200): about M jittered-lattice superpixels per
    keyframe, eight seeded layouts dealt round-robin over the keyframes.  A seeded fraction of pixels is excluded (label
    -1, "low confidence"); the pairs are the 4-adjacent segment pairs found in the label image and Delta_gh the mean over
    the pixel pairs straddling the shared boundary of log|X_p| - log|X_p'| (p in g, p' in h)."""
    H, W = g.spec.height, g.spec.width
    if irregular > 0:
        r = max(1, int(round(np.sqrt(irregular * H / W))))
        c = max(1, -(-irregular // r))
        layouts = [_jittered_labels(H, W, r, c, _rng(g.spec.seed, 10, q)) for q in range(min(8, g.n_kf))]
    else:
        r, c = grid if grid is not None else (g.spec.n_segments if g.spec.n_segments[0] > 0 else (4, 8))
        rr = (np.arange(H) * r // H)[:, None]
        cc = (np.arange(W) * c // W)[None, :]
        layouts = [(rr * c + cc).astype(np.int32)]
    n_seg = r * c
    labels = np.empty((g.n_kf, H * W), dtype=np.int32)
    pairs: List[Optional[np.ndarray]] = [None] * g.n_kf
    delta: List[Optional[np.ndarray]] = [None] * g.n_kf

    def one_keyframe(k: int) -> None:
        lab = layouts[k % len(layouts)].copy()
        lab.reshape(-1)[_rng(g.spec.seed, 9, k).random(H * W) < drop_frac] = -1
        labels[k] = lab.reshape(-1)
        logd = np.log(np.maximum(np.linalg.norm(g.points[k].astype(np.float64), axis=1), 1e-12)).reshape(H, W)
        pairs[k], delta[k] = _boundary_pairs(lab, logd, k * n_seg)

    with ThreadPoolExecutor(max_workers=_n_threads()) as pool:
        list(pool.map(one_keyframe, range(g.n_kf)))
    return DepthInputs(labels=labels, n_seg=n_seg, pairs=np.concatenate(pairs).astype(np.int32).reshape(-1, 2),
                       delta=np.concatenate(delta).astype(np.float64), anchor_kf=g.fixed_kf.copy())


def clean_variant(spec: GraphSpec) -> GraphSpec:
    """Noise-free, outlier-free variant (pins: zero residual/gradient at ground truth)."""
    return replace(spec, sigma_n=0.0, p_out=0.0)
