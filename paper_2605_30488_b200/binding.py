"""ctypes binding of libsim3ba.so (include/sim3ba.h).  Argument marshalling only: every step of the
hot path runs in the library's CUDA kernels.  PyTorch provides device memory and streams.

There is no fallback: if the shared library is missing or no CUDA device is present, loading or
``Sim3BA(...)`` raises."""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsim3ba.so")

EXPORTS = (
    "sim3ba_default_params", "sim3ba_create", "sim3ba_destroy", "sim3ba_set_params", "sim3ba_set_poses",
    "sim3ba_get_poses", "sim3ba_build_system", "sim3ba_solve", "sim3ba_step", "sim3ba_step_graph", "sim3ba_step_host", "sim3ba_optimize_host", "sim3ba_refine_host", "sim3ba_gauge_sync", "sim3ba_gauge_sync_static", "sim3ba_depth_default_params", "sim3ba_depth_refine", "sim3ba_apply_depth",
    "sim3ba_retract", "sim3ba_get_edge_stats", "sim3ba_get_edge_blocks", "sim3ba_get_system",
    "sim3ba_get_update", "sim3ba_get_bookkeeping", "sim3ba_load_system", "sim3ba_get_launch_count",
    "sim3ba_set_solver_mode", "sim3ba_get_solver_info", "sim3ba_get_bb_info",
    "sim3ba_set_profiling", "sim3ba_get_phase_ms", "sim3ba_get_solve_phase_us", "sim3ba_release_memory", "sim3ba_probe_fp64", "sim3ba_copy_d2d", "sim3ba_last_error", "sim3ba_version",
)


class Params(C.Structure):
    _fields_ = [("sigma_ray", C.c_float), ("sigma_dist", C.c_float), ("huber_k", C.c_float),
                ("conf_min", C.c_float), ("lm_lambda", C.c_double), ("eps0", C.c_double),
                ("max_attempts", C.c_int32), ("reserved", C.c_int32)]


class DepthParams(C.Structure):
    _fields_ = [("sigma_point", C.c_float), ("huber_k", C.c_float), ("lambda_smooth", C.c_double),
                ("lambda_prior", C.c_double), ("lambda_lm", C.c_double), ("eta_max", C.c_double)]


class Sim3BAError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libsim3ba error {code}: {msg}")
        self.code = code


_lib = None


def load_library() -> C.CDLL:
    """dlopen libsim3ba.so (built in-tree by ``python -m paper_2605_30488_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2605_30488_b200.build` "
                           "(libsim3ba has no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    P = C.POINTER
    sig = {
        "sim3ba_default_params": [P(Params)],
        "sim3ba_create": [P(vp), i32, i32, i32, i32, vp, vp, vp, vp, P(i32), i32, P(Params), vp],
        "sim3ba_destroy": [vp],
        "sim3ba_set_params": [vp, P(Params)],
        "sim3ba_set_poses": [vp, vp],
        "sim3ba_get_poses": [vp, vp],
        "sim3ba_build_system": [vp],
        "sim3ba_solve": [vp],
        "sim3ba_step": [vp],
        "sim3ba_step_graph": [vp, i32],
        "sim3ba_step_host": [vp, vp, vp, vp],
        "sim3ba_optimize_host": [i32, i32, i32, i32, vp, vp, vp, vp, P(i32), i32, P(Params), vp, i32, vp, vp, vp],
        "sim3ba_refine_host": [i32, i32, i32, i32, vp, vp, vp, vp, P(i32), i32, P(Params), vp, i32, P(i32), P(C.c_double), i32, P(DepthParams),
                               i32, i32, i32, vp, vp, vp, vp, vp, vp],
        "sim3ba_gauge_sync": [vp, i32, P(i32), i32, i32, i32, P(C.c_double), P(i32), P(i32)],
        "sim3ba_gauge_sync_static": [vp, i32, vp, i32, i32, i32, vp],
        "sim3ba_depth_default_params": [P(DepthParams)],
        "sim3ba_depth_refine": [vp, vp, i32, P(i32), P(C.c_double), i32, P(i32), i32, P(DepthParams), i32, vp, P(C.c_double)],
        "sim3ba_apply_depth": [vp, vp, vp, vp, i32, vp],
        "sim3ba_retract": [vp],
        "sim3ba_get_edge_stats": [vp, P(vp), P(vp), P(vp)],
        "sim3ba_get_edge_blocks": [vp, P(vp)],
        "sim3ba_get_system": [vp, P(vp), P(i32), P(vp)],
        "sim3ba_get_update": [vp, P(vp), P(i32), P(C.c_double), P(C.c_double)],
        "sim3ba_get_bookkeeping": [vp, P(vp), P(vp), P(i32), P(vp), P(vp), P(vp)],
        "sim3ba_load_system": [vp, vp, vp],
        "sim3ba_get_launch_count": [vp, P(i64)],
        "sim3ba_set_solver_mode": [vp, i32],
        "sim3ba_get_solver_info": [vp, P(i32), P(i32), P(C.c_double), P(i32)],
        "sim3ba_get_bb_info": [vp, P(i32)],
        "sim3ba_set_profiling": [vp, i32],
        "sim3ba_get_phase_ms": [vp, P(C.c_float)],
        "sim3ba_get_solve_phase_us": [vp, P(C.c_float)],
        "sim3ba_release_memory": [],
        "sim3ba_probe_fp64": [P(C.c_double), P(C.c_double), vp],
        "sim3ba_copy_d2d": [vp, vp, vp, C.c_uint64],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = C.c_int
    lib.sim3ba_last_error.argtypes = [vp]
    lib.sim3ba_last_error.restype = C.c_char_p
    lib.sim3ba_version.argtypes = []
    lib.sim3ba_version.restype = C.c_char_p
    _lib = lib
    return lib


def make_params(sigma_ray=0.003, sigma_dist=10.0, huber_k=1.345, conf_min=0.0, lm_lambda=0.0, eps0=1e-6,
                max_attempts=6) -> Params:
    return Params(sigma_ray, sigma_dist, huber_k, conf_min, lm_lambda, eps0, max_attempts, 0)


def optimize_host(points, conf, edges, match, fixed_kf: Sequence[int], params: Optional[Params], height: int, width: int,
                  poses_in, n_iters: int, poses_out, cost_out=None, stream: int = 0):
    """sim3ba_optimize_host: the whole job with HOST (CPU, pinned recommended) torch tensors -- graph upload, create,
    n_iters GN steps, poses (and per-iteration costs) back.  Argument marshalling only."""
    lib = load_library()
    for t in (points, conf, edges, match, poses_in, poses_out):
        assert t.device.type == "cpu" and t.is_contiguous()
    fk = (C.c_int32 * max(1, len(fixed_kf)))(*fixed_kf)
    prm = params if params is not None else make_params()
    rc = lib.sim3ba_optimize_host(points.shape[0], height, width, edges.shape[0], points.data_ptr(), conf.data_ptr(),
                                  edges.data_ptr(), match.data_ptr(), fk, len(fixed_kf), C.byref(prm), poses_in.data_ptr(),
                                  n_iters, poses_out.data_ptr(), cost_out.data_ptr() if cost_out is not None else None,
                                  stream)
    if rc:
        raise Sim3BAError(rc, (lib.sim3ba_last_error(None) or b"").decode())


def refine_host(points, conf, edges, match, fixed_kf: Sequence[int], params: Optional[Params], height: int, width: int, labels, n_seg: int,
                pairs: np.ndarray, delta: np.ndarray, depth_params: Optional[DepthParams], n_rounds: int, n_depth_iters: int, n_pose_iters: int,
                poses_in, poses_out, eta, pose_cost=None, depth_cost=None, stream: int = 0):
    """sim3ba_refine_host: the pose-depth alternation as one job with HOST (CPU, pinned recommended) torch tensors; eta
    [N * n_seg] float64 is updated in place.  Argument marshalling only."""
    lib = load_library()
    for t in (points, conf, edges, match, labels, poses_in, poses_out, eta):
        assert t.device.type == "cpu" and t.is_contiguous()
    fk = (C.c_int32 * max(1, len(fixed_kf)))(*fixed_kf)
    prm = params if params is not None else make_params()
    dprm = depth_params
    if dprm is None:
        dprm = DepthParams()
        lib.sim3ba_depth_default_params(C.byref(dprm))
    pr = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    dl = np.ascontiguousarray(delta, dtype=np.float64).reshape(-1)
    rc = lib.sim3ba_refine_host(points.shape[0], height, width, edges.shape[0], points.data_ptr(), conf.data_ptr(), edges.data_ptr(),
                                match.data_ptr(), fk, len(fixed_kf), C.byref(prm), labels.data_ptr(), int(n_seg),
                                pr.ctypes.data_as(C.POINTER(C.c_int32)), dl.ctypes.data_as(C.POINTER(C.c_double)), pr.shape[0], C.byref(dprm),
                                int(n_rounds), int(n_depth_iters), int(n_pose_iters), poses_in.data_ptr(), poses_out.data_ptr(), eta.data_ptr(),
                                pose_cost.data_ptr() if pose_cost is not None else None,
                                depth_cost.data_ptr() if depth_cost is not None else None, stream)
    if rc:
        raise Sim3BAError(rc, (lib.sim3ba_last_error(None) or b"").decode())


def probe_fp64(stream: int = 0):
    """sim3ba_probe_fp64: measured (DFMA, DMMA) TFLOP/s of the current device."""
    lib = load_library()
    a, b = C.c_double(), C.c_double()
    rc = lib.sim3ba_probe_fp64(C.byref(a), C.byref(b), stream)
    if rc:
        raise Sim3BAError(rc, (lib.sim3ba_last_error(None) or b"").decode())
    return a.value, b.value


def release_memory():
    """sim3ba_release_memory: give the library pool's unused device memory back to the driver."""
    rc = load_library().sim3ba_release_memory()
    if rc:
        raise Sim3BAError(rc, "sim3ba_release_memory")


class Sim3BA:
    """One Sim(3) pose graph resident on the GPU (sim3ba_create ... sim3ba_destroy)."""

    def __init__(self, points, conf, edges, match, fixed_kf: Sequence[int], params: Optional[Params] = None,
                 height: Optional[int] = None, width: Optional[int] = None, stream=None):
        import torch
        self._torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libsim3ba has no CPU fallback")
        for t, dt, nm in ((points, torch.float32, "points"), (conf, torch.float32, "conf"),
                          (edges, torch.int32, "edges"), (match, torch.int32, "match")):
            if not (t.is_cuda and t.dtype == dt and t.is_contiguous()):
                raise ValueError(f"{nm} must be a contiguous CUDA tensor of dtype {dt}")
        self.N, self.HW = int(points.shape[0]), int(points.shape[1])
        self.E = int(edges.shape[0])
        if height is None or width is None:
            height, width = 1, self.HW
        assert height * width == self.HW and tuple(points.shape) == (self.N, self.HW, 3)
        assert tuple(conf.shape) == (self.N, self.HW) and (self.E == 0 or tuple(match.shape) == (self.E, self.HW))
        self.n = 7 * self.N
        self.device = points.device
        self._match = match  # borrowed by the library: keep alive
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        fixed = np.asarray(list(fixed_kf), dtype=np.int32)
        self.params = params if params is not None else make_params()
        self._h = C.c_void_p()
        rc = self.lib.sim3ba_create(C.byref(self._h), self.N, height, width, self.E, points.data_ptr(),
                                    conf.data_ptr(), edges.data_ptr() if self.E else None,
                                    match.data_ptr() if self.E else None,
                                    fixed.ctypes.data_as(C.POINTER(C.c_int32)), int(fixed.size),
                                    C.byref(self.params), C.c_void_p(self._stream.cuda_stream))
        if rc != 0:
            raise Sim3BAError(rc, self.lib.sim3ba_last_error(None).decode())

    # ------------------------------------------------------------------ helpers
    def _check(self, rc: int):
        if rc != 0:
            raise Sim3BAError(rc, self.lib.sim3ba_last_error(self._h).decode())

    def _fetch(self, ptr, shape, dtype):
        torch = self._torch
        out = torch.empty(shape, dtype=dtype, device=self.device)
        self._check(self.lib.sim3ba_copy_d2d(self._h, out.data_ptr(), ptr, out.numel() * out.element_size()))
        return out

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self.lib.sim3ba_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ the C ABI, one to one
    def set_params(self, params: Params):
        self._check(self.lib.sim3ba_set_params(self._h, C.byref(params)))
        self.params = params

    def set_poses(self, poses):
        assert poses.is_cuda and poses.dtype == self._torch.float64 and poses.is_contiguous() and tuple(poses.shape) == (self.N, 8)
        self._check(self.lib.sim3ba_set_poses(self._h, poses.data_ptr()))

    def get_poses(self):
        out = self._torch.empty((self.N, 8), dtype=self._torch.float64, device=self.device)
        self._check(self.lib.sim3ba_get_poses(self._h, out.data_ptr()))
        return out

    def build_system(self):
        self._check(self.lib.sim3ba_build_system(self._h))

    def solve(self):
        self._check(self.lib.sim3ba_solve(self._h))

    def step(self):
        self._check(self.lib.sim3ba_step(self._h))

    def step_graph(self, n_steps: int = 1):
        """n_steps GN iterations as one CUDA-graph launch (sim3ba_step_graph)."""
        self._check(self.lib.sim3ba_step_graph(self._h, int(n_steps)))

    def gauge_sync(self, edge: int, moving_kf: Sequence[int], moving_is_i: bool = False, n_c_min: int = 64):
        """sim3ba_gauge_sync on the current poses; returns (T* as an 8-vector pose, N_c, fallback used)."""
        mk = (C.c_int32 * max(1, len(moving_kf)))(*[int(k) for k in moving_kf])
        T = (C.c_double * 8)()
        nc, fb = C.c_int32(), C.c_int32()
        self._check(self.lib.sim3ba_gauge_sync(self._h, int(edge), mk, len(moving_kf), int(bool(moving_is_i)), int(n_c_min), T,
                                               C.byref(nc), C.byref(fb)))
        return np.array(list(T)), nc.value, bool(fb.value)

    def gauge_sync_static(self, edge: int, moving_kf, result, moving_is_i: bool = False, n_c_min: int = 64):
        """sim3ba_gauge_sync_static: the same operation with no device allocation (scratch in a file-scope device array,
        images up to 2^18 pixels).  moving_kf: CUDA int32 tensor of keyframe indices (or None); result: CUDA float64 tensor
        [10], written asynchronously on the context's stream (T* [8], N_c, fallback flag)."""
        t = self._torch
        assert result.is_cuda and result.dtype == t.float64 and result.is_contiguous() and result.numel() >= 10
        n_moving = 0 if moving_kf is None else int(moving_kf.numel())
        if n_moving:
            assert moving_kf.is_cuda and moving_kf.dtype == t.int32 and moving_kf.is_contiguous()
        self._check(self.lib.sim3ba_gauge_sync_static(self._h, int(edge), moving_kf.data_ptr() if n_moving else None, n_moving,
                                                      int(bool(moving_is_i)), int(n_c_min), result.data_ptr()))

    def depth_refine(self, labels, n_seg: int, pairs: np.ndarray, delta: np.ndarray, anchor_kf: Sequence[int], eta, n_iters: int = 10,
                     params: Optional[DepthParams] = None):
        """sim3ba_depth_refine: labels int32 [N,HW] and eta float64 [N*n_seg] are CUDA tensors (eta updated in place);
        pairs [P,2] int32 / delta [P] float64 are NumPy host arrays.  Returns the objective at the start of each iteration."""
        t = self._torch
        assert labels.is_cuda and labels.dtype == t.int32 and labels.is_contiguous() and tuple(labels.shape) == (self.N, self.HW)
        assert eta.is_cuda and eta.dtype == t.float64 and eta.is_contiguous() and eta.numel() == self.N * n_seg
        prm = params
        if prm is None:
            prm = DepthParams()
            self._check(self.lib.sim3ba_depth_default_params(C.byref(prm)))
        pr = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
        dl = np.ascontiguousarray(delta, dtype=np.float64).reshape(-1)
        ak = (C.c_int32 * max(1, len(anchor_kf)))(*[int(k) for k in anchor_kf])
        cost = (C.c_double * max(1, n_iters))()
        self._check(self.lib.sim3ba_depth_refine(self._h, labels.data_ptr(), int(n_seg), pr.ctypes.data_as(C.POINTER(C.c_int32)),
                                                 dl.ctypes.data_as(C.POINTER(C.c_double)), pr.shape[0], ak, len(anchor_kf), C.byref(prm),
                                                 int(n_iters), eta.data_ptr(), cost))
        return np.array(list(cost)[:n_iters])

    def apply_depth(self, points, conf, labels, n_seg: int, eta):
        """sim3ba_apply_depth: re-pack the pointmaps scaled by exp(eta) of each pixel's segment."""
        self._check(self.lib.sim3ba_apply_depth(self._h, points.data_ptr(), conf.data_ptr(), labels.data_ptr(), int(n_seg), eta.data_ptr()))

    def retract(self):
        self._check(self.lib.sim3ba_retract(self._h))

    def step_host(self, h_poses_in=None, h_poses_out=None, want_cost: bool = False):
        """h_poses_* are CPU float64 tensors [N,8] (pinned recommended)."""
        cost = C.c_double(0.0)
        self._check(self.lib.sim3ba_step_host(
            self._h, h_poses_in.data_ptr() if h_poses_in is not None else None,
            h_poses_out.data_ptr() if h_poses_out is not None else None,
            C.cast(C.byref(cost), C.c_void_p) if want_cost else None))
        return cost.value if want_cost else None

    def edge_stats(self):
        nv, ck, co = C.c_void_p(), C.c_void_p(), C.c_void_p()
        self._check(self.lib.sim3ba_get_edge_stats(self._h, C.byref(nv), C.byref(ck), C.byref(co)))
        t = self._torch
        return (self._fetch(nv, (self.E,), t.int32), self._fetch(ck, (self.E,), t.int64),
                self._fetch(co, (self.E,), t.float64))

    def edge_blocks(self):
        p = C.c_void_p()
        self._check(self.lib.sim3ba_get_edge_blocks(self._h, C.byref(p)))
        return self._fetch(p, (self.E, 35), self._torch.float64)

    def system(self):
        """(H [7N,7N] lower triangle, g [7N]) of the last build_system, as new tensors."""
        ph, pg, ld = C.c_void_p(), C.c_void_p(), C.c_int32()
        self._check(self.lib.sim3ba_get_system(self._h, C.byref(ph), C.byref(ld), C.byref(pg)))
        Hp = self._fetch(ph, (ld.value, ld.value), self._torch.float64)
        return Hp[: self.n, : self.n].contiguous(), self._fetch(pg, (self.n,), self._torch.float64)

    def update(self):
        pt, att, eps, cost = C.c_void_p(), C.c_int32(), C.c_double(), C.c_double()
        self._check(self.lib.sim3ba_get_update(self._h, C.byref(pt), C.byref(att), C.byref(eps), C.byref(cost)))
        return self._fetch(pt, (self.n,), self._torch.float64), att.value, eps.value, cost.value

    def bookkeeping(self) -> Dict[str, np.ndarray]:
        a, b, c, d, e = (C.c_void_p() for _ in range(5))
        npairs = C.c_int32()
        self._check(self.lib.sim3ba_get_bookkeeping(self._h, C.byref(a), C.byref(b), C.byref(npairs),
                                                    C.byref(c), C.byref(d), C.byref(e)))

        def arr(p, n):
            if n == 0:
                return np.zeros(0, dtype=np.int32)
            return np.ctypeslib.as_array(C.cast(p, C.POINTER(C.c_int32)), shape=(n,)).copy()

        P = npairs.value
        return dict(kf_ptr=arr(a, self.N + 1), kf_edge=arr(b, 2 * self.E), pair_kf=arr(c, 2 * P).reshape(-1, 2),
                    pair_ptr=arr(d, P + 1), pair_edge=arr(e, self.E))

    def load_system(self, H, g):
        t = self._torch
        assert H.is_cuda and H.dtype == t.float64 and H.is_contiguous() and tuple(H.shape) == (self.n, self.n)
        assert g.is_cuda and g.dtype == t.float64 and g.is_contiguous() and tuple(g.shape) == (self.n,)
        self._check(self.lib.sim3ba_load_system(self._h, H.data_ptr(), g.data_ptr()))

    def set_solver_mode(self, mode: int):
        """2: band + border block Cholesky (default); 0: tile-sparse plan of the graph; 1: dense plan (every lower tile)."""
        self._check(self.lib.sim3ba_set_solver_mode(self._h, int(mode)))

    def solver_info(self) -> Dict[str, float]:
        nt, ntd, fl, gr = C.c_int32(), C.c_int32(), C.c_double(), C.c_int32()
        self._check(self.lib.sim3ba_get_solver_info(self._h, C.byref(nt), C.byref(ntd), C.byref(fl), C.byref(gr)))
        return dict(n_tiles=nt.value, n_tiles_dense=ntd.value, flops=fl.value, grid=gr.value)

    def bb_info(self) -> Dict[str, int]:
        """Band + border plan of the graph (solver mode 2)."""
        info = (C.c_int32 * 8)()
        self._check(self.lib.sim3ba_get_bb_info(self._h, info))
        return dict(zip(("valid", "n_interior", "n_segments", "n_border", "max_segment", "max_segment_border", "n_groups_level2",
                         "n_border_dense"), list(info)))

    def launch_count(self) -> int:
        n = C.c_int64()
        self._check(self.lib.sim3ba_get_launch_count(self._h, C.byref(n)))
        return n.value

    def set_profiling(self, on: bool):
        self._check(self.lib.sim3ba_set_profiling(self._h, 1 if on else 0))

    def phase_ms(self) -> Tuple[float, ...]:
        buf = (C.c_float * 8)()
        self._check(self.lib.sim3ba_get_phase_ms(self._h, buf))
        return tuple(buf)

    def solve_phase_us(self) -> Tuple[float, ...]:
        buf = (C.c_float * 8)()
        self._check(self.lib.sim3ba_get_solve_phase_us(self._h, buf))
        return tuple(buf)
