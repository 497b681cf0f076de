"""sim3ba: B200-native Gauss-Newton step of the unified multi-agent Sim(3) pose graph over dense
pointmap correspondences (CoMo3R-SLAM, arxiv 2605.30488, section III-D).

The product is ``libsim3ba.so`` (hand-written CUDA for sm_100a behind the C ABI of
``include/sim3ba.h``); this package is the thin ctypes binding.  No CPU fallback exists."""
from .binding import DepthParams, EXPORTS, LIB_PATH, Params, Sim3BA, Sim3BAError, load_library, make_params, optimize_host, probe_fp64, refine_host, release_memory  # noqa: F401
