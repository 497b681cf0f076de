// Internal context and kernel launchers of libsim3ba (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <string>
#include <vector>

#include "../../include/sim3ba.h"

namespace sim3ba {

// Device memory of the library comes from a stream-ordered memory pool OWNED BY THE LIBRARY (one per device, created on
// first use, release threshold = keep everything until sim3ba_release_memory), on the stream of the running API call
// (set on entry of every entry point that may allocate or free): no device-wide synchronisation per allocation, a warm
// pool costs no map / unmap per context, and the device's default pool (PyTorch's, the caller's) is left alone.
inline thread_local cudaStream_t tl_stream = nullptr;
cudaError_t lib_pool(cudaMemPool_t* pool);          // the library's pool on the current device (sim3ba_api.cu)
inline cudaError_t dmalloc(void** p, size_t bytes) {
  cudaMemPool_t pool;
  cudaError_t e = lib_pool(&pool);
  if (e != cudaSuccess) return e;
  return cudaMallocFromPoolAsync(p, bytes < 16 ? 16 : bytes, pool, tl_stream);
}
inline void dfree(void* p) { if (p) cudaFreeAsync(p, tl_stream); }

constexpr int kAccThreads = 32;      // accumulate CTA: ONE warp -- warps are independent workers, so the finest CTA gives the block
                                     // scheduler the finest grain (a two-warp CTA holds its slot until the slower warp is done)
constexpr int kTilePx = 16 * kAccThreads;   // pixels of a keyframe handled by one accumulate CTA (512 contiguous per warp)
// doubles per (edge, 512-pixel warp slice) partial record: [0..27] upper triangle of M = sum J_xi^T Omega J_xi (row-major,
// r <= c; (3,6), (4,6), (5,6) are structurally zero), [28..34] c = sum J_xi^T Omega e, [35] sum w r^2,
// [36] sum min(r^2, kappa^2) (robust cost = [35] - [36]/2), [37] n_valid (int64 bits), [38] checksum (uint64 bits),
// [39] ballot of the lanes of kernel 1 holding DEFERRED matches (int64 bits; 0 almost always): matches whose x = X_i + delta
// cancels (|x| << |X_i|) are left out of kernel 1's fp32 sums and evaluated in FP64 by k_deferred; their per-lane 16-bit masks
// go to Ctx::def_masks, the edge is marked in Ctx::def_flag
constexpr int kPartialStride = 40;
constexpr int kSlotCnt = 37, kSlotChk = 38, kSlotDef = 39;
constexpr int kNB = 64;              // Cholesky block size

struct DevParams {       // robust-kernel constants, fp32, passed by value to kernel 1
  float inv_var_ray;     // 1 / sigma_r^2
  float inv_var_dist;    // 1 / sigma_d^2
  float k_over_sigma_ray;   // kappa / sigma_r
  float k_over_sigma_dist;  // kappa / sigma_d
  float huber_k2;
};

// Tile-level plan of the Cholesky factorisation (a7), built once per graph on the host (a0): the
// non-zero 64x64 tiles of L (symbolic factorisation of the keyframe graph, fill included) as
// column lists (rows i > k with a non-zero tile (i, k)) and row lists (columns j < k), plus the list
// of all non-zero tiles for the assembly.  The "dense" plan lists every lower tile.
struct SolvePlan {
  int nb = 0, n_tiles = 0, n_off = 0, max_col = 0, max_row = 0, max_upd = 0, grid = 1;
  double flops = 0.0;                                   // tile-level flop count of factor + solves
  int32_t *col_ptr = nullptr, *col_rows = nullptr, *row_ptr = nullptr, *row_cols = nullptr, *tiles = nullptr;
  std::vector<int32_t> h_col_ptr, h_col_rows, h_row_ptr, h_row_cols, h_tiles;
  bool ready = false;
};

// Band + border plan of the block (7x7) Cholesky (a7, solver mode 2), built once per graph on the host (a0).
// Free keyframes are split into BORDER keyframes -- one endpoint of every edge longer than kBand in keyframe
// index (loop closures, inter-agent links), plus separator triples that cap the length of a chain -- and
// INTERIOR keyframes, which form independent SEGMENTS: runs in temporal order whose coupling stays inside a
// block band of kBand.  A segment is eliminated sequentially by one CTA at 7x7 granularity (block column =
// diagonal block, <= kBand band blocks, one block per border keyframe of the segment); the Schur
// complement on the border keyframes is a small dense system for the tile Cholesky; the interior
// update follows by back-substitution.  Same tau as the tile plans up to rounding.
constexpr int kBand = 3;          // block band of a chain (edges (k, k+1..k+3))
constexpr int kMaxSegBorder = 28; // border keyframes one segment may touch (else the plan is not used)
// Further levels of the band + border plan: the Schur complement S on the border keyframes is itself sparse -- a separator
// group (the <= kBand keyframes of a cut) is coupled only to the groups and long-link keyframes that share a segment with
// it.  An independent set of separator groups (no two of them coupled in S) is eliminated from S exactly like the
// segments were from H -- each group a "segment" of <= kBand columns whose blocks are read out of S -- which leaves a
// smaller S' on which the groups that stayed are coupled to their new neighbours: the next level does the same to S', and
// the dense tiled Cholesky runs on what the last level leaves.  Same array roles as in BBPlan; "keyframe" of a column /
// of a border entry of a level is a BORDER INDEX OF THE LEVEL BEFORE.
struct BBLevel2 {
  bool valid = false;
  int n_int = 0, n_seg = 0, n_bord = 0, max_nb = 0, max_len = 0, npadB = 0;
  double flops_saved = 0.0;
  int32_t *seg_ptr = nullptr, *seg_bptr = nullptr, *seg_bord = nullptr, *col_kf = nullptr, *col_nb = nullptr, *bord_kf = nullptr;
  int32_t *bord_sptr = nullptr, *bord_seg = nullptr, *bord_slot = nullptr;
  int64_t* col_ofs = nullptr;
  double *colbuf = nullptr, *seg_rhs = nullptr, *LB = nullptr, *rhsB = nullptr, *ysolB = nullptr, *DinvB = nullptr, *tauB = nullptr;
  SolvePlan dense;
};

struct BBPlan {
  bool ready = false, valid = false;
  static constexpr int kMaxLevels = 3;   // further levels behind the first (each eliminates an independent set of the separator groups left)
  BBLevel2 lv[kMaxLevels];
  int n_lv = 0;
  int n_int = 0, n_seg = 0, n_bord = 0, max_nb = 0, max_len = 0;
  int npadB = 0;                  // padded size of the border system (multiple of kNB), 0 if no border
  size_t col_doubles = 0;         // doubles of all interior block columns
  double flops = 0.0;             // flop count of the plan (factor + solves, 7x7 granularity; border system dense)
  // device arrays
  int32_t *seg_ptr = nullptr;     // [n_seg+1] interior columns of a segment (indices into col_*)
  int32_t *seg_bptr = nullptr;    // [n_seg+1] into seg_bord
  int32_t *seg_bord = nullptr;    // border keyframes of a segment, as border indices (ascending)
  int32_t *col_kf = nullptr;      // [n_int] keyframe of an interior column
  int32_t *col_nb = nullptr;      // [n_int] border keyframes of the column's segment
  int64_t *col_ofs = nullptr;     // [n_int] offset (doubles) of the column in colbuf
  int32_t *col_band = nullptr;    // [n_int][kBand] pair index of block (column c + 1 + a, column c), -1 if none / outside
  int32_t *col_bpair = nullptr;   // [sum len * nb] pair index of block (border keyframe, column), -1 if none
  int64_t *col_bofs = nullptr;    // [n_int] offset into col_bpair
  int32_t *bord_kf = nullptr;     // [n_bord] keyframe of a border index (ascending)
  int32_t *bord_sptr = nullptr;   // [n_bord+1] segments touching a border keyframe ...
  int32_t *bord_seg = nullptr;    //   ... segment id
  int32_t *bord_slot = nullptr;   //   ... position of the keyframe in the segment's border list
  int32_t *bb_pair = nullptr;     // [n_bord][n_bord] pair index of block (border a, border b), b < a, -1 if none
  // device work buffers
  double *colbuf = nullptr;       // interior block columns: [D 49][band kBand*49][border nb*49][rhs 7] per column
  double *seg_rhs = nullptr;      // [sum nb * 7] per-segment contribution sum_c F_c y_c to the border right-hand side
  double *LB = nullptr, *rhsB = nullptr, *ysolB = nullptr, *DinvB = nullptr, *tauB = nullptr;
  SolvePlan dense;                // dense tile plan of the border system
  std::vector<int32_t> h_seg_ptr, h_seg_bptr;
};

struct Ctx {
  int N = 0, H = 0, W = 0, HW = 0, E = 0, n = 0, npad = 0, chunks = 0, n_pairs = 0;
  cudaStream_t stream = nullptr;
  sim3ba_params prm{};
  // inputs
  float4* pm = nullptr;            // [N][HW] packed (x, y, z, w): w = c^(1/4) if c > conf_min else -1
  float4* pm0 = nullptr;           // pristine copy of pm, taken by the first sim3ba_apply_depth (NULL until then: pm is pristine)
  size_t depth_smem = 0;           // dynamic shared memory k_depth_edge has been opted in for
  const int32_t* match = nullptr;  // borrowed [E][HW]
  int32_t* edges = nullptr;        // [E][2]
  // kernel-1 schedule: keyframes with outgoing edges (ascending) and their edges (ascending j, then e)
  int32_t *grp_kf = nullptr, *grp_ptr = nullptr, *grp_edge = nullptr;
  int n_groups = 0;
  double* edgeT = nullptr;         // [E][12] s_ij R_ij, t_ij of the current poses (a1)
  uint8_t* fixed_mask = nullptr;   // [N]
  double* poses = nullptr;         // [N][8]
  // bookkeeping (device + host)
  int32_t *kf_ptr = nullptr, *kf_edge = nullptr, *pair_kf = nullptr, *pair_ptr = nullptr, *pair_edge = nullptr;
  int32_t* pairhi_ptr = nullptr;   // [N+1] first pair whose larger keyframe is >= k (pairs are sorted by (hi, lo))
  std::vector<int32_t> h_edges, h_kf_ptr, h_kf_edge, h_pair_kf, h_pair_ptr, h_pair_edge, h_pairhi_ptr;
  SolvePlan plan_sparse, plan_dense;
  BBPlan plan_bb;
  int solver_mode = 2;             // 0: tile-sparse plan of the graph, 1: dense plan (every lower tile), 2: band + border (falls back to 0)
  std::vector<uint8_t> h_fixed;
  // per-edge results
  double* partials = nullptr;      // [E][chunks * warps per CTA][kPartialStride]: one record per (edge, 512-pixel slice)
  double* def_sums = nullptr;      // [E][40]: FP64 sums over the deferred matches of an edge (k_deferred), slots as in a record
  unsigned short* def_masks = nullptr;   // [E][records][32]: per record and lane of kernel 1, the 16-bit mask of its deferred matches (written only where a record has some)
  int32_t* def_flag = nullptr;     // [E]: non-zero if the edge has deferred matches at the current poses (zeroed by k_edge_prep)
  double* blocks35 = nullptr;      // [E][35]
  double* edge_cost = nullptr;     // [E]
  int32_t* n_valid = nullptr;      // [E]
  unsigned long long* checksum = nullptr;  // [E]
  // dense system
  double* Hd = nullptr;            // [npad][npad] undamped (API read-back)
  double* L = nullptr;             // [npad][npad] working copy, factorised in place
  double* g = nullptr;             // [npad]
  double* rhs = nullptr;           // [npad] working right-hand side b (starts as -g)
  double* ysol = nullptr;          // [npad] y = L^-1 b, then consumed by the backward solve
  double* Dinv = nullptr;          // [npad] reciprocals of the diagonal of L
  double* tau = nullptr;           // [npad]
  double* total_cost = nullptr;    // [1]
  int32_t* fail_flag = nullptr;    // [4] device: [0] failure flag, [1] attempts used, [2] solved
  double* d_eps_used = nullptr;    // [1] device
  unsigned int* bar = nullptr;     // [1] device: grid-barrier counter of k_solve
  unsigned long long* solve_stamps = nullptr;   // [16] device: globaltimer stamps of the phases of k_solve_bb (profiling only)
  int32_t* h_flag = nullptr;       // pinned
  double* h_scalar = nullptr;      // pinned [4]
  bool built = false, solved = false, dense_loaded = false, hd_valid = false, status_stale = false;
  int attempts = 0;
  double eps_used = 0.0;
  int64_t launches = 0;
  int last_solve_grid = 0;
  // per-context launch configuration (function attributes and occupancy are per device: nothing process-wide is cached)
  int num_sms = 0;
  bool acc_ready = false;
  int solve_bpsm = -1, bb_bpsm = -1;     // resident CTAs per SM of k_solve / k_solve_bb at their shared-memory size
  size_t bb_smem = 0;
  // sim3ba_step_graph: n GN iterations captured once as a CUDA graph
  cudaGraphExec_t graph_exec = nullptr;
  int graph_steps = 0;
  int64_t graph_launches = 0;
  bool profiling = false;
  cudaEvent_t ev[8] = {};
  float phase_ms[8] = {};
  std::string err;
};

// kernel launchers (each returns the cudaError of the launch)
cudaError_t launch_pack(Ctx* c, const float* d_points, const float* d_conf);
cudaError_t launch_accumulate(Ctx* c);                   // kernels 1+2: partials -> blocks35, stats, cost
// function attributes / occupancy / lazily allocated work buffers of the launchers, done outside a stream capture
cudaError_t prepare_accumulate(Ctx* c);
cudaError_t prepare_solve(Ctx* c);
cudaError_t prepare_solve_bb(Ctx* c);
cudaError_t ensure_dense(Ctx* c, bool want_Hd, bool want_L);   // Hd (read-back / loaded system) and L (tile plans) exist only when used
cudaError_t launch_assemble(Ctx* c, double* dst, double lambda, double eps, bool from_dense);  // kernel 3
cudaError_t launch_gradient(Ctx* c);                     // g from the per-edge b_e
cudaError_t launch_load_gradient(Ctx* c, const double* d_g);
cudaError_t launch_solve(Ctx* c);                        // kernels 3+4: tile assembly (damped), then the persistent Cholesky / solves / eps retry
bool build_plan(Ctx* c, bool dense, SolvePlan& plan, std::string& err);   // host symbolic factorisation + upload
void free_plan(SolvePlan& plan);
bool build_dense_plan(int nb, SolvePlan& plan, cudaStream_t stream, std::string& err);   // every lower tile of an nb x nb tile grid
bool build_bb_plan(Ctx* c, std::string& err, int lmax_hint = 0);          // host band + border analysis + upload; plan_bb.valid says whether it applies
void free_bb_plan(BBPlan& plan);
cudaError_t launch_solve_bb(Ctx* c);                     // kernels 3+4, band + border variant (solver mode 2)
cudaError_t launch_retract(Ctx* c);                      // kernel 5
// gauge synchronisation (NEXT-2): moments of edge e -> T* (Umeyama / endpoint fallback) -> applied to the moving keyframes
cudaError_t launch_gauge_sync(Ctx* c, int e, const int32_t* d_moving, int n_moving, int moving_is_i, int n_c_min, double* d_work, int grid);
int gauge_sync_grid(int HW);
cudaError_t launch_gauge_sync_static(Ctx* c, int e, const int32_t* d_moving, int n_moving, int moving_is_i, int n_c_min,
                                     double* d_result);   // no allocation: scratch in a file-scope device array (k_gauge_sync.cu)
int gauge_sync_static_max_pixels();
int gauge_sync_work_doubles(int grid);
// segment-level depth refinement with poses fixed (NEXT-1)
cudaError_t run_depth_refine(Ctx* c, const int32_t* d_labels, int n_seg, const int32_t* h_pairs, const double* h_delta, int n_pairs,
                             const int32_t* h_anchor, int n_anchor, const sim3ba_depth_params& p, int n_iters, double* d_eta, double* h_cost);
cudaError_t launch_depth_apply(Ctx* c, const float* d_points, const float* d_conf, const int32_t* d_labels, int n_seg, const double* d_eta);
int depth_max_segments();
cudaError_t run_probe_fp64(cudaStream_t st, double* dfma_tflops, double* dmma_tflops);   // FP64 peak probe (probe_fp64.cu)

}  // namespace sim3ba
