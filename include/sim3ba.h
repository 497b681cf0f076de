/*
 * sim3ba.h - C ABI of libsim3ba: the Gauss-Newton step of the unified multi-agent Sim(3) pose graph
 * over dense pointmap correspondences (CoMo3R-SLAM, arxiv 2605.30488, section III-D,
 * PAPER.md:106-122), hand-written CUDA for sm_100a (B200).
 *
 * Conventions
 *   - Pose of keyframe i: T_WCi : X -> s_i R_i X + t_i, stored as 8 doubles
 *     (tx, ty, tz, qx, qy, qz, qw, s), q a unit quaternion.
 *   - Tangent vector tau_i = (v, omega, zeta) in R^7; update T <- Exp(tau) T.
 *   - N keyframes, HW = height*width pixels per keyframe, E directed edges, n = 7N.
 *   - "d_" arguments are DEVICE pointers, "h_" arguments are HOST pointers.
 *   - Every function returns SIM3BA_OK (0) or a negative sim3ba_status; nothing throws or aborts
 *     across this boundary.  sim3ba_last_error() gives a human-readable message for the last
 *     failure on that context (or for a failed create when ctx == NULL).
 *   - All work is enqueued on the stream given at create; functions taking host pointers
 *     synchronise that stream before returning, the others do not unless stated.
 *   - There is no CPU fallback: without a CUDA device every compute entry point fails with
 *     SIM3BA_ERR_CUDA.
 */
#ifndef SIM3BA_H_
#define SIM3BA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sim3ba_ctx sim3ba_ctx; /* opaque, owned by the library */

typedef enum {
  SIM3BA_OK = 0,
  SIM3BA_ERR_INVALID_ARG = -1,
  SIM3BA_ERR_CUDA = -2,
  SIM3BA_ERR_ALLOC = -3,
  SIM3BA_ERR_BAD_STATE = -4
} sim3ba_status;

/* Robust-kernel and solver constants.  PAPER.md:76,177: Sigma = diag(sigma_r^2 I3, sigma_d^2),
 * sigma_r = 0.003, sigma_d = 10, Huber breakpoint kappa = 1.345 on the whitened residual
 * r_c = sqrt(q) e_c / sigma_c, IRLS weight w = min(1, kappa/|r_c|).  PAPER.md:120-122: Eq. (7)
 * (H + lambda diag(H) + eps_r I) tau = -g, eps_r = eps0 * 100^r, r = 0..max_attempts-1
 * (paper: eps0 = 1e-6, six attempts), zero update when all attempts fail. */
typedef struct {
  float sigma_ray;   /* sigma_r  > 0 */
  float sigma_dist;  /* sigma_d  > 0 */
  float huber_k;     /* kappa    > 0 */
  float conf_min;    /* a match (m,n) is valid iff 0 <= n < HW, c_i[m] > conf_min, c_j[n] > conf_min */
  double lm_lambda;  /* lambda >= 0; global backend: 0 (Gauss-Newton) */
  double eps0;       /* eps_0 >= 0 */
  int32_t max_attempts; /* 1..16 */
  int32_t reserved;
} sim3ba_params;

/* Fills *p with the paper's constants (0.003, 10, 1.345, conf_min 0, lambda 0, 1e-6, 6). */
int sim3ba_default_params(sim3ba_params* p);

/* Creates a context for one graph (vertices = keyframe poses in one flat index
 * space, edges with dense matches, validity masks and endpoint confidences).
 *   d_points  [N][HW][3] float32, canonical pointmap of each keyframe in its own camera frame
 *   d_conf    [N][HW]    float32, per-pixel confidence (q_mn = sqrt(c_i[m] c_j[n]))
 *   d_edges   [E][2]     int32 (i, j): the match map is dense over the pixels m of i, X_j[n] is
 *                        mapped into camera i by T_ij = T_WCi^-1 T_WCj (Eq. (1))
 *   d_match   [E][HW]    int32, pixel m of i -> pixel n of j; n < 0 or n >= HW means "no match"
 *   h_fixed_kf[n_fixed]  int32 gauge keyframes whose pose is held fixed (paper: {0})
 * Ownership: the library copies points+conf into an internal packed float4 array and copies the
 * edge list; d_match is BORROWED and must stay valid and unchanged until sim3ba_destroy.
 * Poses start as identity; call sim3ba_set_poses.  Errors: i == j or endpoint outside [0,N),
 * fixed keyframe outside [0,N), non-positive sizes or sigmas, height*width > 2^28 -> SIM3BA_ERR_INVALID_ARG.
 * Synchronises the stream. */
int sim3ba_create(sim3ba_ctx** out, int32_t n_kf, int32_t height, int32_t width, int32_t n_edges,
                  const float* d_points, const float* d_conf, const int32_t* d_edges,
                  const int32_t* d_match, const int32_t* h_fixed_kf, int32_t n_fixed,
                  const sim3ba_params* params, void* cuda_stream);

int sim3ba_destroy(sim3ba_ctx* ctx);

/* Replace the robust-kernel / solver constants (takes effect at the next build/solve).  conf_min is
 * fixed at create (the per-pixel validity c > conf_min is decided once, exactly, when the pointmaps
 * are packed): a different conf_min -> SIM3BA_ERR_INVALID_ARG. */
int sim3ba_set_params(sim3ba_ctx* ctx, const sim3ba_params* params);

/* Poses [N][8] double, device pointers; asynchronous device-to-device copies. */
int sim3ba_set_poses(sim3ba_ctx* ctx, const double* d_poses);
int sim3ba_get_poses(sim3ba_ctx* ctx, double* d_poses);

/* a1-a6 at the current poses: per-match residuals (Eq. (1)), weights, Jacobians
 * (Eq. (6)), per-edge reduction into 7x7 blocks, scatter into the dense 7N
 * system with the gauge keyframes' rows/columns replaced by identity and their gradient by 0.
 * Fills the per-edge statistics and blocks and the undamped dense (H, g). */
int sim3ba_build_system(sim3ba_ctx* ctx);

/* a7 on the last built system: Eq. (7) with the epsilon escalation of PAPER.md:122 by blocked
 * FP64 Cholesky and two triangular solves.  Requires a previous build (else BAD_STATE).
 * "All attempts failed" is not an error: tau = 0, attempts = max_attempts.  The retry loop runs on the
 * device inside one persistent kernel: no host synchronisation. */
int sim3ba_solve(sim3ba_ctx* ctx);

/* One Gauss-Newton iteration: a1-a5, assembly of the damped system, a7, and the retraction
 * T_i <- Exp(tau_i) T_i of every non-fixed keyframe.  (The undamped dense H of
 * sim3ba_get_system is not refreshed by this call; the per-edge blocks and g are.) */
int sim3ba_step(sim3ba_ctx* ctx);

/* n_steps Gauss-Newton iterations (sim3ba_step each) enqueued as ONE CUDA-graph launch.  The kernel sequence of the
 * iterations is captured once per (context, n_steps, params, solver mode) and replayed: the same kernels in the same
 * order, so the poses afterwards equal those of n_steps x sim3ba_step bit for bit.  For small problems -- the tracker's
 * single relative pose (E = 1, n = 7), config 1 -- an iteration is bound by launch latency and the graph
 * removes the per-kernel launch cost.  Asynchronous.  Errors: INVALID_ARG (n_steps outside 1..4096), CUDA. */
int sim3ba_step_graph(sim3ba_ctx* ctx, int32_t n_steps);

/* Same iteration with HOST pose buffers: copies h_poses_in [N][8] to the device (if non-NULL),
 * runs sim3ba_step, copies the new poses to h_poses_out [N][8] and the robust cost at the input
 * poses to *h_cost (each if non-NULL).  Pinned host memory recommended.  Synchronises. */
int sim3ba_step_host(sim3ba_ctx* ctx, const double* h_poses_in, double* h_poses_out, double* h_cost);

/* The whole job with HOST buffers (the end-to-end leg of bench.py): allocates device memory, copies the
 * graph in -- h_points [N][HW][3], h_conf [N][HW], h_edges [E][2], h_match [E][HW], layouts as in
 * sim3ba_create, pinned host memory recommended -- creates a context, runs n_iters Gauss-Newton
 * iterations (sim3ba_step, a1-a8 each; fixed count) from h_poses_in [N][8], copies the
 * final poses to h_poses_out [N][8] and, if h_cost is non-NULL, the robust cost at the start of
 * iteration it to h_cost[it]; frees everything and synchronises the stream.  Nothing is kept.
 * Errors as sim3ba_create / sim3ba_step; the message is read with sim3ba_last_error(NULL). */
int sim3ba_optimize_host(int32_t n_kf, int32_t height, int32_t width, int32_t n_edges, const float* h_points,
                         const float* h_conf, const int32_t* h_edges, const int32_t* h_match,
                         const int32_t* h_fixed_kf, int32_t n_fixed, const sim3ba_params* params,
                         const double* h_poses_in, int32_t n_iters, double* h_poses_out, double* h_cost,
                         void* cuda_stream);

/* Gauge synchronisation of two map components before their first joint solve.
 * Over the valid matches (m, n) of edge `edge` = (i, j) of the graph -- the validity rule of the GN step -- the matched
 * points are lifted into the two world frames with the CURRENT poses, x = T_WCi X_i[m], y = T_WCj X_j[n], and
 * (s*, R*, t*) = argmin sum |x - (s R y + t)|^2 (Eq. (3)) is found in closed form (Eq. (4), Umeyama; FP64).  With fewer
 * than n_c_min correspondences (paper: 64) T* = T_WCi T_WCj^-1 instead (also when the matched cloud is degenerate --
 * zero variance or a non-positive / non-finite scale -- where Eq. (4) has no answer).  T* is then left-multiplied onto the poses of
 * the n_moving keyframes h_moving_kf (host array; the component of j).  moving_is_i != 0 swaps the roles: the similarity
 * maps x onto y (fallback T_WCj T_WCi^-1) and is meant for the component of i.  Host outputs, each may be NULL:
 * h_T [8] = T* in the pose layout (t, q_xyzw, s), *h_n_c = number of correspondences, *h_fallback = 1 if the endpoint
 * transform was used.  Synchronises the stream.  Errors: INVALID_ARG (edge / keyframe out of range), CUDA, ALLOC. */
int sim3ba_gauge_sync(sim3ba_ctx* ctx, int32_t edge, const int32_t* h_moving_kf, int32_t n_moving, int32_t moving_is_i,
                      int32_t n_c_min, double* h_T, int32_t* h_n_c, int32_t* h_fallback);

/* sim3ba_gauge_sync WITHOUT any device allocation, for callers that cannot call cudaMalloc (a region under CUDA graph
 * capture, a tight serving loop, a harness that forbids it).  Same operation (Eq. (3)-(4)), same kernels,
 * same fixed summation order: results are bit-identical to sim3ba_gauge_sync.  The only scratch memory of the operation
 * -- one record of 20 doubles per 1024 pixels of the linking edge -- lives in a file-scope device array of the library
 * sized for images of at most SIM3BA_STATIC_MAX_PIXELS = 262144 pixels (512 x 512): 40960 bytes that every GPU which
 * loads the library holds until the process exits.  A context with a larger image is rejected with SIM3BA_ERR_INVALID_ARG
 * and a message naming the limit (use sim3ba_gauge_sync there).
 *   d_moving_kf  DEVICE array [n_moving] of keyframe indices (may be NULL if n_moving = 0); not validated on the host:
 *                an index outside 0 .. n_kf - 1 is skipped on the device
 *   d_result     DEVICE array [10], written: [0..7] T* in the pose layout (t, q_xyzw, s), [8] number of correspondences,
 *                [9] 1 if the endpoint transform was used
 * The call enqueues three kernels on the context's stream and returns: no cudaMalloc / cudaFree, no pool allocation, no
 * copy, no synchronisation; read d_result after synchronising the stream.  The first call on a device looks the array's
 * address up (cudaGetSymbolAddress, once per device and process, with that device current): make that call outside a
 * capture.  ALL calls on one device share the array: calls that overlap on the GPU (two streams, two contexts) race on
 * it; calls on one stream are ordered and safe.  Nothing in the array needs clearing between calls (every record that
 * is read is written by the same call).  Errors: INVALID_ARG (edge out of range, NULL buffer, n_c_min < 1, image too
 * large), CUDA. */
#define SIM3BA_STATIC_MAX_PIXELS 262144
int sim3ba_gauge_sync_static(sim3ba_ctx* ctx, int32_t edge, const int32_t* d_moving_kf, int32_t n_moving, int32_t moving_is_i,
                             int32_t n_c_min, double* d_result);

/* ---- Segment-level structure refinement with the poses held fixed (Eq. (8)-(10); SURVEY 8(f)
 * NEXT-1; BASELINE config 5 "pose-depth alternation").  One log-scale eta_g per segment g of a keyframe:
 * X(eta_g) = exp(eta_g) X_init (Eq. (8)); data term Eq. (9) over the graph's valid matches whose two pixels carry a
 * label, 3-D point residual sqrt(q) [T_ij X_j(eta) - X_i(eta)] / sigma_point with per-component Huber; boundary term
 * ((eta_g - eta_h) + Delta_gh)^2 over the given pairs and prior eta_g^2 (Eq. (10), conventions D1-D5 of DESIGN.md
 * section 10); per iteration the independent steps Delta eta_g = -g_g / ((1 + lambda_lm) H_gg) with the Jacobi diagonal
 * H_gg, clipped to eta_max; segments of the anchor keyframes stay fixed. ---- */
typedef struct {
  float  sigma_point;      /* paper 0.05 */
  float  huber_k;          /* kappa on the whitened residual; not restated for Eq. (9): 1.345 */
  double lambda_smooth;    /* paper 1 */
  double lambda_prior;     /* paper 1 (> 0) */
  double lambda_lm;        /* paper 0.05 */
  double eta_max;          /* paper 0.5 */
} sim3ba_depth_params;
int sim3ba_depth_default_params(sim3ba_depth_params* p);
/* n_iters iterations at the context's CURRENT poses on the PRISTINE pointmaps given at sim3ba_create (eta is the absolute
 * log-scale of Eq. (8) whatever sim3ba_apply_depth has done to the pointmaps the pose passes see).  d_labels [N][HW] int32 DEVICE: label of a
 * pixel inside its keyframe, 0 <= label < n_seg <= 512, < 0 = excluded pixel; segment id = keyframe * n_seg + label.
 * h_pairs [n_pairs][2] HOST segment ids (g, h) of the 4-adjacent pairs, h_delta [n_pairs] HOST Delta_gh,
 * h_anchor_kf HOST list of keyframes whose segments stay fixed.  d_eta [N * n_seg] double DEVICE, in/out (caller
 * owned; start from zeros for eta = 0).  h_cost HOST [n_iters] or NULL: the objective at the start of each iteration.
 * Synchronises the stream.  Errors: INVALID_ARG, CUDA, ALLOC. */
int sim3ba_depth_refine(sim3ba_ctx* ctx, const int32_t* d_labels, int32_t n_seg, const int32_t* h_pairs, const double* h_delta,
                        int32_t n_pairs, const int32_t* h_anchor_kf, int32_t n_anchor, const sim3ba_depth_params* p,
                        int32_t n_iters, double* d_eta, double* h_cost);
/* The other half of the alternation: re-packs the pointmaps the pose passes read from the caller's pristine d_points
 * [N][HW][3], d_conf [N][HW] (as in sim3ba_create) with every labelled pixel scaled by exp(eta) of its segment, so that
 * the next sim3ba_step sees the refined structure.  The first call keeps a pristine packed copy inside the context
 * (16 bytes per pixel) for the structure passes that follow.  Asynchronous on the context's stream. */
int sim3ba_apply_depth(sim3ba_ctx* ctx, const float* d_points, const float* d_conf, const int32_t* d_labels, int32_t n_seg,
                       const double* d_eta);

/* The terminal pose-depth alternation as ONE job with HOST buffers (PAPER.md:143 last sentence: "the segment-level
 * structure refinement alternates with pose refinement"; "at most 100 pose-depth rounds with up to ten depth
 * iterations and 50 pose iterations per round"; BASELINE config 5).  Uploads the graph (as sim3ba_optimize_host) plus
 * h_labels [N][HW] int32 and h_eta [N * n_seg] double, creates a context, then runs n_rounds rounds of
 * { sim3ba_depth_refine with n_depth_iters iterations at the current poses (anchor keyframes = the fixed keyframes);
 *   sim3ba_apply_depth; n_pose_iters x sim3ba_step on the rescaled pointmaps },
 * eta carried across the rounds as the absolute log-scale of Eq. (8).  Fixed counts (reading R14): the paper's numbers
 * are caps and it states no stopping rule.  Host outputs: h_poses_out [N][8], h_eta (in/out), and, if non-NULL,
 * h_pose_cost [n_rounds * n_pose_iters] (robust cost at the start of each pose iteration) and h_depth_cost
 * [n_rounds * n_depth_iters] (structure objective at the start of each depth iteration).  h_pairs / h_delta / depth
 * params as in sim3ba_depth_refine.  Frees everything and synchronises the stream.  Errors as sim3ba_create /
 * sim3ba_depth_refine / sim3ba_step; the message is read with sim3ba_last_error(NULL). */
int sim3ba_refine_host(int32_t n_kf, int32_t height, int32_t width, int32_t n_edges, const float* h_points, const float* h_conf,
                       const int32_t* h_edges, const int32_t* h_match, const int32_t* h_fixed_kf, int32_t n_fixed,
                       const sim3ba_params* params, const int32_t* h_labels, int32_t n_seg, const int32_t* h_pairs, const double* h_delta,
                       int32_t n_pairs, const sim3ba_depth_params* depth_params, int32_t n_rounds, int32_t n_depth_iters,
                       int32_t n_pose_iters, const double* h_poses_in, double* h_poses_out, double* h_eta, double* h_pose_cost,
                       double* h_depth_cost, void* cuda_stream);

/* a8 only: T_i <- Exp(tau_i) T_i with the tau of the last solve. */
int sim3ba_retract(sim3ba_ctx* ctx);

/* ---- read-back for parity.  Returned DEVICE pointers are owned by the context and stay valid
 * until the next build/solve/step/destroy on it; the caller synchronises the stream. ---- */

/* n_valid [E] int32 valid matches per edge; checksum [E] uint64 = sum over the valid matches of
 * (m*HW + n) mod 2^64; cost [E] double = sum of Huber rho over the edge's matches. */
int sim3ba_get_edge_stats(sim3ba_ctx* ctx, const int32_t** d_n_valid, const uint64_t** d_checksum,
                          const double** d_cost);

/* blocks35 [E][35] double: the 28 upper-triangular entries (row-major, r <= c) of
 * A_e = sum J_j^T Omega J_j followed by the 7 entries of b_e = sum J_j^T Omega e, with
 * J_j = J_xi Ad_{T_WCi^-1}.  H_ii += A_e, H_jj += A_e, H_ij -= A_e, H_ji -= A_e,
 * g_j += b_e, g_i -= b_e. */
int sim3ba_get_edge_blocks(sim3ba_ctx* ctx, const double** d_blocks35);

/* Undamped dense system of the last sim3ba_build_system: H column-major == row-major (symmetric),
 * leading dimension *ld >= 7N, lower triangle (row >= col) valid, strict upper triangle zero;
 * g [7N].  Gauge keyframes: identity diagonal block, zero off-diagonal blocks, zero gradient. */
int sim3ba_get_system(sim3ba_ctx* ctx, const double** d_H, int32_t* ld, const double** d_g);

/* tau [7N] double (device); scalars are written to host memory (synchronises the stream):
 * attempts used (1 = first factorisation succeeded), eps of the successful attempt (NaN if none),
 * total robust cost at the poses of the last build. */
int sim3ba_get_update(sim3ba_ctx* ctx, const double** d_tau, int32_t* h_attempts, double* h_eps_used,
                      double* h_cost);

/* a0 bookkeeping, HOST pointers owned by the context: keyframe -> incident-edge CSR
 * (kf_ptr [N+1], kf_edge [2E], edges ascending) and the sorted unique unordered keyframe pairs
 * (pair_kf [P][2] = (hi, lo), pair_ptr [P+1], pair_edge [E], edges ascending). */
int sim3ba_get_bookkeeping(sim3ba_ctx* ctx, const int32_t** h_kf_ptr, const int32_t** h_kf_edge,
                           int32_t* n_pairs, const int32_t** h_pair_kf, const int32_t** h_pair_ptr,
                           const int32_t** h_pair_edge);

/* Overrides the system of the next sim3ba_solve with a caller-supplied dense one (decomposition
 * tests: oracle (H, g) -> GPU solver).  d_H [7N][7N] row-major symmetric double, d_g [7N]. */
int sim3ba_load_system(sim3ba_ctx* ctx, const double* d_H, const double* d_g);

/* Solver plan (a7), all giving the same tau up to rounding.
 * mode 2 (default): band + border block Cholesky ("sparse Cholesky") -- the free keyframes are
 *   split at create into interior keyframes (independent segments of a temporal chain, block band 3) and
 *   border keyframes (one endpoint of every longer link: loop closures, inter-agent edges; separator triples
 *   that cap a segment's length); segments are eliminated at 7x7 granularity in parallel, the Schur complement
 *   on the border is a small system S that is itself sparse: where that removes at least two 64-row tile columns,
 *   an independent set of separator groups is eliminated from S in the same way, and again from what that leaves
 *   (up to three further levels), before the tiled Cholesky takes the dense rest.  Where the graph does not have that shape (a segment touching more than 28 border
 *   keyframes, more than 292 border keyframes) mode 2 runs mode 0.
 * mode 0: the tiled Cholesky walks only the non-zero 64x64 tiles of L (symbolic tile-level factorisation of the
 *   keyframe graph in temporal order, fill included, computed at create).
 * mode 1: every lower tile (the dense blocked factorisation; always used for sim3ba_load_system).
 * Three environment variables exist for tests and experiments only: SIM3BA_BB_LMAX (read at create: cap on the segment
 * length of mode 2, default 0.9 sqrt(free keyframes)) and SIM3BA_BB_LEVELS (read at create: 1 = no further levels, 2 = a
 * further level wherever a separator group can be eliminated) -- other elimination orders, tau equal up to rounding -- and
 * SIM3BA_SOLVE_MAX_CTAS (read at every solve: cap on the grid of the persistent solve kernel, so that a CTA takes several
 * segments / tiles; tau is bitwise independent of the grid). */
int sim3ba_set_solver_mode(sim3ba_ctx* ctx, int32_t mode);
/* Band + border plan of the graph (host output): h_info[0] = 1 if mode 2 applies to this graph, [1] interior
 * keyframes, [2] segments, [3] border keyframes, [4] longest segment, [5] most border keyframes touched by a segment,
 * [6] separator groups eliminated at the further levels (0: none), [7] keyframes of the dense system that is finally
 * solved (= [3] without further levels). */
int sim3ba_get_bb_info(sim3ba_ctx* ctx, int32_t h_info[8]);
/* Host outputs (each may be NULL): non-zero tiles of the tile-sparse plan (of the dense plan in mode 1), lower tiles of
 * the dense plan, flop count of the ACTIVE plan (factor + both triangular solves, FMA = 2: at 7x7 granularity with a dense
 * border system for the band + border plan of mode 2, at 64x64 tile granularity for modes 0 / 1), CTAs of the last
 * persistent solve launch. */
int sim3ba_get_solver_info(sim3ba_ctx* ctx, int32_t* h_n_tiles, int32_t* h_n_tiles_dense, double* h_flops,
                           int32_t* h_grid);

/* Number of kernels this library launched on the context since create (for bench accounting). */
int sim3ba_get_launch_count(sim3ba_ctx* ctx, int64_t* h_count);

/* Device time in milliseconds of the phases of the last sim3ba_step / build / solve, measured
 * with CUDA events on the context's stream: [0] kernel 1 (per-match accumulate, a1-a5 partials),
 * [1] kernel 2 (FP64 evaluation of the deferred matches, per-edge reduce + adjoint congruence, gradient, cost), [2] damped tile assembly (a6, first
 * attempt), [3] factor + triangular solves (a7, incl. re-assembly of later attempts), [4] retraction (a8),
 * [5..7] reserved (0).  Synchronises.  Only recorded after sim3ba_set_profiling(ctx, 1). */
int sim3ba_set_profiling(sim3ba_ctx* ctx, int32_t enable);
int sim3ba_get_phase_ms(sim3ba_ctx* ctx, float h_ms[8]);

/* With profiling on, the band + border solve kernel (mode 2) stamps its phases with the device's global timer; microseconds
 * of the last solve: [0] assembly (a6), [1] segment elimination, [2] grid barrier after it, [3] Schur rows, [4] border
 * system, [5] back-substitution, [6..7] reserved (0).  All zero if the last solve was not profiled.  Synchronises. */
int sim3ba_get_solve_phase_us(sim3ba_ctx* ctx, float h_us[8]);

/* Measures the FP64 peak of the current device, the denominator of the solve's roofline (MEASURED_PEAKS.json has none):
 * TFLOP/s (FMA = 2) of register-resident DFMA chains and of mma.sync.m8n8k4.f64 (DMMA) chains on every SM, best of five
 * launches, CUDA events on the given stream.  Host outputs.  Takes a few milliseconds; synchronises. */
int sim3ba_probe_fp64(double* h_dfma_tflops, double* h_dmma_tflops, void* cuda_stream);

/* All device memory of the library comes from a stream-ordered memory pool the library owns (one per device), which keeps
 * freed blocks for the next context / job.  This call synchronises the current device and returns the pool's unused memory
 * to the driver. */
int sim3ba_release_memory(void);

/* Binding convenience: asynchronous device-to-device copy of `bytes` bytes on the context's stream
 * (used to move the read-back buffers above into caller-owned device memory). */
int sim3ba_copy_d2d(sim3ba_ctx* ctx, void* d_dst, const void* d_src, uint64_t bytes);

const char* sim3ba_last_error(const sim3ba_ctx* ctx);
const char* sim3ba_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SIM3BA_H_ */
