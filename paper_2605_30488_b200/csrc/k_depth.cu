// Segment-level structure refinement with the poses held fixed.
//
//   Eq. (8)  :130   X_{k,p}(eta_g) = exp(eta_g) X_init (one log-scale eta_g per segment g of keyframe k)
//   Eq. (9)  :134   r_c = sqrt(q) [T_ij X_j,n(eta) - X_i,m(eta)]_c / sigma_point, per-component Huber
//   :143            J_g = -X_i,m(eta), J_h = s_ij R_ij X_j,n(eta); only H_gg, H_hh of the data term, complete gradient;
//                   boundary term ((eta_g - eta_h) + Delta_gh)^2 and prior eta_g^2 Jacobi-decoupled likewise;
//                   Delta eta_g = -g_g / ((1 + lambda_lm) H_gg), clipped to eta_max, anchor keyframes fixed
// Conventions D1-D5 of DESIGN.md section 10 (objective = sum rho + lambda_s/2 E_bnd + lambda_p/2 E_prior).
//
// The poses are fixed during a structure pass, so the one expensive, cancellation-prone part of the residual does not
// change between its iterations.  With y = T_ij X_j - X_i (both at eta = 0) and E_g = exp(eta_g),
//     res = T_ij X_j(eta_h) - X_i(eta_g) = E_h y + (E_h - E_g) X_i + (1 - E_h) t_ij                      (Eq. (8)-(9))
// an identity: y is evaluated ONCE per call, in FP64, and kept in fp32 (kernel P), and every iteration (kernel A) is a
// pure stream over (X_i, label of m; y, sqrt(q), label of n) with no gather and no FP64 per match.
//
// Kernel P (k_depth_prep): per candidate match of every edge, n = match[e][m]; valid <=> the GN step's rule (R12) and both
// pixels labelled; record (y [3] fp32 from the FP64 difference, sqrt(q) = w_i w_j or 0 if invalid) and the label of n.
// Kernel A (k_depth_edge): one CTA (4 warps) per (edge, tile of image rows of i), in kernel 1's order (edges sorted by
// keyframe, the tiles of an edge together, so X_i and its labels are shared through L2).  A warp's work item is a patch
// of 32 columns x 4 rows: every lane owns one column, i.e. four vertically adjacent pixels, which mostly share their
// segment on both sides.  All loads are per-lane cp.async into a two-stage shared-memory ring one item ahead (a lane
// only reads what it copied itself: no barrier).  Two pixels at a time in the two lanes of packed fp32x2 instructions.
// Precision: the per-segment constants E_g, E_h and (1 - E_h) t_ij are computed in FP64 and carried as unevaluated
// fp32 pairs (hi, lo); res is two nested fused multiply-adds on the leading parts (each rounds an exact sum once) plus the
// trailing parts, so it is as accurate as the FP64 difference rounded to fp32 up to a random 2^-24 of its larger terms --
// the rounding the stored y carries anyway; everything after res is fp32; fp32 partial sums hold at most 128 terms,
// every sum from there up is FP64.
// Binning WITHOUT floating-point atomics, bit-reproducible: a lane first merges the records of its four pixels that
// share the label of its first valid pixel; that record goes through one warp phase per item and side, the few others
// (stray matches, a segment boundary inside the patch) are queued in shared memory and take a phase per 32 of them.  A
// phase (bin_phase): match.any groups the lanes by label, every group is summed in fp32 by a fixed tree of shuffles and
// its first lane adds the total to the warp's FP64 bin.  The warps' bins are added in a fixed order -> one record
// [2 sides][n_seg][g, H] + cost per (edge, tile).
// Kernel B (k_depth_update): one thread per segment gathers its records through the keyframe -> edge CSR, adds boundary
// and prior terms, takes the damped clipped step into a second eta buffer.  Kernel C sums the objective.
//
// X_init: the kernels read the context's PRISTINE packed pointmaps (Ctx::pm0, a snapshot taken before the first
// sim3ba_apply_depth overwrites Ctx::pm with exp(eta) X_init), so eta stays the absolute log-scale of Eq. (8) over any
// number of pose-depth rounds.
#include <math.h>

#include <vector>

#include "f32x2.cuh"
#include "sim3ba_internal.cuh"
#include "sim3_math.cuh"

namespace sim3ba {

namespace {

constexpr int kDpMaxWarps = 4;      // warps per CTA: 4 up to 64 segments per keyframe, 2 above (the per-warp bins grow with n_seg: more CTAs fit an SM)
constexpr int kDpMaxSeg = 512;       // labels per keyframe (the paper's SLIC pass: M_k ~ 200)
constexpr int kDpRows = 4;           // rows of a warp item (pixels per lane)
constexpr int kDpCols = 32;          // columns of a warp item (one per lane)
#ifndef SIM3BA_DP_TILE_PX
#define SIM3BA_DP_TILE_PX 16384
#endif
constexpr int kDpTilePx = SIM3BA_DP_TILE_PX;
constexpr int kDpStages = 2;         // ring of items per warp: copies run one item ahead
constexpr int kDpQueue = 128;        // per-warp queue of (bin, g, H) records waiting for a phase (power of two)
// per-warp shared memory: every ring array is [stage][row][lane], so a warp's 32 lanes touch 32 consecutive words / float4
constexpr size_t kDpOffXi = 0;                                                          // float4 [kDpStages][4][32]
constexpr size_t kDpOffRec = kDpOffXi + sizeof(float4) * kDpStages * kDpRows * 32;      // float4 [kDpStages][4][32]
constexpr size_t kDpOffLi = kDpOffRec + sizeof(float4) * kDpStages * kDpRows * 32;      // int32  [kDpStages][4][32]
constexpr size_t kDpOffLh = kDpOffLi + sizeof(int32_t) * kDpStages * kDpRows * 32;      // int32  [kDpStages][4][32]
constexpr size_t kDpOffQ = kDpOffLh + sizeof(int32_t) * kDpStages * kDpRows * 32;       // int32 bin, float g, float H  [kDpQueue] each
constexpr size_t kDpWarpBytes = kDpOffQ + 12 * kDpQueue;                                // 11776 bytes per warp

struct DepthDev {
  double inv_sigma, huber_k, lambda_smooth, lambda_prior, lambda_lm, eta_max;
  float s_cap, k_cap, hk2;     // 1 / sigma^2, kappa / sigma, kappa^2 in fp32 (host-computed: the per-match arithmetic's constants)
};

__device__ __forceinline__ uint32_t dp_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void dp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void dp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Kernel P: the eta-independent part of every candidate match, once per structure pass.
__global__ void __launch_bounds__(256)
k_depth_prep(const float4* __restrict__ pm, const int32_t* __restrict__ match, const int32_t* __restrict__ edges,
             const int32_t* __restrict__ grp_edge, const int32_t* __restrict__ labels, const double* __restrict__ poses, int HW, int n_seg, int chunks,
             float4* __restrict__ rec, int32_t* __restrict__ lab_n) {
  // kernel 1's launch order (edges sorted by keyframe i): a keyframe's pointmap and labels are fetched from HBM once
  const int k = blockIdx.x / chunks, chunk = blockIdx.x - k * chunks, e = grp_edge[k];
  const int i = edges[2 * e], j = edges[2 * e + 1];
  const Sim3d T = relative_pose(load_pose(poses + 8 * i), load_pose(poses + 8 * j));   // T_ij
  double sR[9];
#pragma unroll
  for (int q = 0; q < 9; ++q) sR[q] = T.s * T.R[q];
  const float4* __restrict__ Pi = pm + (size_t)i * HW;
  const float4* __restrict__ Pj = pm + (size_t)j * HW;
  const int32_t* __restrict__ mt = match + (size_t)e * HW;
  const int32_t* __restrict__ li = labels + (size_t)i * HW;
  const int32_t* __restrict__ lj = labels + (size_t)j * HW;
  const int per = (HW + chunks - 1) / chunks;
  const int m1 = min(HW, (chunk + 1) * per);
  constexpr int kB = 4;                                          // matches in flight per thread: all loads of a batch are issued before its arithmetic
  for (int mb = chunk * per + threadIdx.x; mb < m1; mb += 256 * kB) {
    int n[kB], lg[kB], lh[kB];
    float4 a[kB], b[kB];
#pragma unroll
    for (int u = 0; u < kB; ++u) {
      const int m = mb + 256 * u;
      n[u] = m < m1 ? __ldcs(mt + m) : -1;
    }
#pragma unroll
    for (int u = 0; u < kB; ++u) {
      const int m = mb + 256 * u;
      const bool in = (unsigned)n[u] < (unsigned)HW;
      a[u] = in ? Pi[m] : make_float4(0.f, 0.f, 0.f, -1.f);
      lg[u] = in ? li[m] : -1;
      b[u] = in ? Pj[n[u]] : make_float4(0.f, 0.f, 0.f, -1.f);
      lh[u] = in ? lj[n[u]] : -1;
    }
#pragma unroll
    for (int u = 0; u < kB; ++u) {
      const int m = mb + 256 * u;
      if (m >= m1) break;
      float4 out = make_float4(0.f, 0.f, 0.f, 0.f);
      int lab = -1;
      if (a[u].w >= 0.f && b[u].w >= 0.f && (unsigned)lg[u] < (unsigned)n_seg && (unsigned)lh[u] < (unsigned)n_seg) {
        const double X0 = (double)b[u].x, X1 = (double)b[u].y, X2 = (double)b[u].z;
        out.x = (float)(fma(sR[0], X0, fma(sR[1], X1, fma(sR[2], X2, T.t[0]))) - (double)a[u].x);
        out.y = (float)(fma(sR[3], X0, fma(sR[4], X1, fma(sR[5], X2, T.t[1]))) - (double)a[u].y);
        out.z = (float)(fma(sR[6], X0, fma(sR[7], X1, fma(sR[8], X2, T.t[2]))) - (double)a[u].z);
        out.w = a[u].w * b[u].w;                                 // sqrt(q) = w_i w_j (w = c^(1/4)) > 0
        lab = lh[u];
      }
      __stcs(rec + (size_t)e * HW + m, out);                     // w = 0 marks "no term"
      __stcs(lab_n + (size_t)e * HW + m, lab);
    }
  }
}

// One binning phase: every lane offers (bin, a, b) -- bin < 0 = nothing -- and bins[bin][0..1] += (a, b) over the warp,
// deterministically.  match.any gives every lane the mask of the lanes sharing its bin.  A lane alone with its bin adds
// straight to it (distinct bins: these adds do not meet).  One or two shared bins (the usual patch: one or two segments)
// take one fp32 butterfly each over the warp, the other lanes contributing zero -- a fixed tree.  More shared bins (a
// phase of queued strays) are all reduced at once by a tree over the peer masks: in every round a lane adds the value of
// its next peer above and the odd-ranked lanes of every group drop out, so the rounds needed are log2 of the largest
// group and the order of the additions is fixed by the lane numbers.  The first lane of a group adds its total to the bin.
__device__ __forceinline__ void bin_phase(double* bins, int bin, float a, float b, int lane) {
  bool add;                                                      // a lane adds at most once per phase: (a, b) end up holding its total
  const int bin0 = __shfl_sync(0xffffffffu, bin, 0);
  if (__all_sync(0xffffffffu, bin == bin0)) {                    // the usual patch: one segment across the warp's 32 columns
    f2 x = make_float2(a, b);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) x = x + make_float2(__shfl_xor_sync(0xffffffffu, x.x, o), __shfl_xor_sync(0xffffffffu, x.y, o));
    a = x.x; b = x.y;
    add = lane == 0 && bin >= 0;
  } else {
    const unsigned peers = __match_any_sync(0xffffffffu, bin >= 0 ? bin : -1 - lane);   // nothing to offer: a unique key
    const bool single = peers == (1u << lane);
    const bool first = (peers & (0u - peers)) == (1u << lane);
    unsigned active = __ballot_sync(0xffffffffu, bin >= 0 && first && !single);          // first lanes of the shared bins
    add = bin >= 0 && first;
    if (__popc(active) <= 2) {
      const float a0 = a, b0 = b;
      while (active) {
        const int leader = __ffs(active) - 1;
        const unsigned grp = __shfl_sync(0xffffffffu, peers, leader);
        const bool mine = (grp >> lane) & 1u;
        f2 x = mine ? make_float2(a0, b0) : make_float2(0.f, 0.f);
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) x = x + make_float2(__shfl_xor_sync(0xffffffffu, x.x, o), __shfl_xor_sync(0xffffffffu, x.y, o));
        if (lane == leader) { a = x.x; b = x.y; }
        active &= active - 1;
      }
    } else {
      int rank = __popc(peers & ((1u << lane) - 1u));
      unsigned above = peers & (0xfffffffeu << lane);
      while (__any_sync(0xffffffffu, above != 0u)) {
        const int next = __ffs(above);                           // 1 + lane of the next peer above, 0 if none
        const float ta = __shfl_sync(0xffffffffu, a, (next - 1) & 31), tb = __shfl_sync(0xffffffffu, b, (next - 1) & 31);
        if (next) { a += ta; b += tb; }
        above &= __ballot_sync(0xffffffffu, !(rank & 1));        // odd-ranked lanes have been absorbed: out of every mask
        rank >>= 1;
      }
    }
  }
  if (add) { bins[2 * bin] += (double)a; bins[2 * bin + 1] += (double)b; }   // distinct bins: these adds do not meet
  __syncwarp();                                                  // the next phase's adds may come from other lanes
}

struct DpQueue {       // per-warp queue of records waiting for a phase; head / tail are warp-uniform
  int32_t* bin;
  float *a, *b;
  int head, tail;
};

// lanes with `put` append (bin, a, b) in lane order
__device__ __forceinline__ void dp_push(DpQueue& q, bool put, int bin, float a, float b, int lane) {
  const unsigned bal = __ballot_sync(0xffffffffu, put);
  if (bal == 0u) return;
  if (put) {
    const int pos = (q.tail + __popc(bal & ((1u << lane) - 1u))) & (kDpQueue - 1);
    q.bin[pos] = bin; q.a[pos] = a; q.b[pos] = b;
  }
  q.tail += __popc(bal);
}

// full phases while 32 records wait; `all`: also the remainder.  The loop is a function of its own (one copy of the phase
// code instead of one per call site); the test in front of it is all that the common case executes.
__device__ __noinline__ int dp_drain_loop(const int32_t* qbin, const float* qa, const float* qb, int head, int tail, double* bins, bool all, int lane) {
  while (tail - head >= 32 || (all && tail > head)) {
    __syncwarp();                                                // the records were written by other lanes
    const bool have = lane < tail - head;
    const int pos = (head + lane) & (kDpQueue - 1);
    bin_phase(bins, have ? qbin[pos] : -1, have ? qa[pos] : 0.f, have ? qb[pos] : 0.f, lane);
    head += min(32, tail - head);
  }
  return head;
}
__device__ __forceinline__ void dp_drain(DpQueue& q, double* bins, bool all, int lane) {
  if (q.tail - q.head >= 32 || (all && q.tail > q.head)) q.head = dp_drain_loop(q.bin, q.a, q.b, q.head, q.tail, bins, all, lane);
}

// A lane walks DOWN one image column, so the segment of its pixels -- on both sides -- stays the same for many patches.  Per side
// it keeps ONE running record in registers: the label K and the sums (g, H) as an unevaluated fp32 pair hi + lo (TwoSum: the
// record is as accurate as one rounding of its exact sum, however long it runs).  Nothing is exchanged between lanes while
// the label lasts; the record goes to the queue when the label changes, and at the end of the warp's work.
struct DpRun {
  int K;                 // -2: empty
  f2 hi, lo;             // (g, H)
};

// The four records (key, a, b) of a lane -- its four vertically adjacent pixels -- of one side (`base` = first bin of the
// side): those of the running label (or, if none of the four carries it, of the lane's first valid pixel, which then
// becomes the running label) are added to the running record; the others (stray matches, a boundary inside the patch) are
// queued.  Every decision depends on the lane's own data only and the queue is filled in lane order: a fixed order.
__device__ __forceinline__ void bin_records(double* bins, DpQueue& q, DpRun& run, int base, const int (&key)[kDpRows],
                                            const float (&a)[kDpRows], const float (&b)[kDpRows], int lane) {
  bool hit = false;
#pragma unroll
  for (int r = 0; r < kDpRows; ++r) hit |= key[r] == run.K;      // run.K is never -1: an invalid pixel does not hit
  const int first = key[0] >= 0 ? key[0] : key[1] >= 0 ? key[1] : key[2] >= 0 ? key[2] : key[3];
  const int K = hit ? run.K : first;
  f2 s = make_float2(0.f, 0.f);
  bool extra[kDpRows];
#pragma unroll
  for (int r = 0; r < kDpRows; ++r) {
    const bool same = key[r] == K;
    s.x += same ? a[r] : 0.f;
    s.y += same ? b[r] : 0.f;
    extra[r] = key[r] >= 0 && !same;
  }
  const f2 out = run.hi + run.lo;
  dp_push(q, !hit && K >= 0 && run.K >= 0, base + run.K, out.x, out.y, lane);     // the label has changed: the old record leaves
  dp_drain(q, bins, false, lane);
  if (hit) {                                                      // hi + lo += s, error-free (Knuth's TwoSum on both lanes)
    const f2 t = run.hi + s;
    const f2 bb = t + (-run.hi);
    const f2 e = (run.hi + (-(t + (-bb)))) + (s + (-bb));
    run.hi = t;
    run.lo = run.lo + e;
  } else if (K >= 0) {
    run.K = K;
    run.hi = s;
    run.lo = make_float2(0.f, 0.f);
  }
#pragma unroll
  for (int r = 0; r < kDpRows; ++r) dp_push(q, extra[r], base + key[r], a[r], b[r], lane);   // at most three per lane
  dp_drain(q, bins, false, lane);
}

__global__ void __launch_bounds__(32 * kDpMaxWarps)
k_depth_edge(const float4* __restrict__ pm, const float4* __restrict__ rec, const int32_t* __restrict__ lab_n,
             const int32_t* __restrict__ edges, const int32_t* __restrict__ grp_edge, const int32_t* __restrict__ labels,
             const double* __restrict__ eta, const double* __restrict__ poses, int H, int W, int n_seg, int tiles, int tile_rows,
             DepthDev prm, double* __restrict__ partial) {
  extern __shared__ __align__(16) unsigned char dp_smem[];
  const int kDpWarps = blockDim.x >> 5, kDpThreads = blockDim.x;   // 4 or 2 warps (see the launcher)
  // [kDpWarps] rings + queues | [kDpWarps][2 sides][n_seg][2] FP64 bins | [kDpWarps] cost |
  // [n_seg] 8 floats: E_h (hi, lo), (1 - E_h) t_ij [3] (hi, lo) | [n_seg] float2 E_g (hi, lo)
  double* s_bins = reinterpret_cast<double*>(dp_smem + kDpWarpBytes * kDpWarps);
  double* s_cost = s_bins + (size_t)kDpWarps * 4 * n_seg;
  float4* s_Eh = reinterpret_cast<float4*>(s_cost + kDpWarps);      // two float4 per label (16-byte aligned: 128 n_seg + 32 bytes in)
  float2* s_Eg = reinterpret_cast<float2*>(s_Eh + 2 * n_seg);
  // launch order = kernel 1's: the edges sorted by (i, j), all tiles of an edge together, so the CTAs in flight cover a
  // few neighbouring keyframes completely and X_i and its labels are fetched from HBM once and shared through L2
  const int k = blockIdx.x / tiles, tile = blockIdx.x - k * tiles, e = grp_edge[k];
  const int i = edges[2 * e], j = edges[2 * e + 1];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int HW = H * W;
  const Sim3d T = relative_pose(load_pose(poses + 8 * i), load_pose(poses + 8 * j));   // T_ij
  for (int q = tid; q < kDpWarps * 4 * n_seg; q += kDpThreads) s_bins[q] = 0.0;
  auto split = [](double v, float& hi, float& lo) { hi = (float)v; lo = (float)(v - (double)hi); };
  for (int q = tid; q < n_seg; q += kDpThreads) {
    float2 g;
    split(exp(eta[(size_t)i * n_seg + q]), g.x, g.y);
    s_Eg[q] = g;
    const double eh = eta[(size_t)j * n_seg + q], ome = -expm1(eh);           // 1 - E_h
    float4 h0, h1;
    split(exp(eh), h0.x, h0.y);
    split(ome * T.t[0], h0.z, h0.w);
    split(ome * T.t[1], h1.x, h1.y);
    split(ome * T.t[2], h1.z, h1.w);
    s_Eh[2 * q] = h0;
    s_Eh[2 * q + 1] = h1;
  }
  __syncthreads();
  const float tf[3] = {(float)T.t[0], (float)T.t[1], (float)T.t[2]};
  const float4* __restrict__ Pi = pm + (size_t)i * HW;
  const float4* __restrict__ Rc = rec + (size_t)e * HW;
  const int32_t* __restrict__ li = labels + (size_t)i * HW;
  const int32_t* __restrict__ lh = lab_n + (size_t)e * HW;
  const float s_cap = prm.s_cap, k_cap = prm.k_cap, hk2 = prm.hk2;
  double* my_bins = s_bins + (size_t)warp * 4 * n_seg;
  unsigned char* wb = dp_smem + kDpWarpBytes * warp;
  float4* r_Xi = reinterpret_cast<float4*>(wb + kDpOffXi);
  float4* r_rec = reinterpret_cast<float4*>(wb + kDpOffRec);
  int32_t* r_li = reinterpret_cast<int32_t*>(wb + kDpOffLi);
  int32_t* r_lh = reinterpret_cast<int32_t*>(wb + kDpOffLh);
  DpQueue queue;
  queue.bin = reinterpret_cast<int32_t*>(wb + kDpOffQ);
  queue.a = reinterpret_cast<float*>(queue.bin + kDpQueue);
  queue.b = queue.a + kDpQueue;
  queue.head = queue.tail = 0;
  DpRun run_g, run_h;                                            // running records of the lane's column, side i and side j
  run_g.K = run_h.K = -2;
  run_g.hi = run_g.lo = run_h.hi = run_h.lo = make_float2(0.f, 0.f);

  // the tile: image rows [row_lo, row_hi); its items: (block of 32 columns, quad of rows); the blocks are dealt round-robin to the warps
  const int row_lo = tile * tile_rows, row_hi = min(H, row_lo + tile_rows);
  const int nblk = (W + kDpCols - 1) / kDpCols;
  const int my_blks = nblk > warp ? (nblk - warp + kDpWarps - 1) / kDpWarps : 0;           // blocks of 32 columns of this warp
  const int my_items = my_blks * ((row_hi - row_lo + kDpRows - 1) / kDpRows);              // warp-uniform trip count
  // Copies of the warp's next item into the next ring stage; pixels outside the tile / the image are masked.  Items are
  // dealt so that a warp walks DOWN a block of 32 columns (quad of rows by quad of rows) before it moves to its next
  // block: the four source pointers just advance by four image rows, no index arithmetic per copy.
  const int nrq = (row_hi - row_lo + kDpRows - 1) / kDpRows;
  const uint32_t u_Xi = dp_smem_u32(r_Xi) + 16u * lane, u_rec = dp_smem_u32(r_rec) + 16u * lane;
  const uint32_t u_li = dp_smem_u32(r_li) + 4u * lane, u_lh = dp_smem_u32(r_lh) + 4u * lane;
  const size_t rs16 = (size_t)W * 16, rs4 = (size_t)W * 4;      // bytes per image row
  int is_t = 0, is_rq = 0, is_col = warp * kDpCols + lane;      // state of the item to be issued next
  const char *gXi = nullptr, *gRc = nullptr, *gli = nullptr, *glh = nullptr;
  auto seek = [&]() {                                           // pointers to (row_lo, is_col); a masked column keeps them in range
    const size_t m0 = (size_t)row_lo * W + min(is_col, W - 1);
    gXi = reinterpret_cast<const char*>(Pi + m0);
    gRc = reinterpret_cast<const char*>(Rc + m0);
    gli = reinterpret_cast<const char*>(li + m0);
    glh = reinterpret_cast<const char*>(lh + m0);
  };
  seek();
  auto issue = [&]() {
    if (is_t < my_items) {
      const int row0 = row_lo + is_rq * kDpRows, st = (is_t % kDpStages) * kDpRows * 32;
      const bool col_ok = is_col < W;
      if (__all_sync(0xffffffffu, col_ok) && row0 + kDpRows <= row_hi) {            // interior item: sixteen plain copies
#pragma unroll
        for (int r = 0; r < kDpRows; ++r) {
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(u_Xi + 16u * (st + 32 * r)), "l"(gXi + r * rs16) : "memory");
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(u_rec + 16u * (st + 32 * r)), "l"(gRc + r * rs16) : "memory");
          asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(u_li + 4u * (st + 32 * r)), "l"(gli + r * rs4) : "memory");
          asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(u_lh + 4u * (st + 32 * r)), "l"(glh + r * rs4) : "memory");
        }
      } else {
#pragma unroll
        for (int r = 0; r < kDpRows; ++r) {
          if (col_ok && row0 + r < row_hi) {
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(u_Xi + 16u * (st + 32 * r)), "l"(gXi + r * rs16) : "memory");
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(u_rec + 16u * (st + 32 * r)), "l"(gRc + r * rs16) : "memory");
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(u_li + 4u * (st + 32 * r)), "l"(gli + r * rs4) : "memory");
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(u_lh + 4u * (st + 32 * r)), "l"(glh + r * rs4) : "memory");
          } else {
            r_Xi[st + 32 * r + lane] = make_float4(0.f, 0.f, 0.f, -1.f);     // finite values for the masked lanes' arithmetic
            r_rec[st + 32 * r + lane] = make_float4(0.f, 0.f, 0.f, 0.f);
            r_li[st + 32 * r + lane] = -1;
            r_lh[st + 32 * r + lane] = -1;
          }
        }
      }
      ++is_t;
      if (++is_rq == nrq) {                                      // next block of columns of this warp
        is_rq = 0;
        is_col += kDpWarps * kDpCols;
        seek();
      } else {
        gXi += kDpRows * rs16; gRc += kDpRows * rs16; gli += kDpRows * rs4; glh += kDpRows * rs4;
      }
    }
    dp_commit();                                                 // (possibly empty) group: uniform accounting
  };
  issue();
  f2 c_wr2 = make_float2(0.f, 0.f), c_min = make_float2(0.f, 0.f);   // sum om res^2, sum min(q res^2 / sigma^2, kappa^2): <= 4 items x 6 terms
  double cost = 0.0;
  for (int t = 0; t < my_items; ++t) {
    issue();
    dp_wait<1>();                                                // item t has landed
    const int st = (t % kDpStages) * kDpRows * 32 + lane;
    int kg[kDpRows], kh[kDpRows];
    float vg[kDpRows], Hg[kDpRows], vh[kDpRows], Hh[kDpRows];
    bool any_valid = false;
#pragma unroll
    for (int r = 0; r < kDpRows; ++r) {
      kh[r] = r_lh[st + 32 * r];                                 // >= 0 <=> the match counts (kernel P)
      kg[r] = kh[r] >= 0 ? r_li[st + 32 * r] : -1;
      vg[r] = Hg[r] = vh[r] = Hh[r] = 0.f;
      any_valid |= kh[r] >= 0;
    }
    if (__any_sync(0xffffffffu, any_valid)) {                    // whole invalid bands are skipped warp-uniformly
#pragma unroll
      for (int p = 0; p < kDpRows; p += 2) {                     // rows p, p + 1 in the two lanes of the packed arithmetic
        const float4 aA = r_Xi[st + 32 * p], yA = r_rec[st + 32 * p], aB = r_Xi[st + 32 * (p + 1)], yB = r_rec[st + 32 * (p + 1)];
        const float2 gA = s_Eg[max(kg[p], 0)], gB = s_Eg[max(kg[p + 1], 0)];
        const float4 hA0 = s_Eh[2 * max(kh[p], 0)], hA1 = s_Eh[2 * max(kh[p], 0) + 1];
        const float4 hB0 = s_Eh[2 * max(kh[p + 1], 0)], hB1 = s_Eh[2 * max(kh[p + 1], 0) + 1];
        const f2 a[3] = {make_float2(aA.x, aB.x), make_float2(aA.y, aB.y), make_float2(aA.z, aB.z)};
        const f2 y[3] = {make_float2(yA.x, yB.x), make_float2(yA.y, yB.y), make_float2(yA.z, yB.z)};
        const f2 ct_hi[3] = {make_float2(hA0.z, hB0.z), make_float2(hA1.x, hB1.x), make_float2(hA1.z, hB1.z)};
        const f2 ct_lo[3] = {make_float2(hA0.w, hB0.w), make_float2(hA1.y, hB1.y), make_float2(hA1.w, hB1.w)};
        const f2 Eg = make_float2(gA.x, gB.x), Eh = make_float2(hA0.x, hB0.x);
        // d = E_h - E_g as an unevaluated pair (dh, dl): the difference of the leading parts is exact whenever the two
        // scales lie within a factor of two of each other (Sterbenz), and otherwise |res| is of the order of |d| |X_i| itself
        const f2 dh = Eh + (-Eg);
        const f2 dl = make_float2(hA0.y, hB0.y) + (-make_float2(gA.y, gB.y));
        // sqrt(q) = w_i w_j from kernel P, 0 for a masked lane: all its weights vanish
        const f2 sq = make_float2(yA.w, yB.w);
        const f2 q = sq * sq;
        const f2 sc = q * bc(s_cap), kc = sq * bc(k_cap);        // q / sigma^2 and kappa sqrt(q) / sigma
        f2 pvg = make_float2(0.f, 0.f), pHg = pvg, pvh = pvg, pHh = pvg;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          // res = E_h y + [(E_h - E_g) X_i + (1 - E_h) t]: two nested fused multiply-adds on the leading parts -- each rounds
          // its exact sum once, so what is lost is 2^-24 of the partial result, random from match to match like the rounding y
          // itself carries -- plus the trailing parts, which carry the per-segment (systematic) bits
          const f2 res = fma2(Eh, y[c], fma2(dh, a[c], ct_hi[c])) + fma2(dl, a[c], ct_lo[c]);
          const f2 xi = Eg * a[c];                               // X_i(eta)
          // omega = q w / sigma^2 = min(q / sigma^2, kappa sqrt(q) / (sigma |res|));  rho = omega res^2 - min(q res^2 / sigma^2, kappa^2) / 2
          const f2 tt = kc * make_float2(rcp(fabsf(res.x)), rcp(fabsf(res.y)));
          const f2 om = make_float2(fminf(sc.x, tt.x), fminf(sc.y, tt.y));     // fminf(s, NaN) = s (masked lane: sq = 0)
          const f2 f = om * res;
          c_wr2 = fma2(f, res, c_wr2);
          const f2 r2 = (sc * res) * res;
          c_min = c_min + make_float2(fminf(r2.x, hk2), fminf(r2.y, hk2));
          const f2 Jh = (res + xi) + bc(-tf[c]);                 // J_h = s_ij R_ij X_j(eta) = res - t_ij + X_i(eta)
          pvg = fma2(-f, xi, pvg);                               // J_g = -X_i(eta)
          pHg = fma2(om * xi, xi, pHg);
          pvh = fma2(f, Jh, pvh);
          pHh = fma2(om * Jh, Jh, pHh);
        }
        vg[p] = pvg.x; vg[p + 1] = pvg.y; Hg[p] = pHg.x; Hg[p + 1] = pHg.y;
        vh[p] = pvh.x; vh[p + 1] = pvh.y; Hh[p] = pHh.x; Hh[p + 1] = pHh.y;
      }
      bin_records(my_bins, queue, run_g, 0, kg, vg, Hg, lane);
      bin_records(my_bins, queue, run_h, n_seg, kh, vh, Hh, lane);
    }
    if ((t & 3) == 3) {                                          // fp32 partials of <= 48 terms -> FP64
      cost += (double)(c_wr2.x + c_wr2.y) - 0.5 * (double)(c_min.x + c_min.y);
      c_wr2 = c_min = make_float2(0.f, 0.f);
    }
  }
  dp_wait<0>();
  {
    const f2 og = run_g.hi + run_g.lo, oh = run_h.hi + run_h.lo;
    dp_push(queue, run_g.K >= 0, run_g.K, og.x, og.y, lane);
    dp_drain(queue, my_bins, false, lane);
    dp_push(queue, run_h.K >= 0, n_seg + run_h.K, oh.x, oh.y, lane);
    dp_drain(queue, my_bins, true, lane);
  }
  cost += (double)(c_wr2.x + c_wr2.y) - 0.5 * (double)(c_min.x + c_min.y);
  cost = warp_sum(cost);
  if (lane == 0) s_cost[warp] = cost;
  __syncthreads();
  double* out = partial + ((size_t)e * tiles + tile) * (4 * n_seg + 1);
  for (int q = tid; q < 4 * n_seg; q += kDpThreads) {           // q = (side, label, {g, H})
    double v = 0.0;
    for (int w = 0; w < kDpWarps; ++w) v += s_bins[(size_t)w * 4 * n_seg + q];
    out[q] = v;
  }
  if (tid == 0) {
    double v = 0.0;
    for (int w = 0; w < kDpWarps; ++w) v += s_cost[w];
    out[4 * n_seg] = v;
  }
}

__global__ void k_depth_update(const double* __restrict__ partial, const double* __restrict__ eta_in, double* __restrict__ eta_out,
                               const int32_t* __restrict__ edges, const int32_t* __restrict__ kf_ptr, const int32_t* __restrict__ kf_edge,
                               const int32_t* __restrict__ sp_ptr, const int32_t* __restrict__ sp_other, const double* __restrict__ sp_delta,
                               const uint8_t* __restrict__ anchor, int n_seg, int n_total, int tiles, DepthDev prm) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n_total) return;
  const int k = s / n_seg, lab = s - k * n_seg;
  const double es = eta_in[s];
  if (anchor[k]) { eta_out[s] = es; return; }
  double g = prm.lambda_prior * es, H = prm.lambda_prior;
  const int rec = 4 * n_seg + 1;
  for (int p = kf_ptr[k]; p < kf_ptr[k + 1]; ++p) {
    const int e = kf_edge[p];
    const int side = (edges[2 * e] == k) ? 0 : 1;
    for (int t = 0; t < tiles; ++t) {
      const double* r = partial + ((size_t)e * tiles + t) * rec + (size_t)side * 2 * n_seg + 2 * lab;
      g += r[0];
      H += r[1];
    }
  }
  for (int p = sp_ptr[s]; p < sp_ptr[s + 1]; ++p) {          // sp_delta carries the sign: d = eta_s - eta_other + delta
    g += prm.lambda_smooth * (es - eta_in[sp_other[p]] + sp_delta[p]);
    H += prm.lambda_smooth;
  }
  double step = -g / ((1.0 + prm.lambda_lm) * H);
  step = fmin(fmax(step, -prm.eta_max), prm.eta_max);
  eta_out[s] = es + step;
}

// The objective of an iteration (Eq. (9) data term from the per-CTA records, boundary and prior terms of Eq. (10)), in two
// stages with a fixed order: CTA j of kDpCostCtas sums slice j of the records, of the pairs and of the segments (thread
// partials, then a shared-memory tree) into stage[j]; the CTA that arrives last (a counter that it also resets) adds the
// kDpCostCtas slice sums in index order.  One 1024-thread CTA over everything took 100 us on config 5.
constexpr int kDpCostThreads = 256, kDpCostCtas = 64;
__global__ void __launch_bounds__(kDpCostThreads)
k_depth_cost(const double* __restrict__ partial, int n_rec, int rec, const double* __restrict__ eta, int n_total,
             const int32_t* __restrict__ pairs, const double* __restrict__ delta, int n_pairs, DepthDev prm, double* __restrict__ stage,
             unsigned int* __restrict__ counter, double* __restrict__ out) {
  __shared__ double s[kDpCostThreads];
  __shared__ bool last;
  const int j = blockIdx.x, tid = threadIdx.x;
  auto slice = [&](int n, int& lo, int& hi) { const int per = (n + kDpCostCtas - 1) / kDpCostCtas; lo = min(n, j * per); hi = min(n, lo + per); };
  double v = 0.0;
  int lo, hi;
  slice(n_rec, lo, hi);
  for (int q = lo + tid; q < hi; q += kDpCostThreads) v += __ldcg(partial + (size_t)q * rec + rec - 1);
  slice(n_pairs, lo, hi);
  for (int q = lo + tid; q < hi; q += kDpCostThreads) {
    const double d = eta[pairs[2 * q]] - eta[pairs[2 * q + 1]] + delta[q];
    v += 0.5 * prm.lambda_smooth * d * d;
  }
  slice(n_total, lo, hi);
  for (int q = lo + tid; q < hi; q += kDpCostThreads) v += 0.5 * prm.lambda_prior * eta[q] * eta[q];
  s[tid] = v;
  __syncthreads();
  for (int o = kDpCostThreads / 2; o > 0; o >>= 1) {
    if (tid < o) s[tid] += s[tid + o];
    __syncthreads();
  }
  if (tid == 0) {
    stage[j] = s[0];
    __threadfence();
    last = atomicAdd(counter, 1u) == (unsigned)(kDpCostCtas - 1);
  }
  __syncthreads();
  if (last && tid == 0) {
    __threadfence();
    double t = 0.0;
    for (int q = 0; q < kDpCostCtas; ++q) t += __ldcg(stage + q);
    *out = t;
    *counter = 0u;                                            // ready for the next iteration (stream order)
  }
}

// pm <- packed (exp(eta_label) X, w): the pointmap the next pose passes see (alternation of PAPER.md:143)
__global__ void k_depth_apply(const float* __restrict__ pts, const float* __restrict__ conf, const int32_t* __restrict__ labels,
                              const double* __restrict__ eta, float4* __restrict__ pm, int HW, int n_seg, size_t total, float conf_min) {
  size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; idx < total; idx += stride) {
    const float c = conf[idx];
    const int lab = labels[idx];
    const size_t k = idx / (size_t)HW;
    const double sc = (lab >= 0 && lab < n_seg) ? exp(eta[k * n_seg + lab]) : 1.0;
    pm[idx] = make_float4((float)(sc * (double)pts[3 * idx]), (float)(sc * (double)pts[3 * idx + 1]), (float)(sc * (double)pts[3 * idx + 2]),
                          (c > conf_min) ? sqrtf(sqrtf(fmaxf(c, 0.f))) : -1.f);
  }
}

template <class T>
cudaError_t up(T** dst, const std::vector<T>& src, cudaStream_t s) {
  cudaError_t e = dmalloc(reinterpret_cast<void**>(dst), std::max<size_t>(src.size(), 1) * sizeof(T));
  if (e != cudaSuccess || src.empty()) return e;
  return cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s);
}

}  // namespace

cudaError_t run_depth_refine(Ctx* c, const int32_t* d_labels, int n_seg, const int32_t* h_pairs, const double* h_delta, int n_pairs,
                             const int32_t* h_anchor, int n_anchor, const sim3ba_depth_params& p, int n_iters, double* d_eta,
                             double* h_cost) {
  const int n_total = c->N * n_seg;
  // tiles of whole image rows, ~kDpTilePx pixels each (the per-CTA setup is ~2000 shared-memory words), at least ~4 CTAs per SM in the grid
  const int E1 = std::max(c->E, 1);
  const int want_tiles = std::max((c->HW + kDpTilePx - 1) / kDpTilePx, (592 + E1 - 1) / E1);
  const int tile_rows = std::max(kDpRows, ((c->H + want_tiles - 1) / want_tiles + kDpRows - 1) / kDpRows * kDpRows);
  const int tiles = (c->H + tile_rows - 1) / tile_rows;
  const int rec = 4 * n_seg + 1;
  const int kDpWarps = n_seg <= 64 ? kDpMaxWarps : 2, kDpThreads = 32 * kDpWarps;
  const size_t smem = kDpWarpBytes * kDpWarps + ((size_t)kDpWarps * 4 * n_seg + kDpWarps) * sizeof(double) + (size_t)n_seg * 40;
  if (smem > c->depth_smem) {
    cudaError_t ea = cudaFuncSetAttribute(k_depth_edge, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (ea != cudaSuccess) return ea;
    c->depth_smem = smem;
  }
  const float4* pm_init = c->pm0 ? c->pm0 : c->pm;               // pristine X_init (Eq. (8)): see sim3ba_apply_depth
  DepthDev dev{1.0 / (double)p.sigma_point, (double)p.huber_k, p.lambda_smooth, p.lambda_prior, p.lambda_lm, p.eta_max, 0.f, 0.f, 0.f};
  {
    const float isg = (float)dev.inv_sigma, hk = (float)dev.huber_k;
    dev.s_cap = isg * isg; dev.k_cap = hk * isg; dev.hk2 = hk * hk;
  }
  // segment -> boundary pairs CSR (host), the sign of Delta folded in: d = eta_s - eta_other + delta'
  std::vector<int32_t> sp_ptr(n_total + 1, 0), sp_other(2 * (size_t)n_pairs), pairs(h_pairs, h_pairs + 2 * (size_t)n_pairs);
  std::vector<double> sp_delta(2 * (size_t)n_pairs), delta(h_delta, h_delta + n_pairs);
  for (int q = 0; q < n_pairs; ++q) { ++sp_ptr[pairs[2 * q] + 1]; ++sp_ptr[pairs[2 * q + 1] + 1]; }
  for (int s = 0; s < n_total; ++s) sp_ptr[s + 1] += sp_ptr[s];
  {
    std::vector<int32_t> cur(sp_ptr.begin(), sp_ptr.end() - 1);
    for (int q = 0; q < n_pairs; ++q) {
      const int a = pairs[2 * q], b = pairs[2 * q + 1];
      sp_other[cur[a]] = b; sp_delta[cur[a]++] = delta[q];        // d(eta_a) of ((eta_a - eta_b) + D)^2 / 2
      sp_other[cur[b]] = a; sp_delta[cur[b]++] = -delta[q];       // d(eta_b): -(eta_a - eta_b + D) = eta_b - eta_a - D
    }
  }
  std::vector<uint8_t> anchor(c->N, 0);
  for (int k = 0; k < n_anchor; ++k) anchor[h_anchor[k]] = 1;
  int32_t *d_sp_ptr = nullptr, *d_sp_other = nullptr, *d_pairs = nullptr;
  double *d_sp_delta = nullptr, *d_delta = nullptr, *d_partial = nullptr, *d_eta2 = nullptr, *d_cost = nullptr;
  uint8_t* d_anchor = nullptr;
  float4* d_rec = nullptr;        // kernel P's per-candidate records: y [3], sqrt(q) -- 20 bytes per candidate with the label below
  int32_t* d_labn = nullptr;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; return e == cudaSuccess; };
  ok(up(&d_sp_ptr, sp_ptr, c->stream)); ok(up(&d_sp_other, sp_other, c->stream)); ok(up(&d_sp_delta, sp_delta, c->stream));
  ok(up(&d_pairs, pairs, c->stream)); ok(up(&d_delta, delta, c->stream)); ok(up(&d_anchor, anchor, c->stream));
  ok(dmalloc(reinterpret_cast<void**>(&d_partial), std::max<size_t>((size_t)c->E * tiles * rec, 1) * sizeof(double)));
  ok(dmalloc(reinterpret_cast<void**>(&d_eta2), std::max<size_t>(n_total, 1) * sizeof(double)));
  ok(dmalloc(reinterpret_cast<void**>(&d_cost), (std::max(n_iters, 1) + kDpCostCtas + 1) * sizeof(double)));   // [n_iters] costs, [kDpCostCtas] stage, counter
  const size_t EHW = (size_t)c->E * c->HW;
  ok(dmalloc(reinterpret_cast<void**>(&d_rec), std::max<size_t>(EHW, 1) * sizeof(float4)));
  ok(dmalloc(reinterpret_cast<void**>(&d_labn), std::max<size_t>(EHW, 1) * sizeof(int32_t)));
  if (e == cudaSuccess && c->E > 0 && n_iters > 0) {
    const int chunks = std::max(1, std::min((c->HW + 4095) / 4096, 65535));
    k_depth_prep<<<c->E * chunks, 256, 0, c->stream>>>(pm_init, c->match, c->edges, c->grp_edge, d_labels, c->poses, c->HW, n_seg, chunks, d_rec, d_labn);
    ++c->launches;
    ok(cudaGetLastError());
  }
  double* d_stage = d_cost + std::max(n_iters, 1);            // slice sums of k_depth_cost, then its arrival counter (zeroed here, reset by the kernel)
  if (e == cudaSuccess) ok(cudaMemsetAsync(d_stage + kDpCostCtas, 0, sizeof(double), c->stream));
  double *cur = d_eta, *nxt = d_eta2;
  for (int it = 0; it < n_iters && e == cudaSuccess; ++it) {
    if (c->E > 0)
      k_depth_edge<<<c->E * tiles, kDpThreads, smem, c->stream>>>(pm_init, d_rec, d_labn, c->edges, c->grp_edge, d_labels, cur, c->poses, c->H, c->W,
                                                                 n_seg, tiles, tile_rows, dev, d_partial);
    k_depth_cost<<<kDpCostCtas, kDpCostThreads, 0, c->stream>>>(d_partial, c->E * tiles, rec, cur, n_total, d_pairs, d_delta, n_pairs, dev, d_stage,
                                                               reinterpret_cast<unsigned int*>(d_stage + kDpCostCtas), d_cost + it);
    k_depth_update<<<(n_total + 127) / 128, 128, 0, c->stream>>>(d_partial, cur, nxt, c->edges, c->kf_ptr, c->kf_edge, d_sp_ptr, d_sp_other,
                                                                 d_sp_delta, d_anchor, n_seg, n_total, tiles, dev);
    c->launches += 3;
    ok(cudaGetLastError());
    std::swap(cur, nxt);
  }
  if (e == cudaSuccess && cur != d_eta) ok(cudaMemcpyAsync(d_eta, cur, (size_t)n_total * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  if (e == cudaSuccess && h_cost && n_iters > 0) ok(cudaMemcpyAsync(h_cost, d_cost, (size_t)n_iters * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  cudaError_t es = cudaStreamSynchronize(c->stream);          // the host vectors and temporaries go out of scope
  if (e == cudaSuccess) e = es;
  dfree(d_sp_ptr); dfree(d_sp_other); dfree(d_sp_delta); dfree(d_pairs); dfree(d_delta); dfree(d_anchor);
  dfree(d_partial); dfree(d_eta2); dfree(d_cost); dfree(d_rec); dfree(d_labn);
  return e;
}

cudaError_t launch_depth_apply(Ctx* c, const float* d_points, const float* d_conf, const int32_t* d_labels, int n_seg, const double* d_eta) {
  const size_t total = (size_t)c->N * c->HW;
  if (!c->pm0) {   // first application: keep the pristine packed pointmaps for the structure passes that follow (Eq. (8): eta is absolute)
    cudaError_t e = dmalloc(reinterpret_cast<void**>(&c->pm0), total * sizeof(float4));
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(c->pm0, c->pm, total * sizeof(float4), cudaMemcpyDeviceToDevice, c->stream);
    if (e != cudaSuccess) return e;
  }
  const int grid = (int)std::min<size_t>((total + 255) / 256, 148 * 16);
  k_depth_apply<<<grid, 256, 0, c->stream>>>(d_points, d_conf, d_labels, d_eta, c->pm, c->HW, n_seg, total, c->prm.conf_min);
  ++c->launches;
  return cudaGetLastError();
}

int depth_max_segments() { return kDpMaxSeg; }

}  // namespace sim3ba
