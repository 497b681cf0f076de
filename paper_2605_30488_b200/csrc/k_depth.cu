// Segment-level structure refinement with the poses held fixed.
//
//   Eq. (8)  :130   X_{k,p}(eta_g) = exp(eta_g) X_init (one log-scale eta_g per segment g of keyframe k)
//   Eq. (9)  :134   r_c = sqrt(q) [T_ij X_j,n(eta) - X_i,m(eta)]_c / sigma_point, per-component Huber
//   :143            J_g = -X_i,m(eta), J_h = s_ij R_ij X_j,n(eta); only H_gg, H_hh of the data term, complete gradient;
//                   boundary term ((eta_g - eta_h) + Delta_gh)^2 and prior eta_g^2 Jacobi-decoupled likewise;
//                   Delta eta_g = -g_g / ((1 + lambda_lm) H_gg), clipped to eta_max, anchor keyframes fixed
// Conventions D1-D5 of DESIGN.md section 10 (objective = sum rho + lambda_s/2 E_bnd + lambda_p/2 E_prior).
//
// Kernel A (k_depth_edge): one CTA per (edge, tile of the pixels of i), in kernel 1's order (edges sorted by keyframe,
// the tiles of an edge together: X_j and the labels are shared through L2).  Every thread evaluates TWO adjacent
// pixels at a time in the two lanes of packed fp32x2 instructions.  Precision plan (the one of kernel 1): the one
// cancellation -- res = T_ij X_j(eta) - X_i(eta), a difference of two ~10 m points -- is evaluated in FP64 and rounded
// once; everything after it per match is fp32; fp32 partial sums hold at most 64 terms (the two matches of a lane and
// one 32-lane butterfly), every sum from there upwards is FP64.  The loads run in a software pipeline (streams two
// iterations ahead, gathers one).  The per-segment sums are binned WITHOUT atomics in per-warp FP64 shared-memory bins
// (dynamic shared memory: 32 n_seg bytes per warp): a lane whose label is alone in its warp adds straight to the bin,
// a label shared by several lanes takes one fp32 butterfly over the peers found by match.any; the eight warps' bins are
// added in a fixed order -> one record [2 sides][n_seg][g, H] + cost per (edge, tile).  Bit-reproducible run to run.
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

constexpr int kDpThreads = 256;
constexpr int kDpWarps = kDpThreads / 32;
constexpr int kDpMaxSeg = 512;       // labels per keyframe (the paper's SLIC pass: M_k ~ 200); 16 KB of bins per warp at 512
#ifndef SIM3BA_DP_CTAS
#define SIM3BA_DP_CTAS 2
#endif
#ifndef SIM3BA_DP_TILE_PX
#define SIM3BA_DP_TILE_PX 16384
#endif
constexpr int kDpTilePx = SIM3BA_DP_TILE_PX;
constexpr int kDpIterPx = 2 * kDpThreads;   // pixels of the tile one CTA iteration covers (two adjacent pixels per thread)

struct DepthDev {
  double inv_sigma, huber_k, lambda_smooth, lambda_prior, lambda_lm, eta_max;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// One binning phase: every lane offers (key, a, b) -- key < 0 = nothing -- and bins[key][0..1] += (a, b) over the warp,
// deterministically.  match.any gives every lane the mask of the lanes carrying its key: a lane alone with its key (a
// stray match landing in some far segment) adds straight to the bin -- distinct keys, so these adds do not meet; a key
// shared by several lanes takes one fp32 butterfly over the warp with the other lanes contributing zero (a fixed tree,
// <= 32 x 2 terms) and its first lane adds the total.  The usual warp (one or two segments, a few strays) takes one or
// two butterflies.
__device__ __forceinline__ void bin_phase(double* bins, int key, float a, float b, int lane) {
  const unsigned peers = __match_any_sync(0xffffffffu, key >= 0 ? key : -1 - lane);   // nothing to offer: a unique key
  const bool single = key >= 0 && peers == (1u << lane);
  if (single) { bins[2 * key] += (double)a; bins[2 * key + 1] += (double)b; }
  unsigned active = __ballot_sync(0xffffffffu, key >= 0 && !single);
  while (active) {
    const int leader = __ffs(active) - 1;
    const unsigned grp = __shfl_sync(0xffffffffu, peers, leader);
    const bool mine = (grp >> lane) & 1u;
    f2 x = mine ? make_float2(a, b) : make_float2(0.f, 0.f);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) x = x + make_float2(__shfl_xor_sync(0xffffffffu, x.x, o), __shfl_xor_sync(0xffffffffu, x.y, o));
    if (lane == leader) { bins[2 * key] += (double)x.x; bins[2 * key + 1] += (double)x.y; }
    active &= ~grp;
  }
  __syncwarp();                                                // the next phase's adds may come from other lanes
}

// The two matches (A, B) of every lane -> bins: equal keys are merged in the lane first (adjacent pixels mostly share
// their segment), then one phase for the A slots and, if any lane still holds a B, one for the B slots.
__device__ __forceinline__ void bin_pair(double* bins, int keyA, int keyB, f2 a, f2 b, int lane) {
  if (keyA >= 0 && keyA == keyB) { a.x += a.y; b.x += b.y; keyB = -1; }
  else if (keyA < 0 && keyB >= 0) { keyA = keyB; a.x = a.y; b.x = b.y; keyB = -1; }
  bin_phase(bins, keyA, a.x, b.x, lane);
  if (__any_sync(0xffffffffu, keyB >= 0)) bin_phase(bins, keyB, a.y, b.y, lane);
}

struct DepthStream {     // the streamed loads of one CTA iteration: two adjacent pixels m, m + 1 of keyframe i
  int nA, nB, lgA, lgB;
  float4 aA, aB;
};

__global__ void __launch_bounds__(kDpThreads, SIM3BA_DP_CTAS)
k_depth_edge(const float4* __restrict__ pm, const int32_t* __restrict__ match, const int32_t* __restrict__ edges,
             const int32_t* __restrict__ grp_edge, const int32_t* __restrict__ labels, const double* __restrict__ eta,
             const double* __restrict__ poses, int HW, int n_seg, int tiles, int per, DepthDev prm, double* __restrict__ partial) {
  extern __shared__ __align__(16) unsigned char dp_smem[];
  // [kDpWarps][2 sides][n_seg][2] FP64 bins | [2][n_seg] exp(eta) FP64 | [2][n_seg] exp(eta) fp32 | [kDpWarps] cost
  double* s_bins = reinterpret_cast<double*>(dp_smem);
  double* s_exp = s_bins + (size_t)kDpWarps * 4 * n_seg;
  double* s_cost = s_exp + 2 * n_seg;
  float* s_expf = reinterpret_cast<float*>(s_cost + kDpWarps);
  // launch order = kernel 1's: the edges sorted by (i, j), all tiles of an edge together, so the CTAs in flight cover a
  // few neighbouring keyframes completely and X_i, X_j and the labels are fetched from HBM once and shared through L2
  const int k = blockIdx.x / tiles, tile = blockIdx.x - k * tiles, e = grp_edge[k];
  const int i = edges[2 * e], j = edges[2 * e + 1];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int q = tid; q < kDpWarps * 4 * n_seg; q += kDpThreads) s_bins[q] = 0.0;
  for (int q = tid; q < 2 * n_seg; q += kDpThreads) {
    const double ev = exp(eta[(size_t)(q < n_seg ? i : j) * n_seg + (q < n_seg ? q : q - n_seg)]);
    s_exp[q] = ev;
    s_expf[q] = (float)ev;
  }
  __syncthreads();
  const Sim3d T = relative_pose(load_pose(poses + 8 * i), load_pose(poses + 8 * j));   // T_ij
  double sR[9];
#pragma unroll
  for (int q = 0; q < 9; ++q) sR[q] = T.s * T.R[q];
  const float tf[3] = {(float)T.t[0], (float)T.t[1], (float)T.t[2]};
  const float4* __restrict__ Pi = pm + (size_t)i * HW;
  const float4* __restrict__ Pj = pm + (size_t)j * HW;
  const int32_t* __restrict__ mt = match + (size_t)e * HW;
  const int32_t* __restrict__ li = labels + (size_t)i * HW;
  const int32_t* __restrict__ lj = labels + (size_t)j * HW;
  const int m0 = tile * per, m1 = min(HW, m0 + per);
  const float isg = (float)prm.inv_sigma, hk = (float)prm.huber_k;
  const float s_cap = isg * isg, k_cap = hk * isg, hk2 = hk * hk;
  double* my_bins = s_bins + (size_t)warp * 4 * n_seg;
  // Software pipeline over the CTA's iterations (warp-uniform trip count: the binning uses full-warp shuffles): the
  // streamed loads (match index, X_i, label of m) run two iterations ahead, the gathers they address (X_j, label of n) one.
  const int niter = (m1 - m0 + kDpIterPx - 1) / kDpIterPx;
  auto load_stream = [&](int it, DepthStream& s) {
    const int m = m0 + it * kDpIterPx + 2 * tid;
    s.nA = s.nB = -1;
    if (it < niter) {
      if (m < m1) { s.nA = __ldcs(mt + m); s.aA = Pi[m]; s.lgA = li[m]; }
      if (m + 1 < m1) { s.nB = __ldcs(mt + m + 1); s.aB = Pi[m + 1]; s.lgB = li[m + 1]; }
    }
  };
  auto load_gather = [&](int n, float4& b, int& lh) {
    if ((unsigned)n < (unsigned)HW) { b = Pj[n]; lh = lj[n]; }
  };
  const float4 none = make_float4(0.f, 0.f, 0.f, -1.f);
  DepthStream s0, s1, s2;
  s0.aA = s0.aB = s1.aA = s1.aB = s2.aA = s2.aB = none;
  s0.lgA = s0.lgB = s1.lgA = s1.lgB = s2.lgA = s2.lgB = -1;
  float4 bA0 = none, bB0 = none, bA1 = none, bB1 = none;
  int lhA0 = -1, lhB0 = -1, lhA1 = -1, lhB1 = -1;
  load_stream(0, s0);
  load_stream(1, s1);
  load_gather(s0.nA, bA0, lhA0);
  load_gather(s0.nB, bB0, lhB0);
  f2 c_wr2 = make_float2(0.f, 0.f), c_min = make_float2(0.f, 0.f);   // sum om res^2, sum min(q res^2 / sigma^2, kappa^2): <= 8 iterations x 3
  double cost = 0.0;
  for (int it = 0; it < niter; ++it) {
    load_stream(it + 2, s2);
    load_gather(s1.nA, bA1, lhA1);
    load_gather(s1.nB, bB1, lhB1);
    const bool vA = (unsigned)s0.nA < (unsigned)HW && s0.aA.w >= 0.f && bA0.w >= 0.f && (unsigned)s0.lgA < (unsigned)n_seg &&
                    (unsigned)lhA0 < (unsigned)n_seg;
    const bool vB = (unsigned)s0.nB < (unsigned)HW && s0.aB.w >= 0.f && bB0.w >= 0.f && (unsigned)s0.lgB < (unsigned)n_seg &&
                    (unsigned)lhB0 < (unsigned)n_seg;
    const int kgA = vA ? s0.lgA : -1, kgB = vB ? s0.lgB : -1, khA = vA ? lhA0 : -1, khB = vB ? lhB0 : -1;
    f2 vg = make_float2(0.f, 0.f), Hg = vg, vh = vg, Hh = vg;
    if (__any_sync(0xffffffffu, vA || vB)) {                    // whole invalid bands are skipped warp-uniformly
      // res = s_ij R_ij (e^eta_h X_j) + t_ij - e^eta_g X_i in FP64, rounded once; masked lanes run on zeros
      const int gA = vA ? s0.lgA : 0, gB = vB ? s0.lgB : 0, hA = vA ? lhA0 : 0, hB = vB ? lhB0 : 0;
      f2 res[3], xi[3];
      {
        const float4 a = s0.aA, b = bA0;
        const double eg = s_exp[gA], eh = s_exp[n_seg + hA];
        const double X0 = eh * (double)b.x, X1 = eh * (double)b.y, X2 = eh * (double)b.z;
        res[0].x = (float)fma(-eg, (double)a.x, fma(sR[0], X0, fma(sR[1], X1, fma(sR[2], X2, T.t[0]))));
        res[1].x = (float)fma(-eg, (double)a.y, fma(sR[3], X0, fma(sR[4], X1, fma(sR[5], X2, T.t[1]))));
        res[2].x = (float)fma(-eg, (double)a.z, fma(sR[6], X0, fma(sR[7], X1, fma(sR[8], X2, T.t[2]))));
        const float ef = s_expf[gA];
        xi[0].x = ef * a.x; xi[1].x = ef * a.y; xi[2].x = ef * a.z;
      }
      {
        const float4 a = s0.aB, b = bB0;
        const double eg = s_exp[gB], eh = s_exp[n_seg + hB];
        const double X0 = eh * (double)b.x, X1 = eh * (double)b.y, X2 = eh * (double)b.z;
        res[0].y = (float)fma(-eg, (double)a.x, fma(sR[0], X0, fma(sR[1], X1, fma(sR[2], X2, T.t[0]))));
        res[1].y = (float)fma(-eg, (double)a.y, fma(sR[3], X0, fma(sR[4], X1, fma(sR[5], X2, T.t[1]))));
        res[2].y = (float)fma(-eg, (double)a.z, fma(sR[6], X0, fma(sR[7], X1, fma(sR[8], X2, T.t[2]))));
        const float ef = s_expf[gB];
        xi[0].y = ef * a.x; xi[1].y = ef * a.y; xi[2].y = ef * a.z;
      }
      // sqrt(q) = w_i w_j (w = c^(1/4)), 0 for a masked lane: all its weights vanish
      f2 sq = make_float2(s0.aA.w * bA0.w, s0.aB.w * bB0.w);
      sq.x = vA ? sq.x : 0.f;
      sq.y = vB ? sq.y : 0.f;
      const f2 q = sq * sq;
      const f2 sc = q * bc(s_cap), kc = sq * bc(k_cap);       // q / sigma^2 and kappa sqrt(q) / sigma
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        // omega = q w / sigma^2 = min(q / sigma^2, kappa sqrt(q) / (sigma |res|));  rho = omega res^2 - min(q res^2 / sigma^2, kappa^2) / 2
        const f2 t = kc * make_float2(rcp(fabsf(res[c].x)), rcp(fabsf(res[c].y)));
        const f2 om = make_float2(fminf(sc.x, t.x), fminf(sc.y, t.y));     // fminf(s, NaN) = s (masked lane, res = 0)
        const f2 f = om * res[c];
        c_wr2 = fma2(f, res[c], c_wr2);
        const f2 r2 = (sc * res[c]) * res[c];
        c_min = c_min + make_float2(fminf(r2.x, hk2), fminf(r2.y, hk2));
        const f2 Jh = (res[c] + xi[c]) + bc(-tf[c]);            // J_h = s_ij R_ij X_j(eta) = res - t_ij + X_i(eta)
        vg = fma2(-f, xi[c], vg);                               // J_g = -X_i(eta)
        Hg = fma2(om * xi[c], xi[c], Hg);
        vh = fma2(f, Jh, vh);
        Hh = fma2(om * Jh, Jh, Hh);
      }
      bin_pair(my_bins, kgA, kgB, vg, Hg, lane);
      bin_pair(my_bins + 2 * n_seg, khA, khB, vh, Hh, lane);
    }
    if ((it & 7) == 7) {                                        // fp32 partials of <= 48 terms -> FP64
      cost += (double)(c_wr2.x + c_wr2.y) - 0.5 * (double)(c_min.x + c_min.y);
      c_wr2 = c_min = make_float2(0.f, 0.f);
    }
    s0 = s1; bA0 = bA1; bB0 = bB1; lhA0 = lhA1; lhB0 = lhB1;
    s1 = s2;
  }
  cost += (double)(c_wr2.x + c_wr2.y) - 0.5 * (double)(c_min.x + c_min.y);
  cost = warp_sum(cost);
  if (lane == 0) s_cost[warp] = cost;
  __syncthreads();
  double* out = partial + ((size_t)e * tiles + tile) * (4 * n_seg + 1);
  for (int q = tid; q < 4 * n_seg; q += kDpThreads) {          // q = (side, label, {g, H})
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < kDpWarps; ++w) v += s_bins[(size_t)w * 4 * n_seg + q];
    out[q] = v;
  }
  if (tid == 0) {
    double v = 0.0;
#pragma unroll
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

__global__ void __launch_bounds__(256)
k_depth_cost(const double* __restrict__ partial, int n_rec, int rec, const double* __restrict__ eta, int n_total,
             const int32_t* __restrict__ pairs, const double* __restrict__ delta, int n_pairs, DepthDev prm, double* __restrict__ out) {
  __shared__ double s[256];
  double v = 0.0;
  for (int q = threadIdx.x; q < n_rec; q += 256) v += partial[(size_t)q * rec + rec - 1];
  for (int q = threadIdx.x; q < n_pairs; q += 256) {
    const double d = eta[pairs[2 * q]] - eta[pairs[2 * q + 1]] + delta[q];
    v += 0.5 * prm.lambda_smooth * d * d;
  }
  for (int q = threadIdx.x; q < n_total; q += 256) v += 0.5 * prm.lambda_prior * eta[q] * eta[q];
  s[threadIdx.x] = v;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = s[0];
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
  // tiles of ~kDpTilePx pixels (the per-CTA setup is ~2000 shared-memory words), at least ~4 CTAs per SM in the grid
  const int E1 = std::max(c->E, 1);
  const int tiles0 = std::max(1, std::min(std::max((c->HW + kDpTilePx - 1) / kDpTilePx, (592 + E1 - 1) / E1), std::max(c->HW / kDpIterPx, 1)));
  const int per = ((c->HW + tiles0 - 1) / tiles0 + 63) / 64 * 64;     // pixels per tile: a multiple of a warp's 64-pixel chunk
  const int tiles = (c->HW + per - 1) / per;
  const int rec = 4 * n_seg + 1;
  const size_t smem = ((size_t)kDpWarps * 4 * n_seg + 2 * n_seg + kDpWarps) * sizeof(double) + (size_t)2 * n_seg * sizeof(float);
  if (smem > c->depth_smem) {
    cudaError_t ea = cudaFuncSetAttribute(k_depth_edge, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (ea != cudaSuccess) return ea;
    c->depth_smem = smem;
  }
  const float4* pm_init = c->pm0 ? c->pm0 : c->pm;               // pristine X_init (Eq. (8)): see sim3ba_apply_depth
  DepthDev dev{1.0 / (double)p.sigma_point, (double)p.huber_k, p.lambda_smooth, p.lambda_prior, p.lambda_lm, p.eta_max};
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
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; return e == cudaSuccess; };
  ok(up(&d_sp_ptr, sp_ptr, c->stream)); ok(up(&d_sp_other, sp_other, c->stream)); ok(up(&d_sp_delta, sp_delta, c->stream));
  ok(up(&d_pairs, pairs, c->stream)); ok(up(&d_delta, delta, c->stream)); ok(up(&d_anchor, anchor, c->stream));
  ok(dmalloc(reinterpret_cast<void**>(&d_partial), std::max<size_t>((size_t)c->E * tiles * rec, 1) * sizeof(double)));
  ok(dmalloc(reinterpret_cast<void**>(&d_eta2), std::max<size_t>(n_total, 1) * sizeof(double)));
  ok(dmalloc(reinterpret_cast<void**>(&d_cost), std::max(n_iters, 1) * sizeof(double)));
  double *cur = d_eta, *nxt = d_eta2;
  for (int it = 0; it < n_iters && e == cudaSuccess; ++it) {
    if (c->E > 0)
      k_depth_edge<<<c->E * tiles, kDpThreads, smem, c->stream>>>(pm_init, c->match, c->edges, c->grp_edge, d_labels, cur, c->poses, c->HW, n_seg, tiles,
                                                                 per, dev, d_partial);
    k_depth_cost<<<1, 256, 0, c->stream>>>(d_partial, c->E * tiles, rec, cur, n_total, d_pairs, d_delta, n_pairs, dev, d_cost + it);
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
  dfree(d_partial); dfree(d_eta2); dfree(d_cost);
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
