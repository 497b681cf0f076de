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
// the tiles of an edge together: X_j and the labels are shared through L2).  Per match everything is FP64 (the residual
// is a difference of two ~10 m points); the loads run in a software pipeline (streams two iterations ahead, gathers
// one).  The per-segment sums are binned without atomics: a lane whose label is alone in its warp adds straight to the
// warp's own shared-memory bin, a label shared by several lanes takes one butterfly carrying both sums; the eight warps'
// bins are added in a fixed order -> one record [2 sides][n_seg][g, H] + cost per (edge, tile).
// Kernel B (k_depth_update): one thread per segment gathers its records through the keyframe -> edge CSR, adds boundary
// and prior terms, takes the damped clipped step into a second eta buffer.  Kernel C sums the objective.
#include <math.h>

#include <vector>

#include "sim3ba_internal.cuh"
#include "sim3_math.cuh"

namespace sim3ba {

namespace {

constexpr int kDpThreads = 256;
constexpr int kDpWarps = kDpThreads / 32;
constexpr int kDpMaxSeg = 64;
#ifndef SIM3BA_DP_CTAS
#define SIM3BA_DP_CTAS 2
#endif
#ifndef SIM3BA_DP_TILE_PX
#define SIM3BA_DP_TILE_PX 16384
#endif
constexpr int kDpTilePx = SIM3BA_DP_TILE_PX;

struct DepthDev {
  double inv_sigma, huber_k, lambda_smooth, lambda_prior, lambda_lm, eta_max;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// 1 / x for a normal positive x: the hardware seed and two Newton steps (relative error ~1e-16; the division routine
// costs about twice the instructions and a branch)
__device__ __forceinline__ double rcp_newton(double x) {
#ifdef SIM3BA_DP_EXACT_DIV
  return 1.0 / x;
#else
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
#endif
}

// add (a, b) of the lanes with `valid` into bins[label][0..1] (deterministic).  A lane whose label no other valid lane
// of the warp carries (an outlier match landing in some far segment) adds straight to the bin -- distinct labels, so these
// adds do not meet; the labels shared by several lanes go label by label: butterfly sum of the lanes carrying it,
// lanes 0 and 1 add.  The usual warp (one segment, a few stray matches) takes one butterfly round instead of one per stray lane.
__device__ __forceinline__ void bin_by_label(double* bins, bool valid, int label, double a, double b, int lane) {
  const unsigned peers = __match_any_sync(0xffffffffu, valid ? label : -1 - lane);   // invalid lanes: unique keys
  const bool single = valid && peers == (1u << lane);
  if (single) { bins[2 * label] += a; bins[2 * label + 1] += b; }
  unsigned active = __ballot_sync(0xffffffffu, valid && !single);
  while (active) {
    const int leader = __ffs(active) - 1;
    const int L = __shfl_sync(0xffffffffu, label, leader);
    const bool mine = valid && label == L;
    // both sums in one butterfly: after the first exchange even lanes carry pair sums of a, odd lanes of b
    const double va = mine ? a : 0.0, vb = mine ? b : 0.0;
    double x = (lane & 1) ? vb : va;
    x += __shfl_xor_sync(0xffffffffu, (lane & 1) ? va : vb, 1);
#pragma unroll
    for (int o = 2; o < 32; o <<= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if (lane < 2) bins[2 * L + lane] += x;                     // lane 0: sum of a, lane 1: sum of b
    active &= ~__ballot_sync(0xffffffffu, mine);
  }
  __syncwarp();                                                // the next call's adds may come from other lanes
}

__global__ void __launch_bounds__(kDpThreads, SIM3BA_DP_CTAS)
k_depth_edge(const float4* __restrict__ pm, const int32_t* __restrict__ match, const int32_t* __restrict__ edges,
             const int32_t* __restrict__ grp_edge, const int32_t* __restrict__ labels, const double* __restrict__ eta,
             const double* __restrict__ poses, int HW, int n_seg, int tiles, DepthDev prm, double* __restrict__ partial) {
  __shared__ double s_bins[kDpWarps][2][kDpMaxSeg][2];
  __shared__ double s_exp[2][kDpMaxSeg];
  __shared__ double s_cost[kDpWarps];
  // launch order = kernel 1's: the edges sorted by (i, j), all tiles of an edge together, so the CTAs in flight cover a
  // few neighbouring keyframes completely and X_i, X_j and the labels are fetched from HBM once and shared through L2
  const int k = blockIdx.x / tiles, tile = blockIdx.x - k * tiles, e = grp_edge[k];
  const int i = edges[2 * e], j = edges[2 * e + 1];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int q = tid; q < kDpWarps * 2 * kDpMaxSeg * 2; q += kDpThreads) (&s_bins[0][0][0][0])[q] = 0.0;
  if (tid < n_seg) { s_exp[0][tid] = exp(eta[(size_t)i * n_seg + tid]); s_exp[1][tid] = exp(eta[(size_t)j * n_seg + tid]); }
  __syncthreads();
  const Sim3d T = relative_pose(load_pose(poses + 8 * i), load_pose(poses + 8 * j));   // T_ij
  const float4* __restrict__ Pi = pm + (size_t)i * HW;
  const float4* __restrict__ Pj = pm + (size_t)j * HW;
  const int32_t* __restrict__ mt = match + (size_t)e * HW;
  const int32_t* __restrict__ li = labels + (size_t)i * HW;
  const int32_t* __restrict__ lj = labels + (size_t)j * HW;
  const int per = (HW + tiles - 1) / tiles;
  const int m0 = tile * per, m1 = min(HW, m0 + per);
  double cost = 0.0;
  // Software pipeline over the CTA's iterations (warp-uniform trip count: the binning uses full-warp shuffles): the
  // streamed loads (match index, X_i, label of m) run two iterations ahead, the gathers they address (X_j, label of n) one.
  const int niter = (m1 - m0 + kDpThreads - 1) / kDpThreads;
  auto load_stream = [&](int it, int& n, float4& a, int& lg) {
    const int m = m0 + it * kDpThreads + tid;
    n = -1;
    if (it < niter && m < m1) { n = __ldcs(mt + m); a = Pi[m]; lg = li[m]; }
  };
  auto load_gather = [&](int n, float4& b, int& lh) {
    if ((unsigned)n < (unsigned)HW) { b = Pj[n]; lh = lj[n]; }
  };
  int n0, n1, n2, lg0 = 0, lg1 = 0, lg2 = 0, lh0 = 0, lh1 = 0;
  float4 a0 = make_float4(0.f, 0.f, 0.f, -1.f), a1 = a0, a2 = a0, b0 = a0, b1 = a0;
  load_stream(0, n0, a0, lg0);
  load_stream(1, n1, a1, lg1);
  load_gather(n0, b0, lh0);
  for (int it = 0; it < niter; ++it) {
    load_stream(it + 2, n2, a2, lg2);
    load_gather(n1, b1, lh1);
    bool valid = false;
    const int lg = lg0, lh = lh0;
    double vg = 0.0, Hg = 0.0, vh = 0.0, Hh = 0.0;
    if ((unsigned)n0 < (unsigned)HW) {
      const float4 a = a0, b = b0;
      if (a.w >= 0.f && b.w >= 0.f && lg >= 0 && lh >= 0 && lg < n_seg && lh < n_seg) {
        valid = true;
        const double eg = s_exp[0][lg], eh = s_exp[1][lh];
        const double Xi[3] = {eg * (double)a.x, eg * (double)a.y, eg * (double)a.z};
        const double Xj[3] = {eh * (double)b.x, eh * (double)b.y, eh * (double)b.z};
        const double sq = (double)a.w * (double)b.w, q = sq * sq;     // w = c^(1/4): sqrt(q) = w_i w_j, q = sqrt(c_i c_j)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const double Jh = T.s * (T.R[3 * c] * Xj[0] + T.R[3 * c + 1] * Xj[1] + T.R[3 * c + 2] * Xj[2]);
          const double res = Jh + T.t[c] - Xi[c];
          const double r = sq * res * prm.inv_sigma, ar = fabs(r);
          const double w = ar <= prm.huber_k ? 1.0 : prm.huber_k * rcp_newton(ar);
          const double om = q * w * prm.inv_sigma * prm.inv_sigma;
          cost += ar <= prm.huber_k ? 0.5 * r * r : prm.huber_k * (ar - 0.5 * prm.huber_k);
          vg -= om * Xi[c] * res;                                        // J_g = -X_i(eta)
          Hg += om * Xi[c] * Xi[c];
          vh += om * Jh * res;                                           // J_h = s_ij R_ij X_j(eta)
          Hh += om * Jh * Jh;
        }
      }
    }
    n0 = n1; a0 = a1; lg0 = lg1; b0 = b1; lh0 = lh1;
    n1 = n2; a1 = a2; lg1 = lg2;
    bin_by_label(&s_bins[warp][0][0][0], valid, lg, vg, Hg, lane);
    bin_by_label(&s_bins[warp][1][0][0], valid, lh, vh, Hh, lane);
  }
  cost = warp_sum(cost);
  if (lane == 0) s_cost[warp] = cost;
  __syncthreads();
  double* out = partial + ((size_t)e * tiles + tile) * (4 * n_seg + 1);
  for (int q = tid; q < 4 * n_seg; q += kDpThreads) {          // q = (side, label, {g, H})
    const int side = q / (2 * n_seg), rest = q - side * 2 * n_seg;
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < kDpWarps; ++w) v += (&s_bins[w][side][0][0])[rest];
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
  const int tiles = std::max(1, std::min(std::max((c->HW + kDpTilePx - 1) / kDpTilePx, (592 + E1 - 1) / E1), std::max(c->HW / 256, 1)));
  const int rec = 4 * n_seg + 1;
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
      k_depth_edge<<<c->E * tiles, kDpThreads, 0, c->stream>>>(c->pm, c->match, c->edges, c->grp_edge, d_labels, cur, c->poses, c->HW, n_seg, tiles, dev,
                                                              d_partial);
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
  const int grid = (int)std::min<size_t>((total + 255) / 256, 148 * 16);
  k_depth_apply<<<grid, 256, 0, c->stream>>>(d_points, d_conf, d_labels, d_eta, c->pm, c->HW, n_seg, total, c->prm.conf_min);
  ++c->launches;
  return cudaGetLastError();
}

int depth_max_segments() { return kDpMaxSeg; }

}  // namespace sim3ba
