// Kernels 1+2 of the Sim(3) GN step: per-match residual / weights / Jacobian (a2-a4) and the
// deterministic per-edge block reduction (a5).
//
//   Eq. (1)  PAPER.md:73   e = [psi(x) - psi(X_i); |x| - |X_i|],  x = T_ij X_j
//   PAPER.md:76            r_c = sqrt(q) e_c / sigma_c, w_c = min(1, kappa/|r_c|), q = sqrt(c_i c_j)
//   Eq. (6)  PAPER.md:116  J_xi = [Dpsi/Dx; Dd/Dx] [I, -[x]x, x]  (closed form used here:
//                          J_xi = [[P, -[u]x, 0], [u^T, 0, d]], P = (I - u u^T)/d, u = x/d)
//   PAPER.md:118           J_j = J_xi Ad_{T_i^-1}, J_i = -J_j  ->  the adjoint is applied once per
//                          edge:  A_e = Ad^T (sum J_xi^T Omega J_xi) Ad,  b_e = Ad^T (sum J_xi^T Omega e)
//
// Precision plan: per-match arithmetic and per-thread partial sums (<= 16 terms) in
// fp32; everything from the per-thread partial upwards (warp, CTA, edge, adjoint congruence) in fp64.
// No floating-point atomics anywhere: the reduction order is fixed, results are run-to-run identical.
#include "sim3ba_internal.cuh"
#include "sim3_math.cuh"

namespace sim3ba {

namespace {

constexpr int kPxPerThread = kTilePx / kAccThreads;  // 16
constexpr int kBatch = 4;                            // loads in flight per thread
constexpr int kNumAcc = 36;                          // 28 M + 7 c + cost

__device__ __forceinline__ float4 ldg_f4(const float4* p) { return __ldg(p); }

#ifdef SIM3BA_EXACT_RSQRT   // debugging aid: IEEE-rounded 1/sqrt instead of the 2-ulp MUFU path
__device__ __forceinline__ float rsq(float v) { return __frcp_rn(__fsqrt_rn(v)); }
#else
__device__ __forceinline__ float rsq(float v) { return rsqrtf(v); }
#endif

// One valid match: accumulate J_xi^T Omega J_xi (upper triangle, 25 structurally non-zero
// entries), J_xi^T Omega e (7) and the robust cost into acc[].
__device__ __forceinline__ void accumulate_match(float (&acc)[kNumAcc], const float4 Xi, const float4 Xj,
                                                 const double* __restrict__ Td, const DevParams prm) {
  // delta = T_ij X_j - X_i in FP64 (Td = s_ij R_ij row-major [9], t_ij [3]).  This difference is the
  // one cancellation of the residual (|delta| ~ noise << |x|): evaluated in fp32 it would carry an
  // absolute error of ~ulp(|x|) per match, i.e. 1e-4..1e-3 of the residual itself.  Everything after
  // it works on small quantities, so fp32 is accurate to ~1e-7 RELATIVE to the residual.
  const double Xjx = (double)Xj.x, Xjy = (double)Xj.y, Xjz = (double)Xj.z;
  const float del0 = (float)fma(Td[0], Xjx, fma(Td[1], Xjy, fma(Td[2], Xjz, Td[9] - (double)Xi.x)));
  const float del1 = (float)fma(Td[3], Xjx, fma(Td[4], Xjy, fma(Td[5], Xjz, Td[10] - (double)Xi.y)));
  const float del2 = (float)fma(Td[6], Xjx, fma(Td[7], Xjy, fma(Td[8], Xjz, Td[11] - (double)Xi.z)));
  const float x0 = Xi.x + del0, x1 = Xi.y + del1, x2 = Xi.z + del2;   // x = T_ij X_j (fp32)
  const float d2 = fmaxf(fmaf(x0, x0, fmaf(x1, x1, x2 * x2)), 1e-20f);
  const float rd = rsq(d2);
  const float d = d2 * rd;
  const float u0 = x0 * rd, u1 = x1 * rd, u2 = x2 * rd;
  const float di2 = fmaxf(fmaf(Xi.x, Xi.x, fmaf(Xi.y, Xi.y, Xi.z * Xi.z)), 1e-20f);
  const float rdi = rsq(di2);
  const float di = di2 * rdi;
  // e3 = |x| - |X_i| = delta . (x + X_i) / (|x| + |X_i|);  e_r = x/|x| - X_i/|X_i| = delta/|x| - psi(X_i) e3/|x|
  const float e3 = __fdividef(fmaf(del0, x0 + Xi.x, fmaf(del1, x1 + Xi.y, del2 * (x2 + Xi.z))), d + di);
  const float e3rd = e3 * rd;
  const float e0 = fmaf(del0, rd, -(Xi.x * rdi) * e3rd);
  const float e1 = fmaf(del1, rd, -(Xi.y * rdi) * e3rd);
  const float e2 = fmaf(del2, rd, -(Xi.z * rdi) * e3rd);
  // q = sqrt(c_i c_j); s_c = q / sigma_c^2; r_c^2 = s_c e_c^2
  const float cc = Xi.w * Xj.w;
  const float q = cc * rsqrtf(fmaxf(cc, 1e-30f));
  const float sr = q * prm.inv_var_ray, sd = q * prm.inv_var_dist;
  float om[4], cost = 0.f;
  {
    const float ee[4] = {e0, e1, e2, e3};
    const float ss[4] = {sr, sr, sr, sd};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const float r2 = ss[c] * ee[c] * ee[c];
      const bool out = r2 > prm.huber_k2;
      const float rs = rsqrtf(out ? r2 : 1.f);
      om[c] = out ? ss[c] * (prm.huber_k * rs) : ss[c];                       // q w / sigma^2
      cost += out ? fmaf(prm.huber_k, r2 * rs, -0.5f * prm.huber_k2) : 0.5f * r2;
    }
  }
  const float a = om[0], b = om[1], c = om[2], w3 = om[3];
  // P = (I - u u^T) / d   (symmetric)
  const float P00 = (1.f - u0 * u0) * rd, P11 = (1.f - u1 * u1) * rd, P22 = (1.f - u2 * u2) * rd;
  const float P01 = -(u0 * u1) * rd, P02 = -(u0 * u2) * rd, P12 = -(u1 * u2) * rd;
  // B = diag(a,b,c) P  (rows scaled)
  const float B00 = a * P00, B01 = a * P01, B02 = a * P02;
  const float B10 = b * P01, B11 = b * P11, B12 = b * P12;
  const float B20 = c * P02, B21 = c * P12, B22 = c * P22;
  const float wu0 = w3 * u0, wu1 = w3 * u1, wu2 = w3 * u2;
  // M_vv = P B + w3 u u^T
  acc[0] += fmaf(P00, B00, fmaf(P01, B10, fmaf(P02, B20, wu0 * u0)));
  acc[1] += fmaf(P00, B01, fmaf(P01, B11, fmaf(P02, B21, wu0 * u1)));
  acc[2] += fmaf(P00, B02, fmaf(P01, B12, fmaf(P02, B22, wu0 * u2)));
  acc[7] += fmaf(P01, B01, fmaf(P11, B11, fmaf(P12, B21, wu1 * u1)));
  acc[8] += fmaf(P01, B02, fmaf(P11, B12, fmaf(P12, B22, wu1 * u2)));
  acc[13] += fmaf(P02, B02, fmaf(P12, B12, fmaf(P22, B22, wu2 * u2)));
  // M_vw(l, m) = sum_k B_kl S_km,  S = -[u]x = [[0,u2,-u1],[-u2,0,u0],[u1,-u0,0]]
  acc[3] += fmaf(B20, u1, -B10 * u2);
  acc[4] += fmaf(B00, u2, -B20 * u0);
  acc[5] += fmaf(B10, u0, -B00 * u1);
  acc[9] += fmaf(B21, u1, -B11 * u2);
  acc[10] += fmaf(B01, u2, -B21 * u0);
  acc[11] += fmaf(B11, u0, -B01 * u1);
  acc[14] += fmaf(B22, u1, -B12 * u2);
  acc[15] += fmaf(B02, u2, -B22 * u0);
  acc[16] += fmaf(B12, u0, -B02 * u1);
  // M_v zeta = w3 d u,  M_zeta zeta = w3 d^2
  const float w3d = w3 * d;
  acc[6] += w3d * u0;
  acc[12] += w3d * u1;
  acc[17] += w3d * u2;
  acc[27] += w3d * d;
  // M_ww = S^T diag(a,b,c) S
  acc[18] += fmaf(b * u2, u2, c * u1 * u1);
  acc[22] += fmaf(a * u2, u2, c * u0 * u0);
  acc[25] += fmaf(a * u1, u1, b * u0 * u0);
  acc[19] -= c * u0 * u1;
  acc[20] -= b * u0 * u2;
  acc[23] -= a * u1 * u2;
  // c_v = B^T e_r + w3 e3 u ; c_w = S^T (Omega e_r) ; c_zeta = w3 d e3
  const float we3 = w3 * e3;
  acc[28] += fmaf(B00, e0, fmaf(B10, e1, fmaf(B20, e2, we3 * u0)));
  acc[29] += fmaf(B01, e0, fmaf(B11, e1, fmaf(B21, e2, we3 * u1)));
  acc[30] += fmaf(B02, e0, fmaf(B12, e1, fmaf(B22, e2, we3 * u2)));
  const float f0 = a * e0, f1 = b * e1, f2 = c * e2;
  acc[31] += fmaf(f2, u1, -f1 * u2);
  acc[32] += fmaf(f0, u2, -f2 * u0);
  acc[33] += fmaf(f1, u0, -f0 * u1);
  acc[34] += we3 * d;
  acc[35] += cost;
}

__global__ void __launch_bounds__(kAccThreads)
k_accumulate(const float4* __restrict__ pm, const int32_t* __restrict__ match, const int32_t* __restrict__ edges,
             const int32_t* __restrict__ sched, const double* __restrict__ poses, double* __restrict__ partials,
             int HW, int chunks, DevParams prm) {
  __shared__ double s_T[12];  // s_ij R_ij [9], t_ij [3]
  __shared__ double s_red[kAccThreads / 32][kNumAcc];
  __shared__ unsigned long long s_chk[kAccThreads / 32];
  __shared__ int s_cnt[kAccThreads / 32];

  const int e = sched[blockIdx.x / chunks];
  const int chunk = blockIdx.x % chunks;
  const int i = edges[2 * e], j = edges[2 * e + 1];
  if (threadIdx.x == 0) {
    const Sim3d Tij = relative_pose(load_pose(poses + 8 * i), load_pose(poses + 8 * j));
#pragma unroll
    for (int k = 0; k < 9; ++k) s_T[k] = Tij.s * Tij.R[k];
#pragma unroll
    for (int k = 0; k < 3; ++k) s_T[9 + k] = Tij.t[k];
  }
  __syncthreads();
  double Td[12];
#pragma unroll
  for (int k = 0; k < 12; ++k) Td[k] = s_T[k];

  const float4* __restrict__ Pi = pm + (size_t)i * HW;
  const float4* __restrict__ Pj = pm + (size_t)j * HW;
  const int32_t* __restrict__ mt = match + (size_t)e * HW;

  float acc[kNumAcc];
#pragma unroll
  for (int k = 0; k < kNumAcc; ++k) acc[k] = 0.f;
  int cnt = 0;
  unsigned long long chk = 0ull;

  const int base = chunk * kTilePx + threadIdx.x;
#pragma unroll 1
  for (int k0 = 0; k0 < kPxPerThread; k0 += kBatch) {
    int n[kBatch];
    float4 Xi[kBatch], Xj[kBatch];
    bool ok[kBatch];
#pragma unroll
    for (int b = 0; b < kBatch; ++b) {
      const int m = base + (k0 + b) * kAccThreads;
      n[b] = (m < HW) ? __ldg(mt + m) : -1;
    }
#pragma unroll
    for (int b = 0; b < kBatch; ++b) {
      const int m = base + (k0 + b) * kAccThreads;
      ok[b] = (n[b] >= 0) && (n[b] < HW);
      if (ok[b]) {
        Xi[b] = ldg_f4(Pi + m);
        Xj[b] = ldg_f4(Pj + n[b]);
      }
    }
#pragma unroll
    for (int b = 0; b < kBatch; ++b) {
      const int m = base + (k0 + b) * kAccThreads;
      if (ok[b] && Xi[b].w > prm.conf_min && Xj[b].w > prm.conf_min) {
        accumulate_match(acc, Xi[b], Xj[b], Td, prm);
        ++cnt;
        chk += (unsigned long long)m * (unsigned long long)HW + (unsigned long long)n[b];
      }
    }
  }

  // thread partial (<= 16 fp32 terms) -> fp64; warp shuffle tree; fixed-order cross-warp sum
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < kNumAcc; ++k) {
    double v = (double)acc[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) s_red[warp][k] = v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    chk += __shfl_xor_sync(0xffffffffu, chk, o);
  }
  if (lane == 0) { s_cnt[warp] = cnt; s_chk[warp] = chk; }
  __syncthreads();
  double* out = partials + ((size_t)e * chunks + chunk) * kPartialStride;
  if (threadIdx.x < kNumAcc) {
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < kAccThreads / 32; ++w) v += s_red[w][threadIdx.x];
    out[threadIdx.x] = v;
  } else if (threadIdx.x == 64) {
    long long c = 0;
    unsigned long long h = 0ull;
#pragma unroll
    for (int w = 0; w < kAccThreads / 32; ++w) { c += s_cnt[w]; h += s_chk[w]; }
    reinterpret_cast<long long*>(out)[36] = c;
    reinterpret_cast<unsigned long long*>(out)[37] = h;
  }
}

// Kernel 2: per edge, sum the chunk partials in chunk order (fp64), then the adjoint congruence
// A_e = Ad^T M Ad, b_e = Ad^T c with Ad = Ad_{T_i^-1}.
__global__ void __launch_bounds__(64)
k_finalize(const double* __restrict__ partials, const int32_t* __restrict__ edges, const double* __restrict__ poses,
           double* __restrict__ blocks35, double* __restrict__ edge_cost, int32_t* __restrict__ n_valid,
           unsigned long long* __restrict__ checksum, int chunks) {
  __shared__ double s_sum[kNumAcc];
  __shared__ double s_M[49], s_Ad[49], s_T[49];
  const int e = blockIdx.x, t = threadIdx.x;
  const double* p = partials + (size_t)e * chunks * kPartialStride;
  if (t < kNumAcc) {
    double v = 0.0;
    for (int c = 0; c < chunks; ++c) v += p[(size_t)c * kPartialStride + t];
    s_sum[t] = v;
  } else if (t == 36) {
    long long v = 0;
    for (int c = 0; c < chunks; ++c) v += reinterpret_cast<const long long*>(p + (size_t)c * kPartialStride)[36];
    n_valid[e] = (int32_t)v;
  } else if (t == 37) {
    unsigned long long v = 0ull;
    for (int c = 0; c < chunks; ++c) v += reinterpret_cast<const unsigned long long*>(p + (size_t)c * kPartialStride)[37];
    checksum[e] = v;
  } else if (t == 38) {
    adjoint_of_inverse(load_pose(poses + 8 * edges[2 * e]), s_Ad);
  }
  __syncthreads();
  if (t < 49) {
    const int r = t / 7, c = t % 7;
    const int lo = r < c ? r : c, hi = r < c ? c : r;
    s_M[t] = s_sum[lo * 7 - lo * (lo - 1) / 2 + (hi - lo)];
  }
  __syncthreads();
  if (t < 49) {  // T = M Ad
    const int r = t / 7, c = t % 7;
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < 7; ++k) v += s_M[7 * r + k] * s_Ad[7 * k + c];
    s_T[t] = v;
  }
  __syncthreads();
  if (t < 49) {  // A = Ad^T T
    const int r = t / 7, c = t % 7;
    if (r <= c) {
      double v = 0.0;
#pragma unroll
      for (int k = 0; k < 7; ++k) v += s_Ad[7 * k + r] * s_T[7 * k + c];
      blocks35[(size_t)e * 35 + r * 7 - r * (r - 1) / 2 + (c - r)] = v;
    }
  } else if (t < 56) {  // b = Ad^T c
    const int r = t - 49;
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < 7; ++k) v += s_Ad[7 * k + r] * s_sum[28 + k];
    blocks35[(size_t)e * 35 + 28 + r] = v;
  } else if (t == 56) {
    edge_cost[e] = s_sum[35];
  }
}

// packs [N][HW][3] points + [N][HW] confidences into float4 (x, y, z, c)
__global__ void k_pack(const float* __restrict__ pts, const float* __restrict__ conf, float4* __restrict__ pm, size_t total) {
  size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; idx < total; idx += stride)
    pm[idx] = make_float4(pts[3 * idx], pts[3 * idx + 1], pts[3 * idx + 2], conf[idx]);
}

}  // namespace

cudaError_t launch_pack(Ctx* c, const float* d_points, const float* d_conf) {
  const size_t total = (size_t)c->N * c->HW;
  const int grid = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
  k_pack<<<grid, 256, 0, c->stream>>>(d_points, d_conf, c->pm, total);
  ++c->launches;
  return cudaGetLastError();
}

cudaError_t launch_accumulate(Ctx* c) {
  if (c->E == 0) return cudaSuccess;
  DevParams p;
  p.inv_var_ray = 1.0f / (c->prm.sigma_ray * c->prm.sigma_ray);
  p.inv_var_dist = 1.0f / (c->prm.sigma_dist * c->prm.sigma_dist);
  p.huber_k = c->prm.huber_k;
  p.huber_k2 = c->prm.huber_k * c->prm.huber_k;
  p.conf_min = c->prm.conf_min;
  k_accumulate<<<c->E * c->chunks, kAccThreads, 0, c->stream>>>(c->pm, c->match, c->edges, c->sched, c->poses,
                                                                 c->partials, c->HW, c->chunks, p);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  if (c->profiling) cudaEventRecord(c->ev[1], c->stream);
  k_finalize<<<c->E, 64, 0, c->stream>>>(c->partials, c->edges, c->poses, c->blocks35, c->edge_cost, c->n_valid,
                                         c->checksum, c->chunks);
  c->launches += 2;
  return cudaGetLastError();
}

}  // namespace sim3ba
