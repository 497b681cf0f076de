// Kernels 1+2 of the Sim(3) GN step: per-match residual / weights / Jacobian (a2-a4) and the
// deterministic per-edge block reduction (a5).
//
//   Eq. (1)  PAPER.md:73   e = [psi(x) - psi(X_i); |x| - |X_i|],  x = T_ij X_j
//   PAPER.md:76            r_c = sqrt(q) e_c / sigma_c, w_c = min(1, kappa/|r_c|), q = sqrt(c_i c_j)
//   Eq. (6)  PAPER.md:116  J_xi = [Dpsi/Dx; Dd/Dx] [I, -[x]x, x]  (closed form used here, with
//                          S = -[u]x, u = x/d:  J_xi = [[S S^T / d, S, 0], [u^T, 0, d]])
//   PAPER.md:118           J_j = J_xi Ad_{T_i^-1}, J_i = -J_j  ->  the adjoint is applied once per
//                          edge:  A_e = Ad^T (sum J_xi^T Omega J_xi) Ad,  b_e = Ad^T (sum J_xi^T Omega e)
//
// Work decomposition: one CTA per (keyframe i, tile of 3072 pixels of i), 192 threads,
// two CTAs per SM.  The tile of X_i is staged in shared memory ONCE by a TMA bulk copy (cp.async.bulk +
// mbarrier) and reused by every edge (i, j) that leaves i; per edge the match indices are streamed
// (coalesced, evict-first) and X_j is gathered (128-bit loads), software-pipelined one pair ahead.
// Every thread evaluates TWO matches at a time in the two lanes of packed fp32x2 instructions
// (FFMA2 / FMUL2 / FADD2: one issue slot per two lanes), accumulators included.
//
// Precision plan: delta = T_ij X_j - X_i in FP64 (the one cancellation of the residual); everything
// after it and the per-thread partial sums (<= 8 terms per lane, 16 per thread) in fp32; every sum from
// the per-thread partial upwards (warp, CTA, edge, adjoint congruence) in FP64.  No floating-point
// atomics: the reduction order is fixed, results are run-to-run identical.
#include "sim3ba_internal.cuh"
#include "sim3_math.cuh"

namespace sim3ba {

namespace {

static_assert(kTilePx == 16 * kAccThreads, "precision plan: <= 16 fp32 terms per thread partial (8 per lane)");
constexpr int kPairs = kTilePx / (2 * kAccThreads);   // match pairs per thread and edge
constexpr int kWarps = kAccThreads / 32;
constexpr int kSlots = kPartialStride;         // 40 reduction slots (layout: sim3ba_internal.cuh)
constexpr int kAccSlots = 37;                  // slots that carry floating-point sums

// shared-memory carve-up of k_accumulate (dynamic)
constexpr size_t kOffXi = 0;                                      // float4 [kTilePx], re-laid as lane pairs
constexpr size_t kOffDer = kOffXi + sizeof(float4) * kTilePx;     // float4 [kTilePx / 2] (1/|X_A|, 1/|X_B|, |X_A|, |X_B|)
constexpr size_t kOffRed = kOffDer + sizeof(float4) * (kTilePx / 2);   // double [kWarps][kSlots]
constexpr size_t kOffT = kOffRed + sizeof(double) * kWarps * kSlots;   // double [12]
constexpr size_t kOffCnt = kOffT + sizeof(double) * 12;           // unsigned [kWarps] (8 B stride)
constexpr size_t kOffChk = kOffCnt + sizeof(long long) * kWarps;  // unsigned long long [kWarps]
constexpr size_t kOffBar = kOffChk + sizeof(long long) * kWarps;  // mbarrier
constexpr size_t kAccSmem = kOffBar + 16;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// TMA 1-D bulk copy global -> shared, completion signalled on the mbarrier (bytes % 16 == 0)
__device__ __forceinline__ void tma_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// MUFU.RSQ / MUFU.RCP without the denormal pre/post-scaling of rsqrtf() / 1/x: arguments are clamped or
// may legitimately give +inf (handled by the min() that follows)
__device__ __forceinline__ float rsq(float v) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}
__device__ __forceinline__ float rcp(float v) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}

// ---- packed fp32x2 arithmetic (sm_100: FFMA2 / FMUL2 / FADD2, one issue slot for two lanes) -------
// The two lanes of every float2 below are TWO DIFFERENT MATCHES (A, B) of the same thread: the whole
// per-match algebra is evaluated 2-wide, accumulators included; lanes are summed once per (edge, tile).
using f2 = float2;
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 operator-(f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 bc(float s) { return make_float2(s, s); }

// Two valid-or-masked matches: accumulate J_xi^T Omega J_xi (25 structurally non-zero upper-triangular
// entries), J_xi^T Omega e (7) and the two robust-cost sums into acc[] (slot layout: sim3ba_internal.cuh).
//   del = T_ij X_j - X_i (fp32 rounding of the FP64 value), Xi, rdi = 1/|X_i|, di = |X_i|,
//   sq = sqrt(q) = (c_i c_j)^(1/4), 0 for a masked lane (all its weights vanish).
__device__ __forceinline__ void accumulate_pair(f2 (&acc)[kAccSlots], const f2 del0, const f2 del1, const f2 del2,
                                                const f2 Xi0, const f2 Xi1, const f2 Xi2, const f2 rdi, const f2 di,
                                                const f2 sq, const DevParams& prm) {
  const f2 x0 = Xi0 + del0, x1 = Xi1 + del1, x2 = Xi2 + del2;   // x = T_ij X_j
  f2 d2 = fma2(x0, x0, fma2(x1, x1, x2 * x2));
  d2.x = fmaxf(d2.x, 1e-20f); d2.y = fmaxf(d2.y, 1e-20f);
  const f2 rd = make_float2(rsq(d2.x), rsq(d2.y));
  const f2 d = d2 * rd;
  const f2 u0 = x0 * rd, u1 = x1 * rd, u2 = x2 * rd;
  // e3 = |x| - |X_i| = delta . (x + X_i) / (|x| + |X_i|);  e_r = x/|x| - X_i/|X_i| = delta/|x| - X_i e3 / (|x| |X_i|)
  const f2 den = d + di;
  const f2 e3 = fma2(del0, x0 + Xi0, fma2(del1, x1 + Xi1, del2 * (x2 + Xi2))) * make_float2(rcp(den.x), rcp(den.y));
  const f2 gsc = (e3 * rd) * rdi;
  const f2 e0 = fma2(del0, rd, -(Xi0 * gsc));
  const f2 e1 = fma2(del1, rd, -(Xi1 * gsc));
  const f2 e2 = fma2(del2, rd, -(Xi2 * gsc));
  // q = sqrt(c_i c_j); s_c = q / sigma_c^2; omega_c = q w_c / sigma_c^2 = min(s_c, kappa sqrt(q) / (sigma_c |e_c|));
  // rho_c = omega_c e_c^2 - min(s_c e_c^2, kappa^2) / 2
  const f2 q = sq * sq;
  const f2 sr = q * bc(prm.inv_var_ray), sd = q * bc(prm.inv_var_dist);
  const f2 kr = sq * bc(prm.k_over_sigma_ray), kd = sq * bc(prm.k_over_sigma_dist);
  f2 om[4], f[4];
  {
    const f2 ee[4] = {e0, e1, e2, e3};
    const f2 ss[4] = {sr, sr, sr, sd};
    const f2 kk[4] = {kr, kr, kr, kd};
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const f2 t = kk[c] * make_float2(rcp(fabsf(ee[c].x)), rcp(fabsf(ee[c].y)));
      om[c] = make_float2(fminf(ss[c].x, t.x), fminf(ss[c].y, t.y));   // fminf(s, NaN) = s (masked lane, e = 0)
      f[c] = om[c] * ee[c];
      acc[35] = fma2(f[c], ee[c], acc[35]);                            // sum w r^2
      const f2 r2 = (ss[c] * ee[c]) * ee[c];
      acc[36] = acc[36] + make_float2(fminf(r2.x, prm.huber_k2), fminf(r2.y, prm.huber_k2));   // sum min(r^2, k^2)
    }
  }
  const f2 a = om[0], b = om[1], c = om[2], w3 = om[3];
  const f2 u00 = u0 * u0, u11 = u1 * u1, u22 = u2 * u2, u01 = u0 * u1, u02 = u0 * u2, u12 = u1 * u2;
  // K = S^T diag(a,b,c) S = M_ww,  S = -[u]x
  const f2 K00 = fma2(b, u22, c * u11), K11 = fma2(a, u22, c * u00), K22 = fma2(a, u11, b * u00);
  const f2 K01 = -(c * u01), K02 = -(b * u02), K12 = -(a * u12);
  acc[18] = acc[18] + K00; acc[19] = acc[19] + K01; acc[20] = acc[20] + K02;
  acc[22] = acc[22] + K11; acc[23] = acc[23] + K12; acc[25] = acc[25] + K22;
  // G = (S/d) K = M_vw,  S/d = [[0, v2, -v1], [-v2, 0, v0], [v1, -v0, 0]]
  const f2 v0 = u0 * rd, v1 = u1 * rd, v2 = u2 * rd;
  const f2 G00 = fma2(v2, K01, -(v1 * K02)), G01 = fma2(v2, K11, -(v1 * K12)), G02 = fma2(v2, K12, -(v1 * K22));
  const f2 G10 = fma2(v0, K02, -(v2 * K00)), G11 = fma2(v0, K12, -(v2 * K01)), G12 = fma2(v0, K22, -(v2 * K02));
  const f2 G20 = fma2(v1, K00, -(v0 * K01)), G21 = fma2(v1, K01, -(v0 * K11)), G22 = fma2(v1, K02, -(v0 * K12));
  acc[3] = acc[3] + G00; acc[4] = acc[4] + G01; acc[5] = acc[5] + G02;
  acc[9] = acc[9] + G10; acc[10] = acc[10] + G11; acc[11] = acc[11] + G12;
  acc[14] = acc[14] + G20; acc[15] = acc[15] + G21; acc[16] = acc[16] + G22;
  // M_vv = G (S/d)^T + w3 u u^T
  acc[0] = fma2(G01, v2, fma2(-G02, v1, fma2(w3, u00, acc[0])));
  acc[1] = fma2(G02, v0, fma2(-G00, v2, fma2(w3, u01, acc[1])));
  acc[2] = fma2(G00, v1, fma2(-G01, v0, fma2(w3, u02, acc[2])));
  acc[7] = fma2(G12, v0, fma2(-G10, v2, fma2(w3, u11, acc[7])));
  acc[8] = fma2(G10, v1, fma2(-G11, v0, fma2(w3, u12, acc[8])));
  acc[13] = fma2(G20, v1, fma2(-G21, v0, fma2(w3, u22, acc[13])));
  // M_v zeta = w3 d u,  M_zeta zeta = w3 d^2
  const f2 w3d = w3 * d;
  acc[6] = fma2(w3d, u0, acc[6]);
  acc[12] = fma2(w3d, u1, acc[12]);
  acc[17] = fma2(w3d, u2, acc[17]);
  acc[27] = fma2(w3d, d, acc[27]);
  // c_v = (f - u (u.f)) / d + f3 u ;  c_w = S^T f = u x f ;  c_zeta = f3 d
  const f2 uf = fma2(u0, f[0], fma2(u1, f[1], u2 * f[2]));
  acc[28] = fma2(rd, fma2(-u0, uf, f[0]), fma2(f[3], u0, acc[28]));
  acc[29] = fma2(rd, fma2(-u1, uf, f[1]), fma2(f[3], u1, acc[29]));
  acc[30] = fma2(rd, fma2(-u2, uf, f[2]), fma2(f[3], u2, acc[30]));
  acc[31] = fma2(u1, f[2], fma2(-u2, f[1], acc[31]));
  acc[32] = fma2(u2, f[0], fma2(-u0, f[2], acc[32]));
  acc[33] = fma2(u0, f[1], fma2(-u1, f[0], acc[33]));
  acc[34] = fma2(f[3], d, acc[34]);
}

// Warp reduction of the 40 fp32 thread partials into FP64 warp sums by recursive halving: at every
// level a lane keeps one half of its slots and hands the other half to its partner, so the whole tree
// costs 20 + 10 + 5 + 5 + 5 exchanges instead of 40 x 5.  Level 1 exchanges the fp32 partials and
// converts both operands (the sums are FP64 from here on).  Lanes with (lane & 3) == 0 end up holding
// the warp totals of slots base .. base + 4, base = 20 b4 + 10 b3 + 5 b2 (bits of the lane index).
__device__ __forceinline__ void warp_reduce_slots(const float (&acc)[kSlots], double* __restrict__ s_red_warp, const int lane) {
  double v[20];
  {
    const bool up = lane & 16;
#pragma unroll
    for (int k = 0; k < 20; ++k) {
      const float keep = up ? acc[20 + k] : acc[k];
      const float send = up ? acc[k] : acc[20 + k];
      v[k] = (double)keep + (double)__shfl_xor_sync(0xffffffffu, send, 16);
    }
  }
  {
    const bool up = lane & 8;
#pragma unroll
    for (int k = 0; k < 10; ++k) {
      const double keep = up ? v[10 + k] : v[k];
      const double send = up ? v[k] : v[10 + k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
  }
  {
    const bool up = lane & 4;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const double keep = up ? v[5 + k] : v[k];
      const double send = up ? v[k] : v[5 + k];
      v[k] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    v[k] += __shfl_xor_sync(0xffffffffu, v[k], 2);
    v[k] += __shfl_xor_sync(0xffffffffu, v[k], 1);
  }
  if ((lane & 3) == 0) {
    const int base = ((lane >> 4) & 1) * 20 + ((lane >> 3) & 1) * 10 + ((lane >> 2) & 1) * 5;
#pragma unroll
    for (int k = 0; k < 5; ++k) s_red_warp[base + k] = v[k];
  }
}

__global__ void __launch_bounds__(kAccThreads, 2)
k_accumulate(const float4* __restrict__ pm, const int32_t* __restrict__ match, const int32_t* __restrict__ edges,
             const int32_t* __restrict__ grp_kf, const int32_t* __restrict__ grp_ptr, const int32_t* __restrict__ grp_edge,
             const double* __restrict__ edgeT, double* __restrict__ partials, int HW, int tiles, DevParams prm) {
  extern __shared__ __align__(128) unsigned char smem[];
  float4* s_Xi = reinterpret_cast<float4*>(smem + kOffXi);
  float4* s_der = reinterpret_cast<float4*>(smem + kOffDer);
  double* s_red = reinterpret_cast<double*>(smem + kOffRed);
  double* s_T = reinterpret_cast<double*>(smem + kOffT);
  unsigned int* s_cnt = reinterpret_cast<unsigned int*>(smem + kOffCnt);
  unsigned long long* s_chk = reinterpret_cast<unsigned long long*>(smem + kOffChk);
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(smem + kOffBar);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = blockIdx.x / tiles, tile = blockIdx.x - g * tiles;
  const int i = grp_kf[g];
  const int px0 = tile * kTilePx;
  const int npx = min(kTilePx, HW - px0);

  // ---- stage the tile of X_i: one TMA bulk copy per 16 KB, completion on the mbarrier ----
  if (tid == 0) mbar_init(s_bar, 1);
  __syncthreads();
  if (tid == 0) {
    const uint32_t bytes = (uint32_t)npx * (uint32_t)sizeof(float4);
    mbar_expect_tx(s_bar, bytes);
    const unsigned char* src = reinterpret_cast<const unsigned char*>(pm + (size_t)i * HW + px0);
    for (uint32_t off = 0; off < bytes; off += 16384u)
      tma_bulk_g2s(smem + kOffXi + off, src + off, min(16384u, bytes - off), s_bar);
  }
  mbar_wait(s_bar, 0);
  // Pair p of this thread = pixels A = 2p T + tid and B = (2p + 1) T + tid (T = kAccThreads).  Re-lay the two
  // staged float4 in place as lane pairs, (xA, xB, yA, yB) in A's slot and (zA, zB, wA, wB) in B's, and keep
  // (1/|X_A|, 1/|X_B|, |X_A|, |X_B|): everything the edges leaving i share.  Pixels past the ragged end of the
  // keyframe were not staged: they become masked lanes (w = -1).
#pragma unroll 2
  for (int p = 0; p < kPairs; ++p) {
    const int pa = 2 * p * kAccThreads + tid, pb = pa + kAccThreads;
    float4 A = make_float4(0.f, 0.f, 0.f, -1.f), B = A;
    if (pa < npx) A = s_Xi[pa];
    if (pb < npx) B = s_Xi[pb];
    const float da2 = fmaxf(fmaf(A.x, A.x, fmaf(A.y, A.y, A.z * A.z)), 1e-20f);
    const float db2 = fmaxf(fmaf(B.x, B.x, fmaf(B.y, B.y, B.z * B.z)), 1e-20f);
    const float ra = rsq(da2), rb = rsq(db2);
    s_Xi[pa] = make_float4(A.x, B.x, A.y, B.y);
    s_Xi[pb] = make_float4(A.z, B.z, A.w, B.w);
    s_der[p * kAccThreads + tid] = make_float4(ra, rb, da2 * ra, db2 * rb);
  }

  for (int ei = grp_ptr[g]; ei < grp_ptr[g + 1]; ++ei) {
    const int e = grp_edge[ei];
    const int j = edges[2 * e + 1];
    if (tid < 12) s_T[tid] = edgeT[(size_t)e * 12 + tid];   // s_ij R_ij [9], t_ij [3] (kernel k_edge_prep)
    __syncthreads();
    double Td[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) Td[k] = s_T[k];

    const float4* __restrict__ Pj = pm + (size_t)j * HW;
    const int32_t* __restrict__ mt = match + (size_t)e * HW + px0;

    f2 acc[kAccSlots];
#pragma unroll
    for (int k = 0; k < kAccSlots; ++k) acc[k] = make_float2(0.f, 0.f);
    unsigned int cnt = 0, sum_m = 0, sum_n = 0;   // <= 16 terms each < 2^28: no overflow (HW <= 2^28 checked at create)

    auto ld_idx = [&](int row) -> int {
      const int p = row * kAccThreads + tid;
      return (p < npx) ? __ldcs(mt + p) : -1;
    };
    auto gather = [&](int n) -> float4 {
      return ((unsigned)n < (unsigned)HW) ? __ldg(Pj + n) : make_float4(0.f, 0.f, 0.f, -1.f);
    };
    // delta = T_ij X_j - X_i in FP64: |delta| ~ noise << |x|; in fp32 it would carry ~ulp(|x|) per match
    auto delta = [&](const float4 Xj, float xi0, float xi1, float xi2, float& d0, float& d1, float& d2_) {
      const double Xjx = (double)Xj.x, Xjy = (double)Xj.y, Xjz = (double)Xj.z;
      d0 = (float)fma(Td[0], Xjx, fma(Td[1], Xjy, fma(Td[2], Xjz, Td[9] - (double)xi0)));
      d1 = (float)fma(Td[3], Xjx, fma(Td[4], Xjy, fma(Td[5], Xjz, Td[10] - (double)xi1)));
      d2_ = (float)fma(Td[6], Xjx, fma(Td[7], Xjy, fma(Td[8], Xjz, Td[11] - (double)xi2)));
    };
    auto process = [&](int p, int nA, int nB, const float4 XjA, const float4 XjB) {
      if (XjA.w < 0.f && XjB.w < 0.f) return;               // neither lane has a match (whole invalid bands: warp-uniform)
      const int pa = 2 * p * kAccThreads + tid, pb = pa + kAccThreads;
      const float4 P0 = s_Xi[pa], P1 = s_Xi[pb];           // (xA, xB, yA, yB), (zA, zB, wA, wB)
      const bool vA = (XjA.w >= 0.f) && (P1.z >= 0.f), vB = (XjB.w >= 0.f) && (P1.w >= 0.f);
      if (!(vA || vB)) return;
      const float4 der = s_der[p * kAccThreads + tid];
      f2 del0, del1, del2;
      delta(XjA, P0.x, P0.z, P1.x, del0.x, del1.x, del2.x);
      delta(XjB, P0.y, P0.w, P1.y, del0.y, del1.y, del2.y);
      f2 sq = make_float2(P1.z, P1.w) * make_float2(XjA.w, XjB.w);
      sq.x = vA ? sq.x : 0.f;
      sq.y = vB ? sq.y : 0.f;
      accumulate_pair(acc, del0, del1, del2, make_float2(P0.x, P0.y), make_float2(P0.z, P0.w), make_float2(P1.x, P1.y),
                      make_float2(der.x, der.y), make_float2(der.z, der.w), sq, prm);
      cnt += (vA ? 1u : 0u) + (vB ? 1u : 0u);
      sum_m += (vA ? (unsigned)pa : 0u) + (vB ? (unsigned)pb : 0u);
      sum_n += (vA ? (unsigned)nA : 0u) + (vB ? (unsigned)nB : 0u);
    };

    // software pipeline over the thread's pairs: indices two pairs ahead, gathers one pair ahead
    int nA0 = ld_idx(0), nA1 = ld_idx(1);
    int nB0 = ld_idx(2), nB1 = ld_idx(3);
    float4 XA0 = gather(nA0), XA1 = gather(nA1);
#pragma unroll 1
    for (int p = 0; p < kPairs; ++p) {
      const float4 XB0 = gather(nB0), XB1 = gather(nB1);
      const int nC0 = ld_idx(2 * p + 4), nC1 = ld_idx(2 * p + 5);
      process(p, nA0, nA1, XA0, XA1);
      nA0 = nB0; nA1 = nB1; XA0 = XB0; XA1 = XB1; nB0 = nC0; nB1 = nC1;
    }

    // ---- lanes A + B -> thread partials (fp32, <= 16 terms) -> FP64 warp sums -> fixed-order cross-warp sum ----
    {
      float accs[kSlots];
#pragma unroll
      for (int k = 0; k < kSlots; ++k) accs[k] = (k < kAccSlots) ? acc[k].x + acc[k].y : 0.f;
      warp_reduce_slots(accs, s_red + warp * kSlots, lane);
    }
    unsigned long long chk = (unsigned long long)sum_m + (unsigned long long)cnt * (unsigned long long)px0;   // sum of m
    chk = chk * (unsigned long long)HW + (unsigned long long)sum_n;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
      chk += __shfl_xor_sync(0xffffffffu, chk, o);
    }
    if (lane == 0) { s_cnt[warp] = cnt; s_chk[warp] = chk; }
    __syncthreads();
    double* out = partials + ((size_t)e * tiles + tile) * kPartialStride;
    if (tid < kSlotCnt) {
      double v = 0.0;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) v += s_red[w * kSlots + tid];
      out[tid] = v;
    } else if (tid == kSlotCnt) {
      long long c = 0;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) c += s_cnt[w];
      reinterpret_cast<long long*>(out)[kSlotCnt] = c;
    } else if (tid == kSlotChk) {
      unsigned long long h = 0ull;
#pragma unroll
      for (int w = 0; w < kWarps; ++w) h += s_chk[w];
      reinterpret_cast<unsigned long long*>(out)[kSlotChk] = h;
    }
  }
}

// a1: per-edge pose prep, T_ij = T_i^-1 T_j -> s_ij R_ij [9] row-major, t_ij [3], FP64
__global__ void __launch_bounds__(128)
k_edge_prep(const double* __restrict__ poses, const int32_t* __restrict__ edges, double* __restrict__ edgeT, int E) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= E) return;
  const Sim3d Tij = relative_pose(load_pose(poses + 8 * edges[2 * e]), load_pose(poses + 8 * edges[2 * e + 1]));
  double* o = edgeT + (size_t)e * 12;
#pragma unroll
  for (int k = 0; k < 9; ++k) o[k] = Tij.s * Tij.R[k];
#pragma unroll
  for (int k = 0; k < 3; ++k) o[9 + k] = Tij.t[k];
}

// Kernel 2: per edge, sum the tile partials in tile order (FP64), then the adjoint congruence
// A_e = Ad^T M Ad, b_e = Ad^T c with Ad = Ad_{T_i^-1}.
__global__ void __launch_bounds__(64)
k_finalize(const double* __restrict__ partials, const int32_t* __restrict__ edges, const double* __restrict__ poses,
           double* __restrict__ blocks35, double* __restrict__ edge_cost, int32_t* __restrict__ n_valid,
           unsigned long long* __restrict__ checksum, int chunks) {
  __shared__ double s_sum[kSlots];
  __shared__ double s_M[49], s_Ad[49], s_T[49];
  const int e = blockIdx.x, t = threadIdx.x;
  const double* p = partials + (size_t)e * chunks * kPartialStride;
  if (t < kSlotCnt) {
    double v = 0.0;
    for (int c = 0; c < chunks; ++c) v += p[(size_t)c * kPartialStride + t];
    s_sum[t] = v;
  } else if (t == kSlotCnt) {
    long long v = 0;
    for (int c = 0; c < chunks; ++c) v += reinterpret_cast<const long long*>(p + (size_t)c * kPartialStride)[kSlotCnt];
    n_valid[e] = (int32_t)v;
  } else if (t == kSlotChk) {
    unsigned long long v = 0ull;
    for (int c = 0; c < chunks; ++c) v += reinterpret_cast<const unsigned long long*>(p + (size_t)c * kPartialStride)[kSlotChk];
    checksum[e] = v;
  } else if (t == 39) {
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
    edge_cost[e] = s_sum[35] - 0.5 * s_sum[36];   // rho = w r^2 - min(r^2, kappa^2) / 2
  }
}

// packs [N][HW][3] points + [N][HW] confidences into float4 (x, y, z, w): w = c^(1/4) (sqrt q = w_i w_j) when the pixel
// passes the confidence test c > conf_min (decided here, exactly, on the caller's c), else -1.
__global__ void k_pack(const float* __restrict__ pts, const float* __restrict__ conf, float4* __restrict__ pm, size_t total,
                       float conf_min) {
  size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (; idx < total; idx += stride) {
    const float c = conf[idx];
    pm[idx] = make_float4(pts[3 * idx], pts[3 * idx + 1], pts[3 * idx + 2], (c > conf_min) ? sqrtf(sqrtf(fmaxf(c, 0.f))) : -1.f);
  }
}

}  // namespace

cudaError_t launch_pack(Ctx* c, const float* d_points, const float* d_conf) {
  const size_t total = (size_t)c->N * c->HW;
  const int grid = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
  k_pack<<<grid, 256, 0, c->stream>>>(d_points, d_conf, c->pm, total, c->prm.conf_min);
  ++c->launches;
  return cudaGetLastError();
}

cudaError_t launch_accumulate(Ctx* c) {
  if (c->E == 0) return cudaSuccess;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k_accumulate, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAccSmem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  DevParams p;
  p.inv_var_ray = 1.0f / (c->prm.sigma_ray * c->prm.sigma_ray);
  p.inv_var_dist = 1.0f / (c->prm.sigma_dist * c->prm.sigma_dist);
  p.k_over_sigma_ray = c->prm.huber_k / c->prm.sigma_ray;
  p.k_over_sigma_dist = c->prm.huber_k / c->prm.sigma_dist;
  p.huber_k2 = c->prm.huber_k * c->prm.huber_k;
  k_edge_prep<<<(c->E + 127) / 128, 128, 0, c->stream>>>(c->poses, c->edges, c->edgeT, c->E);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  k_accumulate<<<c->n_groups * c->chunks, kAccThreads, kAccSmem, c->stream>>>(
      c->pm, c->match, c->edges, c->grp_kf, c->grp_ptr, c->grp_edge, c->edgeT, c->partials, c->HW, c->chunks, p);
  err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  if (c->profiling) cudaEventRecord(c->ev[1], c->stream);
  k_finalize<<<c->E, 64, 0, c->stream>>>(c->partials, c->edges, c->poses, c->blocks35, c->edge_cost, c->n_valid,
                                         c->checksum, c->chunks);
  c->launches += 3;
  return cudaGetLastError();
}

}  // namespace sim3ba
