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
// Work decomposition: one warp = one CTA = one (keyframe i, slice of 512 pixels of i), 14-15 CTAs per
// SM.  The slice of X_i is staged in shared memory ONCE by a TMA bulk copy (cp.async.bulk + mbarrier) and reused by every
// edge (i, j) that leaves i; per edge the match indices arrive by a TMA bulk copy one edge ahead, X_j is gathered by
// per-lane cp.async into a two-slot ring one pair ahead of the arithmetic.  Every thread evaluates TWO matches at a time
// in the two lanes of packed fp32x2 instructions (FFMA2 / FMUL2 / FADD2: one issue slot per two lanes), accumulators
// included.
//
// Precision plan: delta = T_ij X_j - X_i in FP64 (the one cancellation of the residual); everything
// after it, the per-thread partial sums (<= 8 terms per lane, 16 per thread) and the first two levels of
// the warp tree (<= 64 terms) in fp32; every sum from there upwards (warp, edge, adjoint congruence) in FP64.  The rare
// matches whose x = X_i + delta itself cancels (|x| < |X_i| / 32: a stray match mapped next to the camera centre) are
// DEFERRED: kernel 1 leaves them out of its fp32 sums and marks them, k_deferred evaluates them in FP64 from the
// definitions, k_finalize adds them to the edge.  No floating-point atomics: every reduction has a fixed order,
// results are run-to-run identical.
#include "f32x2.cuh"
#include "sim3ba_internal.cuh"
#include "sim3_math.cuh"

namespace sim3ba {

namespace {

static_assert(kTilePx == 16 * kAccThreads, "precision plan: <= 16 fp32 terms per thread partial (8 per lane)");
constexpr int kPairs = kTilePx / (2 * kAccThreads);   // match pairs per thread and edge
constexpr int kWarps = kAccThreads / 32;
constexpr int kWarpPx = kTilePx / kWarps;      // contiguous pixels owned by one warp (64 per pair: A = 64 p + lane, B = A + 32)
constexpr int kStages = 2;                     // ring of gathered X_j pairs per warp: gathers run kStages - 1 pairs ahead.  Two stages and
                                               // no stored 1/|X_i| (14.1 KB + 1 KB reserved per one-warp CTA) let 14 warps share the 228 KB
                                               // of an SM.  Measured on C2: 12 warps / 3 stages 177.6 us, 13 / 2 171.3, 14 / 2 165.8; 16 warps
                                               // with the index buffer refilled in halves 167.8 (not kept)
constexpr float kCancel = 1.0f / 1024.0f;      // |x|^2 < kCancel |X_i|^2: x = X_i + del has lost 5 bits or more -> the match is deferred to FP64
constexpr int kSlots = 40;                     // reduction slots of a record (layout: sim3ba_internal.cuh)
constexpr int kAccSlots = 37;                  // slots that carry floating-point sums
#ifndef SIM3BA_ACC_UNROLL
#define SIM3BA_ACC_UNROLL 4
#endif
constexpr int kPairUnroll = SIM3BA_ACC_UNROLL;  // unrolling of the pair loop (8 pairs per edge and slice)

// shared-memory carve-up of k_accumulate (dynamic); every array is sliced per warp
// one contiguous region per warp, so that every shared-memory address of the pair loop is (warp base + lane * size) + constant
constexpr size_t kOffXi = 0;                                            // float4 [kWarpPx], re-laid as lane pairs
constexpr size_t kOffIdx = kOffXi + sizeof(float4) * kWarpPx;           // int32 [2][kWarpPx]
constexpr size_t kOffRing = kOffIdx + sizeof(int32_t) * 2 * kWarpPx;    // float4 [kStages][64]: gathered X_j in flight
constexpr size_t kOffBar = kOffRing + sizeof(float4) * kStages * 64;    // mbarrier [3]
constexpr size_t kWarpBytes = (kOffBar + sizeof(uint64_t) * 3 + 127) / 128 * 128;
constexpr size_t kAccSmem = kWarpBytes * kWarps;
#ifndef SIM3BA_ACC_WARPS_PER_SM
#define SIM3BA_ACC_WARPS_PER_SM 14
#endif
constexpr int kAccCtasPerSm = SIM3BA_ACC_WARPS_PER_SM / kWarps;     // warps per SM: bounded by registers (<= 152) and shared memory
static_assert(kAccCtasPerSm * (kAccSmem + 1024) <= 228 * 1024, "kAccCtasPerSm CTAs per SM (228 KB of shared memory per SM, 1 KB reserved per CTA)");

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

// per-thread 16-byte asynchronous gather global -> shared (LDGSTS, L2 only): nothing is held in registers while in flight
__device__ __forceinline__ void cp_async16(void* dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Two valid-or-masked matches: accumulate J_xi^T Omega J_xi (25 structurally non-zero upper-triangular
// entries), J_xi^T Omega e (7) and the two robust-cost sums into acc[] (slot layout: sim3ba_internal.cuh).
//   del = T_ij X_j - X_i (fp32 rounding of the FP64 value), x = T_ij X_j and d2 = |x|^2 (from the caller: X_i + del, or
//   the FP64 value rounded where that sum cancels), Xi, rdi = 1/|X_i|,
//   sq = sqrt(q) = (c_i c_j)^(1/4), 0 for a masked lane (all its weights vanish).
__device__ __forceinline__ void accumulate_pair(f2 (&acc)[kAccSlots], const f2 del0, const f2 del1, const f2 del2,
                                                const f2 x0, const f2 x1, const f2 x2, f2 d2,
                                                const f2 Xi0, const f2 Xi1, const f2 Xi2, const f2 rdi,
                                                const f2 sq, const DevParams& prm) {
  const f2 di = fma2(Xi0, Xi0, fma2(Xi1, Xi1, Xi2 * Xi2)) * rdi;   // |X_i| (rdi is clamped: 0 for X_i = 0)
  d2.x = fmaxf(d2.x, 1e-20f); d2.y = fmaxf(d2.y, 1e-20f);
  const f2 rd = make_float2(rsq(d2.x), rsq(d2.y));
  const f2 d = d2 * rd;
  const f2 u0 = x0 * rd, u1 = x1 * rd, u2 = x2 * rd;
  // e3 = |x| - |X_i| = delta . (x + X_i) / (|x| + |X_i|);  e_r = x/|x| - X_i/|X_i| = delta/|x| - X_i e3 / (|x| |X_i|)
  const f2 den = d + di;
  const f2 e3d = fma2(del0, x0 + Xi0, fma2(del1, x1 + Xi1, del2 * (x2 + Xi2))) * make_float2(rcp(den.x), rcp(den.y));
  const f2 gsc = (e3d * rd) * rdi;
  const f2 e0 = fma2(del0, rd, -(Xi0 * gsc));
  const f2 e1 = fma2(del1, rd, -(Xi1 * gsc));
  const f2 e2 = fma2(del2, rd, -(Xi2 * gsc));
  const f2 e3 = e3d;
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
      const f2 fe = f[c] * ee[c];
      acc[35] = acc[35] + fe;                                          // sum w r^2
      // sum min(r^2, k^2) with r^2 = s e^2: where the weight is not clamped fe IS r^2 (<= k^2); where it is, fe = k |r| >= k^2
      acc[36] = acc[36] + make_float2(fminf(fe.x, prm.huber_k2), fminf(fe.y, prm.huber_k2));
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
// costs 20 + 10 + 5 + 5 + 5 exchanges instead of 40 x 5.  The first two levels add fp32 partials (two
// roundings of 2^-24 on sums of <= 64 terms -- the same order as the rounding every term already
// carries); from the 64-term partial upwards every sum is FP64.  Lanes with (lane & 3) == 0 end up
// holding the warp totals of slots base .. base + 4, base = 20 b4 + 10 b3 + 5 b2 (bits of the lane
// index), and write them to the warp's record; the lane holding slots 35..39 stores the two integers
// (warp totals, every lane has them) in slots 37 and 38.
__device__ __forceinline__ void warp_reduce_slots(const float (&acc)[kSlots], double* __restrict__ out, const int lane,
                                                  unsigned long long cnt, unsigned long long chk) {
  float h[20];
  {
    const bool up = lane & 16;
#pragma unroll
    for (int k = 0; k < 20; ++k) {
      const float keep = up ? acc[20 + k] : acc[k];
      const float send = up ? acc[k] : acc[20 + k];
      h[k] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
  }
  double v[10];
  {
    const bool up = lane & 8;
#pragma unroll
    for (int k = 0; k < 10; ++k) {
      const float keep = up ? h[10 + k] : h[k];
      const float send = up ? h[k] : h[10 + k];
      v[k] = (double)(keep + __shfl_xor_sync(0xffffffffu, send, 8));
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
    if (base == 35) {
      out[35] = v[0];
      out[36] = v[1];
      reinterpret_cast<unsigned long long*>(out)[kSlotCnt] = cnt;
      reinterpret_cast<unsigned long long*>(out)[kSlotChk] = chk;
    } else {
#pragma unroll
      for (int k = 0; k < 5; ++k) out[base + k] = v[k];
    }
  }
}

// One warp = one independent worker: it owns kWarpPx contiguous pixels of the tile (its slice of X_i and of every
// edge's match indices arrive by its own TMA bulk copies on its own mbarriers) and walks the edges leaving i without
// any CTA-wide barrier, and writes one 40-double record per (edge, slice); k_finalize sums the records in slice order.
// X_j is gathered by per-lane cp.async into a per-warp shared-memory ring, kStages - 1 pairs ahead of the arithmetic.
__global__ void __launch_bounds__(kAccThreads, kAccCtasPerSm)
k_accumulate(const float4* __restrict__ pm, const int32_t* __restrict__ match, const int32_t* __restrict__ edges,
             const int32_t* __restrict__ grp_kf, const int32_t* __restrict__ grp_ptr, const int32_t* __restrict__ grp_edge,
             const double* __restrict__ edgeT, double* __restrict__ partials, unsigned short* __restrict__ def_masks,
             int32_t* __restrict__ def_flag, int HW, int tiles, int idx_tma, DevParams prm) {
  extern __shared__ __align__(128) unsigned char smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  unsigned char* wb = smem + warp * kWarpBytes;                               // this warp's region
  float4* s_Xi = reinterpret_cast<float4*>(wb + kOffXi);                      // the warp's slice, re-laid as lane pairs
  float4* s_ring = reinterpret_cast<float4*>(wb + kOffRing);                  // [kStages][64], slot = pair % kStages
  int32_t* s_idx = reinterpret_cast<int32_t*>(wb + kOffIdx);                  // [2][kWarpPx], double-buffered over edges
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(wb + kOffBar);                // [0] X_i slice, [1], [2] index buffers

  const int g = blockIdx.x / tiles, tile = blockIdx.x - g * tiles;
  const int i = grp_kf[g];
  const int px0 = tile * kTilePx + warp * kWarpPx;                   // first pixel of this warp's slice
  const int npx = max(0, min(kWarpPx, HW - px0));                    // pixels of the slice inside the keyframe
  const int e_beg = grp_ptr[g], n_e = grp_ptr[g + 1] - e_beg;

  if (lane == 0) { mbar_init(s_bar, 1); mbar_init(s_bar + 1, 1); mbar_init(s_bar + 2, 1); }
  // pixels past the ragged end are never written by the copies: masked once (w = -1, index -1)
  for (int p = npx + lane; p < kWarpPx; p += 32) {
    s_Xi[p] = make_float4(0.f, 0.f, 0.f, -1.f);
    s_idx[p] = -1;
    s_idx[kWarpPx + p] = -1;
  }
  __syncwarp();
  // match indices of edge k (k-th edge leaving i) -> index buffer k & 1.  TMA needs 16-byte granules: HW % 4 == 0
  // (idx_tma); otherwise the lanes copy (same data, synchronous).
  auto issue_idx = [&](int k) {
    if (npx == 0) return;
    const int32_t* src = match + (size_t)grp_edge[e_beg + k] * HW + px0;
    int32_t* dst = s_idx + (k & 1) * kWarpPx;
    if (idx_tma) {
      if (lane == 0) {
        mbar_expect_tx(s_bar + 1 + (k & 1), (uint32_t)npx * 4u);
        tma_bulk_g2s(dst, src, (uint32_t)npx * 4u, s_bar + 1 + (k & 1));
      }
    } else {
      for (int p = lane; p < npx; p += 32) dst[p] = __ldcs(src + p);
      __syncwarp();
    }
  };
  auto wait_idx = [&](int k) {
    if (idx_tma && npx > 0) mbar_wait(s_bar + 1 + (k & 1), (uint32_t)(k >> 1) & 1u);
  };
  if (npx > 0 && lane == 0) {
    mbar_expect_tx(s_bar, (uint32_t)npx * 16u);
    tma_bulk_g2s(s_Xi, pm + (size_t)i * HW + px0, (uint32_t)npx * 16u, s_bar);
  }
  if (n_e > 0) issue_idx(0);
  if (npx > 0) mbar_wait(s_bar, 0);
  // Pair p of a lane = pixels A = 64 p + lane and B = A + 32 of the slice.  Re-lay the two staged float4 in place as
  // lane pairs, (xA, xB, yA, yB) in A's slot and (zA, zB, wA, wB) in B's: what the edges leaving i share.
  // Thread-private slots: no synchronisation needed.
#pragma unroll 2
  for (int p = 0; p < kPairs; ++p) {
    const int pa = 64 * p + lane, pb = pa + 32;
    const float4 A = s_Xi[pa], B = s_Xi[pb];
    s_Xi[pa] = make_float4(A.x, B.x, A.y, B.y);
    s_Xi[pb] = make_float4(A.z, B.z, A.w, B.w);
  }

  // Gathers: per-lane 16-byte cp.async into the warp's ring, kStages - 1 pairs ahead of the arithmetic, flat over the
  // (edge, pair) sequence so the pipeline never drains between edges.  An out-of-range index is a masked match.
  auto gather_pair = [&](const float4* __restrict__ Pj, const int32_t* __restrict__ ix, int p, int stage) {
    const int nA = ix[64 * p + lane], nB = ix[64 * p + 32 + lane];
    float4* dst = s_ring + stage * 64 + lane;
    if ((unsigned)nA < (unsigned)HW) cp_async16(dst, Pj + nA); else *dst = make_float4(0.f, 0.f, 0.f, -1.f);
    if ((unsigned)nB < (unsigned)HW) cp_async16(dst + 32, Pj + nB); else dst[32] = make_float4(0.f, 0.f, 0.f, -1.f);
  };
  auto pj_of = [&](int k) -> const float4* { return pm + (size_t)edges[2 * grp_edge[e_beg + k] + 1] * HW; };

  static_assert(2 * kPairs <= 16, "one 16-bit mask of deferred matches per lane and record");
  static_assert(kStages - 1 <= kPairs, "the prologue stays inside the first edge");
  if (n_e > 0) {
    wait_idx(0);
    const float4* Pj = pj_of(0);
#pragma unroll
    for (int t = 0; t < kStages - 1; ++t) { gather_pair(Pj, s_idx, t, t); cp_async_commit(); }
  }

  for (int k = 0; k < n_e; ++k) {
    const int e = grp_edge[e_beg + k];
    // index buffer (k + 1) & 1 was last read while edge k - 1 was processed: free for edge k + 1
    const bool has_next = k + 1 < n_e;
    if (has_next) issue_idx(k + 1);
    const float4* __restrict__ Pj = pj_of(k);
    const float4* __restrict__ Pj_next = has_next ? pj_of(k + 1) : Pj;
    const int32_t* __restrict__ idx = s_idx + (k & 1) * kWarpPx;
    const int32_t* __restrict__ idx_next = s_idx + ((k + 1) & 1) * kWarpPx;
    double Td[12];   // s_ij R_ij [9], t_ij [3] (kernel k_edge_prep)
#pragma unroll
    for (int q = 0; q < 12; ++q) Td[q] = __ldg(edgeT + (size_t)e * 12 + q);

    f2 acc[kAccSlots];
#pragma unroll
    for (int q = 0; q < kAccSlots; ++q) acc[q] = make_float2(0.f, 0.f);
    unsigned int cnt = 0, sum_m = 0, sum_n = 0;   // <= 16 terms each < 2^28: no overflow (HW <= 2^28 checked at create)
    unsigned defmask = 0u;                        // this thread's deferred matches of the edge (16 bits)

    // delta = T_ij X_j - X_i in FP64: |delta| ~ noise << |x|; in fp32 it would carry ~ulp(|x|) per match
    auto delta = [&](const float4 Xj, float xi0, float xi1, float xi2, float& d0, float& d1, float& d2_) {
      const double Xjx = (double)Xj.x, Xjy = (double)Xj.y, Xjz = (double)Xj.z;
      d0 = (float)fma(Td[0], Xjx, fma(Td[1], Xjy, fma(Td[2], Xjz, Td[9] - (double)xi0)));
      d1 = (float)fma(Td[3], Xjx, fma(Td[4], Xjy, fma(Td[5], Xjz, Td[10] - (double)xi1)));
      d2_ = (float)fma(Td[6], Xjx, fma(Td[7], Xjy, fma(Td[8], Xjz, Td[11] - (double)xi2)));
    };

#pragma unroll kPairUnroll
    for (int p = 0; p < kPairs; ++p) {
      // issue the gathers of the pair kStages - 1 ahead (of this edge, or of the next edge) into the slot freed last iteration
      {
        const int pn = p + kStages - 1;
        const int stage = (k * kPairs + pn) % kStages;
        if (pn < kPairs) {
          gather_pair(Pj, idx, pn, stage);
        } else if (has_next) {
          if (pn == kPairs) wait_idx(k + 1);
          gather_pair(Pj_next, idx_next, pn - kPairs, stage);
        }
        cp_async_commit();                                   // (possibly empty) group: uniform accounting
        cp_async_wait<kStages - 1>();                        // the group of pair p has landed
      }
      const float4* ring = s_ring + ((k * kPairs + p) % kStages) * 64 + lane;
      const float4 XA0 = ring[0], XA1 = ring[32];
      const int pa = 64 * p + lane, pb = pa + 32;
      const float4 P1 = s_Xi[pb];                            // (zA, zB, wA, wB)
      const bool vA = (XA0.w >= 0.f) && (P1.z >= 0.f), vB = (XA1.w >= 0.f) && (P1.w >= 0.f);
      if (__any_sync(0xffffffffu, vA || vB)) {               // whole invalid bands are skipped warp-uniformly
        const float4 P0 = s_Xi[pa];                          // (xA, xB, yA, yB)
        const f2 Xi0 = make_float2(P0.x, P0.y), Xi1 = make_float2(P0.z, P0.w), Xi2 = make_float2(P1.x, P1.y);
        const f2 d2i = fma2(Xi0, Xi0, fma2(Xi1, Xi1, Xi2 * Xi2));
        // 1 / |X_i|, recomputed per edge: a stored copy would cost the 14th warp
        const f2 rdi = make_float2(rsq(fmaxf(d2i.x, 1e-20f)), rsq(fmaxf(d2i.y, 1e-20f)));
        f2 del0, del1, del2;
        delta(XA0, P0.x, P0.z, P1.x, del0.x, del1.x, del2.x);
        delta(XA1, P0.y, P0.w, P1.y, del0.y, del1.y, del2.y);
        f2 x0 = Xi0 + del0, x1 = Xi1 + del1, x2 = Xi2 + del2;   // x = T_ij X_j
        f2 d2 = fma2(x0, x0, fma2(x1, x1, x2 * x2));
        // X_i + del carries 2^-24 |del|: where the sum cancels (a stray match mapped to within |X_i| / 32 of the camera
        // centre; the 1 / |x|^2 terms of the Jacobian then dominate its edge's block) the match is DEFERRED: its pixel goes
        // into the record's bit mask, its lane sits out with zero weight, and k_deferred evaluates it in FP64.  About one match
        // in 1e4; no branch here.
        const bool dA = vA && d2.x < d2i.x * kCancel, dB = vB && d2.y < d2i.y * kCancel;
        defmask |= (dA ? 1u : 0u) << (2 * p) | (dB ? 2u : 0u) << (2 * p);   // bit 2p: match A of pair p, bit 2p + 1: match B
        f2 sq = make_float2(P1.z, P1.w) * make_float2(XA0.w, XA1.w);
        sq.x = (vA && !dA) ? sq.x : 0.f;
        sq.y = (vB && !dB) ? sq.y : 0.f;
        accumulate_pair(acc, del0, del1, del2, x0, x1, x2, d2, Xi0, Xi1, Xi2, rdi, sq, prm);
        const unsigned mA = vA ? 0xffffffffu : 0u, mB = vB ? 0xffffffffu : 0u;
        cnt += (mA & 1u) + (mB & 1u);
        sum_m += ((unsigned)pa & mA) + ((unsigned)pb & mB);
        sum_n += ((unsigned)idx[pa] & mA) + ((unsigned)idx[pb] & mB);
      }
    }

    // ---- lanes A + B -> thread partials (fp32, <= 16 terms) -> FP64 warp sums -> the (edge, slice) record ----
    unsigned long long chk = (unsigned long long)sum_m + (unsigned long long)cnt * (unsigned long long)px0;   // sum of m
    chk = chk * (unsigned long long)HW + (unsigned long long)sum_n;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
      chk += __shfl_xor_sync(0xffffffffu, chk, o);
    }
    {
      float accs[kSlots];
#pragma unroll
      for (int q = 0; q < kSlots; ++q) accs[q] = (q < kAccSlots) ? acc[q].x + acc[q].y : 0.f;
      double* rec = partials + ((size_t)e * (tiles * kWarps) + tile * kWarps + warp) * kPartialStride;
      warp_reduce_slots(accs, rec, lane, (unsigned long long)cnt, chk);
      // deferred matches: slot kSlotDef = the lanes that hold some (0 almost always); then their 16-bit masks and the edge's flag
      const unsigned lanes_def = __ballot_sync(0xffffffffu, defmask != 0u);
      if (lane == 0) reinterpret_cast<unsigned long long*>(rec)[kSlotDef] = lanes_def;
      if (lanes_def) {
        def_masks[((size_t)e * (tiles * kWarps) + tile * kWarps + warp) * 32 + lane] = (unsigned short)defmask;
        if (lane == 0) atomicOr(def_flag + e, 1);
      }
    }
    __syncwarp();   // every lane is done with index buffer k & 1 (free for edge k + 2)
  }
}

// a1: per-edge pose prep, T_ij = T_i^-1 T_j -> s_ij R_ij [9] row-major, t_ij [3], FP64
__global__ void __launch_bounds__(128)
k_edge_prep(const double* __restrict__ poses, const int32_t* __restrict__ edges, double* __restrict__ edgeT, int32_t* __restrict__ def_flag, int E) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= E) return;
  def_flag[e] = 0;                                             // no deferred matches yet at these poses (kernel 1 marks the edge)
  const Sim3d Tij = relative_pose(load_pose(poses + 8 * edges[2 * e]), load_pose(poses + 8 * edges[2 * e + 1]));
  double* o = edgeT + (size_t)e * 12;
#pragma unroll
  for (int k = 0; k < 9; ++k) o[k] = Tij.s * Tij.R[k];
#pragma unroll
  for (int k = 0; k < 3; ++k) o[9 + k] = Tij.t[k];
}

// Kernel 2: per edge, sum the slice records (FP64, fixed order: kFinGroups interleaved running sums, then group
// 0 .. kFinGroups - 1), then the adjoint congruence A_e = Ad^T M Ad, b_e = Ad^T c with Ad = Ad_{T_i^-1}.
// Two shapes: 6 groups / 256 threads, and 24 groups / 1024 threads for few edges with many records (latency of the serial
// record loop against the number of resident CTAs); the choice depends on (E, records) only, so results stay reproducible.
// One DEFERRED match (pixel m of i, see kernel 1) in FP64, straight from the definitions: x = T_ij X_j[n], e = [u - u_i; d - d_i]
// (Eq. (1)), J_xi = [[(I - u u^T)/d, -[u]x, 0], [u^T, 0, d]] (Eq. (6)), omega_c = q min(1, kappa/|r_c|)/sigma_c^2
// (PAPER.md:76); its terms are added to the slots of the edge's sums (layout: sim3ba_internal.cuh).
struct RareParams { double sigma_ray, sigma_dist, huber_k; };
__device__ __forceinline__ void add_deferred_match(double* __restrict__ sum, const float4 Xi4, const float4 Xj4, const double* __restrict__ T, RareParams rp) {
  const double Xj[3] = {(double)Xj4.x, (double)Xj4.y, (double)Xj4.z}, Xi[3] = {(double)Xi4.x, (double)Xi4.y, (double)Xi4.z};
  double x[3];
  for (int r = 0; r < 3; ++r) x[r] = fma(T[3 * r], Xj[0], fma(T[3 * r + 1], Xj[1], fma(T[3 * r + 2], Xj[2], T[9 + r])));
  const double d = fmax(sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]), 1e-12);
  const double di = fmax(sqrt(Xi[0] * Xi[0] + Xi[1] * Xi[1] + Xi[2] * Xi[2]), 1e-12);
  const double u[3] = {x[0] / d, x[1] / d, x[2] / d};
  const double e[4] = {u[0] - Xi[0] / di, u[1] - Xi[1] / di, u[2] - Xi[2] / di, d - di};
  const double sq = (double)Xi4.w * (double)Xj4.w, q = sq * sq;            // w = c^(1/4)
  double J[4][7];
  for (int r = 0; r < 3; ++r) {
    for (int c = 0; c < 3; ++c) J[r][c] = ((r == c ? 1.0 : 0.0) - u[r] * u[c]) / d;
    J[r][6] = 0.0;
    J[3][r] = u[r];
    J[3][3 + r] = 0.0;
  }
  J[0][3] = 0.0;   J[0][4] = u[2];  J[0][5] = -u[1];                        // -[u]x
  J[1][3] = -u[2]; J[1][4] = 0.0;   J[1][5] = u[0];
  J[2][3] = u[1];  J[2][4] = -u[0]; J[2][5] = 0.0;
  J[3][6] = d;
  for (int c = 0; c < 4; ++c) {
    const double sig = c < 3 ? rp.sigma_ray : rp.sigma_dist;
    const double r = sq * e[c] / sig, ar = fabs(r);
    const double om = q * (ar <= rp.huber_k ? 1.0 : rp.huber_k / ar) / (sig * sig);
    sum[35] += om * e[c] * e[c];
    sum[36] += fmin(r * r, rp.huber_k * rp.huber_k);
    for (int a = 0; a < 7; ++a) {
      sum[28 + a] += om * J[c][a] * e[c];
      for (int b = a; b < 7; ++b) sum[a * 7 - a * (a - 1) / 2 + (b - a)] += om * J[c][a] * J[c][b];
    }
  }
}

// The deferred matches of every edge: one CTA of four warps per edge.  A thread visits the records tid, tid + 128, ... of the edge; a record
// whose slot kSlotDef is non-zero names the lanes of kernel 1 that hold deferred matches; def_masks has their 16-bit masks (bit
// 2p: pixel 64 p + lane of the record's 512-pixel slice, bit 2p + 1: pixel 64 p + 32 + lane).  Sums in FP64, in a fixed order.  def_sums [E][kSlots]: slots 0..36 as in a record.
constexpr int kDefWarps = 4;
__global__ void __launch_bounds__(32 * kDefWarps)
k_deferred(const double* __restrict__ partials, const unsigned short* __restrict__ def_masks, const int32_t* __restrict__ def_flag, int records,
           const int32_t* __restrict__ edges, const float4* __restrict__ pm, const int32_t* __restrict__ match,
           const double* __restrict__ edgeT, int HW, RareParams rp, double* __restrict__ def_sums) {
  __shared__ double s_w[kDefWarps][kSlots];
  const int e = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (def_flag[e] == 0) return;                               // almost every edge: k_finalize does not read def_sums then
  const double* p = partials + (size_t)e * records * kPartialStride;
  double sum[kAccSlots];
#pragma unroll
  for (int q = 0; q < kAccSlots; ++q) sum[q] = 0.0;
  const int i = edges[2 * e], j = edges[2 * e + 1];
  for (int c = tid; c < records; c += 32 * kDefWarps) {       // thread tid: records tid, tid + 128, ...
    const double* r = p + (size_t)c * kPartialStride;
    unsigned lanes = (unsigned)reinterpret_cast<const unsigned long long*>(r)[kSlotDef];
    while (lanes) {
      const int l = __ffs(lanes) - 1;
      lanes &= lanes - 1;
      unsigned bits = def_masks[((size_t)e * records + c) * 32 + l];
      while (bits) {
        const int b = __ffs(bits) - 1;
        bits &= bits - 1;
        const int m = c * kWarpPx + 64 * (b >> 1) + 32 * (b & 1) + l;
        if (m >= HW) continue;
        const int n = match[(size_t)e * HW + m];
        add_deferred_match(sum, pm[(size_t)i * HW + m], pm[(size_t)j * HW + n], edgeT + (size_t)e * 12, rp);
      }
    }
  }
  // per thread in record / lane / bit order, butterfly over the lanes, then the warps in order: a fixed order
#pragma unroll
  for (int q = 0; q < kAccSlots; ++q) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum[q] += __shfl_xor_sync(0xffffffffu, sum[q], o);
  }
  if (lane == 0) {
#pragma unroll
    for (int q = 0; q < kAccSlots; ++q) s_w[warp][q] = sum[q];
  }
  __syncthreads();
  if (tid < kAccSlots) {
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < kDefWarps; ++w) v += s_w[w][tid];
    def_sums[(size_t)e * kSlots + tid] = v;
  }
}

template <int kFinGroups>
__global__ void __launch_bounds__(kFinGroups * 40 + 16)
k_finalize(const double* __restrict__ partials, const int32_t* __restrict__ edges, const double* __restrict__ poses,
           double* __restrict__ blocks35, double* __restrict__ edge_cost, int32_t* __restrict__ n_valid,
           unsigned long long* __restrict__ checksum, int records, const double* __restrict__ def_sums, const int32_t* __restrict__ def_flag) {
  __shared__ double s_part[kFinGroups][kSlots];
  __shared__ double s_sum[kSlots];
  __shared__ double s_M[49], s_Ad[49], s_T[49];
  const int e = blockIdx.x, t = threadIdx.x;
  const double* p = partials + (size_t)e * records * kPartialStride;
  if (t < kFinGroups * kSlots) {
    const int grp = t / kSlots, q = t - grp * kSlots;
    if (q < kSlotCnt) {
      double v = 0.0;
      for (int c = grp; c < records; c += kFinGroups) v += p[(size_t)c * kPartialStride + q];
      s_part[grp][q] = v;
    } else {   // integer slots (and the deferred-lane masks, unused here): exact in any order
      unsigned long long v = 0ull;
      for (int c = grp; c < records; c += kFinGroups) v += reinterpret_cast<const unsigned long long*>(p + (size_t)c * kPartialStride)[q];
      reinterpret_cast<unsigned long long*>(&s_part[grp][0])[q] = v;
    }
  } else if (t == kFinGroups * kSlots) {
    adjoint_of_inverse(load_pose(poses + 8 * edges[2 * e]), s_Ad);
  }
  __syncthreads();
  if (t < kSlotCnt) {
    double v = 0.0;
#pragma unroll
    for (int grp = 0; grp < kFinGroups; ++grp) v += s_part[grp][t];
    s_sum[t] = v;
  } else if (t == kSlotCnt || t == kSlotChk) {
    unsigned long long v = 0ull;
#pragma unroll
    for (int grp = 0; grp < kFinGroups; ++grp) v += reinterpret_cast<const unsigned long long*>(&s_part[grp][0])[t];
    if (t == kSlotCnt) n_valid[e] = (int32_t)v; else checksum[e] = v;
  }
  if (t < kSlotCnt && def_flag[e] != 0) s_sum[t] += def_sums[(size_t)e * kSlots + t];   // the deferred matches of the edge, evaluated in FP64 (k_deferred)
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

cudaError_t prepare_accumulate(Ctx* c) {
  if (c->acc_ready) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(k_accumulate, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAccSmem);
  if (e == cudaSuccess) c->acc_ready = true;
  return e;
}

cudaError_t launch_accumulate(Ctx* c) {
  if (c->E == 0) return cudaSuccess;
  {
    cudaError_t e = prepare_accumulate(c);
    if (e != cudaSuccess) return e;
  }
  DevParams p;
  p.inv_var_ray = 1.0f / (c->prm.sigma_ray * c->prm.sigma_ray);
  p.inv_var_dist = 1.0f / (c->prm.sigma_dist * c->prm.sigma_dist);
  p.k_over_sigma_ray = c->prm.huber_k / c->prm.sigma_ray;
  p.k_over_sigma_dist = c->prm.huber_k / c->prm.sigma_dist;
  p.huber_k2 = c->prm.huber_k * c->prm.huber_k;
  k_edge_prep<<<(c->E + 127) / 128, 128, 0, c->stream>>>(c->poses, c->edges, c->edgeT, c->def_flag, c->E);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  // TMA bulk copies of the match indices need 16-byte granules and addresses
  const int idx_tma = (c->HW % 4 == 0) && (reinterpret_cast<uintptr_t>(c->match) % 16 == 0);
  k_accumulate<<<c->n_groups * c->chunks, kAccThreads, kAccSmem, c->stream>>>(
      c->pm, c->match, c->edges, c->grp_kf, c->grp_ptr, c->grp_edge, c->edgeT, c->partials, c->def_masks, c->def_flag, c->HW, c->chunks, idx_tma, p);
  err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  if (c->profiling) cudaEventRecord(c->ev[1], c->stream);
  const int records = c->chunks * (kAccThreads / 32);
  const RareParams rp{(double)c->prm.sigma_ray, (double)c->prm.sigma_dist, (double)c->prm.huber_k};
  k_deferred<<<c->E, 32 * kDefWarps, 0, c->stream>>>(c->partials, c->def_masks, c->def_flag, records, c->edges, c->pm, c->match, c->edgeT, c->HW, rp, c->def_sums);
  if (records >= 256 && c->E <= 600)
    k_finalize<24><<<c->E, 24 * 40 + 16, 0, c->stream>>>(c->partials, c->edges, c->poses, c->blocks35, c->edge_cost, c->n_valid,
                                                         c->checksum, records, c->def_sums, c->def_flag);
  else
    k_finalize<6><<<c->E, 6 * 40 + 16, 0, c->stream>>>(c->partials, c->edges, c->poses, c->blocks35, c->edge_cost, c->n_valid,
                                                       c->checksum, records, c->def_sums, c->def_flag);
  c->launches += 4;
  return cudaGetLastError();
}

}  // namespace sim3ba
