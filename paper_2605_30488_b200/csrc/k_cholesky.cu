// Kernel 4 of the Sim(3) GN step: blocked FP64 Cholesky + triangular solves (a7) for
// Eq. (7) (H + lambda diag(H) + eps_r I) tau = -g; a non-positive or non-finite
// pivot raises the failure flag that drives the eps escalation of PAPER.md:122.
//
// Layout: L is npad x npad row-major (npad multiple of kNB, identity padding), lower triangle used,
// factorised in place (L L^T).  Right-looking, block size kNB = 64, per panel k:
//   k_panel : every CTA re-factorises the 64x64 diagonal block in shared memory (redundantly, which
//             removes one grid-wide dependency), forward-substitutes the right-hand side block
//             y_k = L_kk^-1 b_k, and CTA b >= 1 solves its row block L_ik = A_ik L_kk^-T and updates
//             b_i -= L_ik y_k (the forward solve rides along with the factorisation).
//   k_update: trailing update C_ij -= L_ik L_jk^T over the lower-triangular tiles (SYRK/GEMM).
// Backward substitution L^T tau = y: one k_back launch per block, last to first.
// The factorised diagonal blocks live in a side buffer Dfac[nb][64*64]; the diagonal blocks of L
// itself are left unfactorised (nothing reads them again).
#include "sim3ba_internal.cuh"

namespace sim3ba {

namespace {

constexpr int NB = kNB;
constexpr int LDS = NB + 1;  // padded shared-memory row stride (doubles)

// In-place unblocked Cholesky of the lower triangle of the NB x NB block D (shared memory).
// Returns false (for every thread) if a pivot is <= 0 or not finite.
__device__ bool potrf_block(double* D, int tid, int nthreads) {
  bool ok = true;
  for (int c = 0; c < NB; ++c) {
    const double p = D[c * LDS + c];
    const bool good = (p > 0.0) && (p < 1.0e300);  // false for NaN, <= 0, inf
    if (!good) ok = false;
    const double s = good ? sqrt(p) : 1.0;
    const double inv = 1.0 / s;
    __syncthreads();  // everybody has read the pivot
    if (tid == 0) D[c * LDS + c] = s;
    for (int r = c + 1 + tid; r < NB; r += nthreads) D[r * LDS + c] *= inv;
    __syncthreads();
    const int m = NB - 1 - c;  // trailing size
    for (int idx = tid; idx < m * m; idx += nthreads) {
      const int r = c + 1 + idx / m, cc = c + 1 + idx % m;
      if (cc <= r) D[r * LDS + cc] -= D[r * LDS + c] * D[cc * LDS + c];
    }
    __syncthreads();
  }
  return ok;
}

__global__ void __launch_bounds__(256)
k_panel(double* __restrict__ L, double* __restrict__ rhs, double* __restrict__ ysol, double* __restrict__ Dfac,
        int npad, int k, int32_t* __restrict__ fail_flag) {
  __shared__ double D[NB * LDS];
  __shared__ double y[NB];
  if (*fail_flag) return;
  const int tid = threadIdx.x;
  const size_t ld = (size_t)npad;
  const double* Lkk = L + (size_t)k * NB * ld + (size_t)k * NB;
  for (int idx = tid; idx < NB * NB; idx += 256) {
    const int r = idx / NB, c = idx % NB;
    D[r * LDS + c] = Lkk[r * ld + c];
  }
  if (tid < NB) y[tid] = rhs[k * NB + tid];
  __syncthreads();
  const bool ok = potrf_block(D, tid, 256);
  if (!ok) {
    if (blockIdx.x == 0 && tid == 0) *fail_flag = 1;
    return;
  }
  // y_k = D^-1 b_k  (warp 0; lane owns rows lane and lane+32)
  if (tid < 32) {
    double b0 = y[tid], b1 = y[tid + 32];
    for (int c = 0; c < NB; ++c) {
      const double own = (c < 32) ? b0 : b1;
      const double xc = __shfl_sync(0xffffffffu, own, c & 31) / D[c * LDS + c];
      if (tid == (c & 31)) { if (c < 32) b0 = xc; else b1 = xc; }
      if (tid > c) b0 -= D[tid * LDS + c] * xc;
      if (tid + 32 > c) b1 -= D[(tid + 32) * LDS + c] * xc;
    }
    y[tid] = b0;
    y[tid + 32] = b1;
  }
  __syncthreads();
  if (blockIdx.x == 0) {
    // The factor of the diagonal block and y_k go to side buffers: the other CTAs of this launch
    // are still reading the unfactorised block and b_k from L / rhs.
    double* Dk = Dfac + (size_t)k * NB * NB;
    for (int idx = tid; idx < NB * NB; idx += 256) {
      const int r = idx / NB, c = idx % NB;
      Dk[idx] = (c <= r) ? D[r * LDS + c] : 0.0;
    }
    if (tid < NB) ysol[k * NB + tid] = y[tid];
    return;
  }
  // row block i = k + blockIdx.x :  X D^T = A.  Thread (r = tid/4, g = tid%4) keeps the 16 columns
  // cc = g (mod 4) of row r in registers; x_c is broadcast inside the 4-lane group by shuffle.
  const int i = k + blockIdx.x;
  double* Aik = L + (size_t)i * NB * ld + (size_t)k * NB;
  const int r = tid >> 2, g = tid & 3, lane = tid & 31;
  double a[16];
#pragma unroll
  for (int q = 0; q < 16; ++q) a[q] = Aik[r * ld + 4 * q + g];
  double dot = 0.0;  // sum_c X[r][c] y[c] over my columns
#pragma unroll
  for (int c = 0; c < NB; ++c) {
    const int q = c >> 2, owner = c & 3;
    double xc = a[q] / D[c * LDS + c];
    xc = __shfl_sync(0xffffffffu, xc, (lane & ~3) | owner);
    if (g == owner) { a[q] = xc; dot += xc * y[c]; }
#pragma unroll
    for (int qq = 0; qq < 16; ++qq) {
      const int cc = 4 * qq + g;
      if (cc > c) a[qq] -= xc * D[cc * LDS + c];
    }
  }
#pragma unroll
  for (int q = 0; q < 16; ++q) Aik[r * ld + 4 * q + g] = a[q];
  dot += __shfl_xor_sync(0xffffffffu, dot, 1);
  dot += __shfl_xor_sync(0xffffffffu, dot, 2);
  if (g == 0) rhs[i * NB + r] -= dot;
}

// C_ij -= L_ik L_jk^T for the lower-triangular tiles of the trailing matrix (j <= i, both > k).
__global__ void __launch_bounds__(256)
k_update(double* __restrict__ L, int npad, int k, const int32_t* __restrict__ fail_flag) {
  constexpr int KC = 32, LDK = KC + 1;
  __shared__ double As[NB * LDK];
  __shared__ double Bs[NB * LDK];
  if (*fail_flag) return;
  // tile index -> (ti, tj), tj <= ti, row-by-row enumeration of a lower triangle
  const int t = blockIdx.x;
  int ti = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
  while ((ti + 1) * (ti + 2) / 2 <= t) ++ti;
  while (ti * (ti + 1) / 2 > t) --ti;
  const int tj = t - ti * (ti + 1) / 2;
  const int i = k + 1 + ti, j = k + 1 + tj;
  const size_t ld = (size_t)npad;
  const double* Ag = L + (size_t)i * NB * ld + (size_t)k * NB;
  const double* Bg = L + (size_t)j * NB * ld + (size_t)k * NB;
  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;  // rows ty + 16 ii, cols tx + 16 jj
  double acc[4][4];
#pragma unroll
  for (int ii = 0; ii < 4; ++ii)
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) acc[ii][jj] = 0.0;
  for (int kc = 0; kc < NB; kc += KC) {
    if (kc) __syncthreads();
    for (int idx = tid; idx < NB * KC; idx += 256) {
      const int r = idx / KC, c = idx % KC;
      As[r * LDK + c] = Ag[r * ld + kc + c];
      Bs[r * LDK + c] = Bg[r * ld + kc + c];
    }
    __syncthreads();
#pragma unroll 8
    for (int kk = 0; kk < KC; ++kk) {
      double av[4], bv[4];
#pragma unroll
      for (int ii = 0; ii < 4; ++ii) av[ii] = As[(ty + 16 * ii) * LDK + kk];
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) bv[jj] = Bs[(tx + 16 * jj) * LDK + kk];
#pragma unroll
      for (int ii = 0; ii < 4; ++ii)
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) acc[ii][jj] = fma(av[ii], bv[jj], acc[ii][jj]);
    }
  }
  double* Cg = L + (size_t)i * NB * ld + (size_t)j * NB;
#pragma unroll
  for (int ii = 0; ii < 4; ++ii)
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) {
      const int r = ty + 16 * ii, c = tx + 16 * jj;
      if (i != j || c <= r) Cg[r * ld + c] -= acc[ii][jj];
    }
}

// Backward substitution step for block kb: tau_kb = L_kk^-T y_kb (every CTA, redundantly), then
// CTA jb < kb updates y_jb -= L[kb, jb]^T tau_kb; CTA kb stores tau_kb.
__global__ void __launch_bounds__(64)
k_back(const double* __restrict__ L, const double* __restrict__ Dfac, double* __restrict__ ysol,
       double* __restrict__ tau, int npad, int kb, const int32_t* __restrict__ fail_flag) {
  __shared__ double D[NB * LDS];
  __shared__ double x[NB];
  if (*fail_flag) return;
  const int tid = threadIdx.x;
  const size_t ld = (size_t)npad;
  const double* Dk = Dfac + (size_t)kb * NB * NB;
  for (int idx = tid; idx < NB * NB; idx += 64) {
    const int r = idx / NB, c = idx % NB;
    D[r * LDS + c] = Dk[idx];
  }
  x[tid] = ysol[kb * NB + tid];
  __syncthreads();
  // D^T x = y : x_c = (y_c - sum_{r>c} D[r][c] x_r) / D[c][c], c = NB-1 .. 0
  for (int c = NB - 1; c >= 0; --c) {
    if (tid == c) x[c] = x[c] / D[c * LDS + c];
    __syncthreads();
    if (tid < c) x[tid] -= D[c * LDS + tid] * x[c];
    __syncthreads();
  }
  const int jb = blockIdx.x;
  if (jb == kb) {
    tau[kb * NB + tid] = x[tid];
    return;
  }
  const double* Lkj = L + (size_t)kb * NB * ld + (size_t)jb * NB;
  double acc = 0.0;
#pragma unroll 8
  for (int r = 0; r < NB; ++r) acc += Lkj[r * ld + tid] * x[r];
  ysol[jb * NB + tid] -= acc;
}

__global__ void k_neg_copy(double* __restrict__ dst, const double* __restrict__ g, int n, int npad) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < npad) dst[idx] = idx < n ? -g[idx] : 0.0;
}

}  // namespace

cudaError_t launch_factor_solve(Ctx* c) {
  const int nb = c->npad / NB;
  cudaError_t err = cudaMemsetAsync(c->fail_flag, 0, sizeof(int32_t), c->stream);
  if (err != cudaSuccess) return err;
  k_neg_copy<<<(c->npad + 255) / 256, 256, 0, c->stream>>>(c->rhs, c->g, c->n, c->npad);
  ++c->launches;
  for (int k = 0; k < nb; ++k) {
    k_panel<<<nb - k, 256, 0, c->stream>>>(c->L, c->rhs, c->ysol, c->Dfac, c->npad, k, c->fail_flag);
    ++c->launches;
    const int m = nb - k - 1;
    if (m > 0) {
      k_update<<<m * (m + 1) / 2, 256, 0, c->stream>>>(c->L, c->npad, k, c->fail_flag);
      ++c->launches;
    }
  }
  for (int kb = nb - 1; kb >= 0; --kb) {
    k_back<<<kb + 1, 64, 0, c->stream>>>(c->L, c->Dfac, c->ysol, c->tau, c->npad, kb, c->fail_flag);
    ++c->launches;
  }
  return cudaGetLastError();
}

}  // namespace sim3ba
