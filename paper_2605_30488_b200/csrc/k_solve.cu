// Kernels 3+4 of the Sim(3) GN step as ONE persistent cooperative kernel: damped assembly of the
// dense system (a6), blocked FP64 Cholesky, forward and backward triangular solves (a7) and the
// epsilon escalation of PAPER.md:122 -- all on the device, no host round trip between attempts.
//
//   Eq. (7)  PAPER.md:120   (H + lambda diag(H) + eps_r I) tau = -g
//   PAPER.md:122            eps_r = eps0 * 100^r on factorisation failure, r < max_attempts, else tau = 0
//
// Layout: L is npad x npad row-major (npad multiple of NB = 64, identity padding), lower triangle.
// One attempt:
//   phase 0  every CTA zero-fills its share of the lower-triangular 64x64 tiles, then the 7x7 blocks
//            are gathered from the per-edge blocks through the bookkeeping CSRs (fixed summation
//            order, no atomics); gauge keyframes get identity blocks; rhs = -g.
//   panel k  phase A: each participating CTA re-factorises the diagonal block L_kk in registers /
//            shared memory (redundant work instead of one more grid-wide dependency), forward-
//            substitutes y_k = L_kk^-1 b_k, solves its row blocks L_ik = A_ik L_kk^-T and updates
//            b_i -= L_ik y_k.   phase B: trailing update C_ij -= L_ik L_jk^T over the lower tiles.
//   back     L^T tau = y block by block, last to first.
// Grid-wide barriers are a monotonically increasing global counter (all CTAs are co-resident:
// the kernel is launched with cudaLaunchCooperativeKernel).
#include <cooperative_groups.h>

#include "sim3ba_internal.cuh"

namespace sim3ba {

namespace {

constexpr int NB = kNB;          // 64
constexpr int LDS = NB + 1;      // padded shared-memory row stride (doubles)
constexpr int KC = 32, LDK = KC + 1;
constexpr int kSolveThreads = 256;

struct SolveArgs {
  double* L; int npad, n, nb;
  const double* blocks35; const int32_t *kf_ptr, *kf_edge, *pair_kf, *pair_ptr, *pair_edge;
  const uint8_t* fixed; int N, n_pairs;
  const double* dense;           // non-NULL: caller-supplied dense H [n][n] instead of the blocks
  const double* g;
  double *rhs, *ysol, *Dfac, *Dinv, *tau;
  double lambda, eps0; int max_attempts;
  int32_t* status;               // [0] failure flag of the running attempt, [1] attempts used, [2] ok
  double* eps_used;
  unsigned int* bar;
};

__device__ __forceinline__ unsigned int ld_acquire(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ void grid_barrier(unsigned int* bar, unsigned int G, unsigned int& gen) {
  __syncthreads();
  gen += 1;
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(bar, 1u);
    const unsigned int target = gen * G;
    while (ld_acquire(bar) < target) { __nanosleep(32); }
    __threadfence();
  }
  __syncthreads();
}

__device__ __forceinline__ int tri_index(int r, int c) { return r * 7 - r * (r - 1) / 2 + (c - r); }

// ---- phase 0 -----------------------------------------------------------------------------------
__device__ void assemble_zero(const SolveArgs& a, int G) {
  const int nb = a.nb;
  const int ntiles = nb * (nb + 1) / 2;
  for (int t = blockIdx.x; t < ntiles; t += G) {
    int ti = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= t) ++ti;
    while (ti * (ti + 1) / 2 > t) --ti;
    const int tj = t - ti * (ti + 1) / 2;
    double2* base = reinterpret_cast<double2*>(a.L + (size_t)ti * NB * a.npad + (size_t)tj * NB);
    const size_t ld2 = (size_t)a.npad / 2;
    for (int idx = threadIdx.x; idx < NB * NB / 2; idx += kSolveThreads) {
      const int r = idx / (NB / 2), c2 = idx % (NB / 2);
      base[r * ld2 + c2] = make_double2(0.0, 0.0);
    }
  }
}

__device__ void assemble_blocks(const SolveArgs& a, int G, double eps) {
  const int grp = threadIdx.x >> 6, t = threadIdx.x & 63;   // 4 groups of 64 threads
  const int r = t / 7, c = t % 7;
  const size_t ld = (size_t)a.npad;
  const int items = a.N + a.n_pairs;
  for (int it = blockIdx.x * 4 + grp; it < items; it += G * 4) {
    if (t >= 49) continue;
    if (it < a.N) {
      if (r < c) continue;
      double v = 0.0;
      if (a.fixed[it]) {
        v = (r == c) ? 1.0 : 0.0;
      } else {
        const int idx = tri_index(c, r);
        for (int p = a.kf_ptr[it]; p < a.kf_ptr[it + 1]; ++p) v += a.blocks35[(size_t)a.kf_edge[p] * 35 + idx];
      }
      if (r == c) v = v * (1.0 + a.lambda) + eps;
      a.L[(size_t)(7 * it + r) * ld + 7 * it + c] = v;
    } else {
      const int p = it - a.N;
      const int hi = a.pair_kf[2 * p], lo = a.pair_kf[2 * p + 1];
      if (a.fixed[hi] || a.fixed[lo]) continue;
      const int idx = r <= c ? tri_index(r, c) : tri_index(c, r);
      double v = 0.0;
      for (int q = a.pair_ptr[p]; q < a.pair_ptr[p + 1]; ++q) v += a.blocks35[(size_t)a.pair_edge[q] * 35 + idx];
      a.L[(size_t)(7 * hi + r) * ld + 7 * lo + c] = -v;
    }
  }
  if (blockIdx.x == 0)
    for (int k = a.n + threadIdx.x; k < a.npad; k += kSolveThreads) a.L[(size_t)k * ld + k] = 1.0;
}

__device__ void assemble_dense(const SolveArgs& a, int G, double eps) {
  const size_t ld = (size_t)a.npad;
  for (int r = blockIdx.x; r < a.npad; r += G) {
    for (int c = threadIdx.x; c <= r; c += kSolveThreads) {
      double v;
      if (r >= a.n || c >= a.n) v = (r == c) ? 1.0 : 0.0;
      else {
        if (a.fixed[r / 7] || a.fixed[c / 7]) v = (r == c) ? 1.0 : 0.0;
        else v = a.dense[(size_t)r * a.n + c];
        if (r == c) v = v * (1.0 + a.lambda) + eps;
      }
      a.L[r * ld + c] = v;
    }
  }
}

// ---- diagonal block --------------------------------------------------------------------------
// Cholesky of the 64x64 block held as: thread (r = tid/4, g = tid%4) owns columns 4q+g of row r.
// Result is written to the shared block D (lower triangle).  Returns false on a bad pivot.
__device__ bool potrf_block(double (&a)[16], double* D, double* col, double* dinv, double* s_p, int tid) {
  const int r = tid >> 2, g = tid & 3;
  bool ok = true;
#pragma unroll
  for (int c = 0; c < NB; ++c) {
    const int qc = c >> 2, owner = c & 3;
    if (r == c && g == owner) *s_p = a[qc];
    __syncthreads();
    const double p = *s_p;
    const bool good = (p > 0.0) && (p < 1.0e300);   // false for NaN, <= 0, inf
    if (!good) ok = false;
    const double inv = good ? rsqrt(p) : 1.0;     // 1 / L_cc; one dependent rsqrt per column
    if (g == owner && r >= c) {
      const double l = (r == c) ? p * inv : a[qc] * inv;
      a[qc] = l;
      col[r] = l;
      if (r == c) dinv[c] = inv;
    }
    __syncthreads();
    if (r > c) {
      const double lr = col[r];
#pragma unroll
      for (int q = 0; q < 16; ++q) {
        const int cc = 4 * q + g;
        if (cc > c && cc <= r) a[q] = fma(-lr, col[cc], a[q]);
      }
    }
  }
#pragma unroll
  for (int q = 0; q < 16; ++q) D[r * LDS + 4 * q + g] = a[q];
  __syncthreads();
  return ok;
}

struct Smem {
  double D[NB * LDS];
  double As[NB * LDK];
  double Bs[NB * LDK];
  double y[NB];
  double col[NB];
  double dinv[NB];   // 1 / diag(L_kk)
  double s_p;
};

// phase A of panel k
__device__ bool panel_phase(const SolveArgs& a, Smem& sm, int k, int G) {
  const int tid = threadIdx.x;
  const size_t ld = (size_t)a.npad;
  const int nrows = a.nb - k;                 // block rows k .. nb-1 (row 0 = the diagonal block)
  if ((int)blockIdx.x >= nrows) return true;  // nothing to do for this CTA
  const int r = tid >> 2, g = tid & 3, lane = tid & 31;
  const double* Lkk = a.L + (size_t)k * NB * ld + (size_t)k * NB;
  double d[16];
#pragma unroll
  for (int q = 0; q < 16; ++q) d[q] = __ldcg(Lkk + r * ld + 4 * q + g);
  if (tid < NB) sm.y[tid] = __ldcg(a.rhs + k * NB + tid);
  const bool ok = potrf_block(d, sm.D, sm.col, sm.dinv, &sm.s_p, tid);
  if (!ok) {
    if (blockIdx.x == 0 && tid == 0) a.status[0] = 1;
    return false;
  }
  // y_k = D^-1 b_k (warp 0; lane owns rows lane and lane+32)
  if (tid < 32) {
    double b0 = sm.y[tid], b1 = sm.y[tid + 32];
    for (int c = 0; c < NB; ++c) {
      const double own = (c < 32) ? b0 : b1;
      const double xc = __shfl_sync(0xffffffffu, own, c & 31) * sm.dinv[c];
      if (tid == (c & 31)) { if (c < 32) b0 = xc; else b1 = xc; }
      if (tid > c) b0 -= sm.D[tid * LDS + c] * xc;
      if (tid + 32 > c) b1 -= sm.D[(tid + 32) * LDS + c] * xc;
    }
    sm.y[tid] = b0;
    sm.y[tid + 32] = b1;
  }
  __syncthreads();
  if (blockIdx.x == 0) {
    double* Dk = a.Dfac + (size_t)k * NB * NB;
    for (int idx = tid; idx < NB * NB; idx += kSolveThreads) {
      const int rr = idx / NB, cc = idx % NB;
      Dk[idx] = (cc <= rr) ? sm.D[rr * LDS + cc] : 0.0;
    }
    if (tid < NB) { a.ysol[k * NB + tid] = sm.y[tid]; a.Dinv[k * NB + tid] = sm.dinv[tid]; }
  }
  // row blocks: X D^T = A, thread (r, g) keeps columns 4q+g of row r; x_c broadcast by shuffle
  const int first = (blockIdx.x == 0) ? G : (int)blockIdx.x;   // CTA 0 only helps when G < nrows
  for (int b = first; b < nrows; b += G) {
    const int i = k + b;
    double* Aik = a.L + (size_t)i * NB * ld + (size_t)k * NB;
    double x[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = __ldcg(Aik + r * ld + 4 * q + g);
    double dot = 0.0;
#pragma unroll
    for (int c = 0; c < NB; ++c) {
      const int q = c >> 2, owner = c & 3;
      double xc = x[q] * sm.dinv[c];
      xc = __shfl_sync(0xffffffffu, xc, (lane & ~3) | owner);
      if (g == owner) { x[q] = xc; dot += xc * sm.y[c]; }
#pragma unroll
      for (int qq = 0; qq < 16; ++qq) {
        const int cc = 4 * qq + g;
        if (cc > c) x[qq] = fma(-xc, sm.D[cc * LDS + c], x[qq]);
      }
    }
#pragma unroll
    for (int q = 0; q < 16; ++q) Aik[r * ld + 4 * q + g] = x[q];
    dot += __shfl_xor_sync(0xffffffffu, dot, 1);
    dot += __shfl_xor_sync(0xffffffffu, dot, 2);
    if (g == 0) a.rhs[i * NB + r] -= dot;
  }
  return true;
}

// phase B of panel k: C_ij -= L_ik L_jk^T over the lower tiles of the trailing matrix
__device__ void update_phase(const SolveArgs& a, Smem& sm, int k, int G) {
  const int m = a.nb - k - 1;
  const int ntiles = m * (m + 1) / 2;
  const int tid = threadIdx.x;
  const size_t ld = (size_t)a.npad;
  const int tx = tid & 15, ty = tid >> 4;   // rows ty + 16 ii, cols tx + 16 jj
  for (int t = blockIdx.x; t < ntiles; t += G) {
    int ti = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= t) ++ti;
    while (ti * (ti + 1) / 2 > t) --ti;
    const int tj = t - ti * (ti + 1) / 2;
    const int i = k + 1 + ti, j = k + 1 + tj;
    const double* Ag = a.L + (size_t)i * NB * ld + (size_t)k * NB;
    const double* Bg = a.L + (size_t)j * NB * ld + (size_t)k * NB;
    double acc[4][4];
#pragma unroll
    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) acc[ii][jj] = 0.0;
    for (int kc = 0; kc < NB; kc += KC) {
      __syncthreads();
      for (int idx = tid; idx < NB * KC; idx += kSolveThreads) {
        const int rr = idx / KC, cc = idx % KC;
        sm.As[rr * LDK + cc] = __ldcg(Ag + rr * ld + kc + cc);
        sm.Bs[rr * LDK + cc] = __ldcg(Bg + rr * ld + kc + cc);
      }
      __syncthreads();
#pragma unroll 8
      for (int kk = 0; kk < KC; ++kk) {
        double av[4], bv[4];
#pragma unroll
        for (int ii = 0; ii < 4; ++ii) av[ii] = sm.As[(ty + 16 * ii) * LDK + kk];
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) bv[jj] = sm.Bs[(tx + 16 * jj) * LDK + kk];
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
          for (int jj = 0; jj < 4; ++jj) acc[ii][jj] = fma(av[ii], bv[jj], acc[ii][jj]);
      }
    }
    double* Cg = a.L + (size_t)i * NB * ld + (size_t)j * NB;
#pragma unroll
    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        const int rr = ty + 16 * ii, cc = tx + 16 * jj;
        if (i != j || cc <= rr) Cg[rr * ld + cc] = __ldcg(Cg + rr * ld + cc) - acc[ii][jj];
      }
  }
}

// backward step for block kb: tau_kb = L_kk^-T y_kb (each participating CTA, redundantly), then
// y_jb -= L[kb, jb]^T tau_kb for the block columns jb < kb this CTA owns; CTA 0 stores tau_kb.
__device__ void back_phase(const SolveArgs& a, Smem& sm, int kb, int G) {
  const int tid = threadIdx.x;
  if ((int)blockIdx.x > kb) return;
  const size_t ld = (size_t)a.npad;
  const double* Dk = a.Dfac + (size_t)kb * NB * NB;
  for (int idx = tid; idx < NB * NB; idx += kSolveThreads) {
    const int rr = idx / NB, cc = idx % NB;
    sm.D[rr * LDS + cc] = __ldcg(Dk + idx);
  }
  if (tid < NB) { sm.y[tid] = __ldcg(a.ysol + kb * NB + tid); sm.dinv[tid] = __ldcg(a.Dinv + kb * NB + tid); }
  __syncthreads();
  // D^T x = y, warp 0: lane owns x[lane], x[lane+32]; c from NB-1 down to 0
  if (tid < 32) {
    double b0 = sm.y[tid], b1 = sm.y[tid + 32];
    for (int c = NB - 1; c >= 0; --c) {
      const double own = (c < 32) ? b0 : b1;
      const double xc = __shfl_sync(0xffffffffu, own, c & 31) * sm.dinv[c];
      if (tid == (c & 31)) { if (c < 32) b0 = xc; else b1 = xc; }
      if (tid < c) b0 -= sm.D[c * LDS + tid] * xc;
      if (tid + 32 < c) b1 -= sm.D[c * LDS + tid + 32] * xc;
    }
    sm.y[tid] = b0;
    sm.y[tid + 32] = b1;
  }
  __syncthreads();
  if (blockIdx.x == 0 && tid < NB) a.tau[kb * NB + tid] = sm.y[tid];
  // 256 threads: column c = tid & 63, quarter of the rows each; reduce the 4 partial sums in smem
  const int c = tid & 63, part = tid >> 6;
  for (int jb = blockIdx.x; jb < kb; jb += G) {
    const double* Lkj = a.L + (size_t)kb * NB * ld + (size_t)jb * NB;
    double acc = 0.0;
#pragma unroll 4
    for (int rr = part * 16; rr < part * 16 + 16; ++rr) acc = fma(__ldcg(Lkj + rr * ld + c), sm.y[rr], acc);
    __syncthreads();
    sm.As[part * 64 + c] = acc;
    __syncthreads();
    if (tid < NB) a.ysol[jb * NB + tid] -= (sm.As[tid] + sm.As[64 + tid]) + (sm.As[128 + tid] + sm.As[192 + tid]);
  }
}

__global__ void __launch_bounds__(kSolveThreads)
k_solve(SolveArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
  const int G = gridDim.x;
  unsigned int gen = 0;
  bool solved = false;
  double eps = a.eps0;
  int r = 0;
  for (; r < a.max_attempts; ++r, eps *= 100.0) {
    // ---- phase 0: damped assembly, rhs = -g ----
    if (a.dense) {
      assemble_dense(a, G, eps);
    } else {
      assemble_zero(a, G);
      grid_barrier(a.bar, G, gen);
      assemble_blocks(a, G, eps);
    }
    for (int idx = blockIdx.x * kSolveThreads + threadIdx.x; idx < a.npad; idx += G * kSolveThreads)
      a.rhs[idx] = idx < a.n ? -a.g[idx] : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) a.status[0] = 0;
    grid_barrier(a.bar, G, gen);
    // ---- factorisation with the forward solve riding along ----
    bool failed = false;
    for (int k = 0; k < a.nb; ++k) {
      panel_phase(a, sm, k, G);
      grid_barrier(a.bar, G, gen);
      if (*reinterpret_cast<volatile int32_t*>(a.status) != 0) { failed = true; break; }
      if (k + 1 < a.nb) {
        update_phase(a, sm, k, G);
        grid_barrier(a.bar, G, gen);
      }
    }
    if (failed) {
      grid_barrier(a.bar, G, gen);   // everybody has seen the flag before it is cleared again
      continue;
    }
    // ---- backward substitution ----
    for (int kb = a.nb - 1; kb >= 0; --kb) {
      back_phase(a, sm, kb, G);
      if (kb > 0) grid_barrier(a.bar, G, gen);
    }
    solved = true;
    break;
  }
  if (!solved) {   // all attempts failed: zero update
    for (int idx = blockIdx.x * kSolveThreads + threadIdx.x; idx < a.npad; idx += G * kSolveThreads) a.tau[idx] = 0.0;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    a.status[1] = solved ? r + 1 : a.max_attempts;
    a.status[2] = solved ? 1 : 0;
    a.status[0] = solved ? 0 : 1;
    *a.eps_used = solved ? eps : nan("");
  }
}

}  // namespace

cudaError_t launch_solve(Ctx* c) {
  static int max_blocks_per_sm = -1, num_sms = 0;
  const size_t smem = sizeof(Smem);
  if (max_blocks_per_sm < 0) {
    cudaError_t e = cudaFuncSetAttribute(k_solve, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&max_blocks_per_sm, k_solve, kSolveThreads, smem);
    if (e != cudaSuccess) return e;
    if (max_blocks_per_sm < 1) return cudaErrorLaunchOutOfResources;
  }
  const int nb = c->npad / NB;
  // enough CTAs for the widest phase, never more than can be co-resident
  long long want = std::max<long long>({(long long)nb * (nb - 1) / 2, (long long)nb, (long long)(c->N + c->n_pairs + 3) / 4, 1LL});
  const int G = (int)std::min<long long>(want, (long long)num_sms * std::min(max_blocks_per_sm, 2));
  SolveArgs a;
  a.L = c->L; a.npad = c->npad; a.n = c->n; a.nb = nb;
  a.blocks35 = c->blocks35; a.kf_ptr = c->kf_ptr; a.kf_edge = c->kf_edge; a.pair_kf = c->pair_kf;
  a.pair_ptr = c->pair_ptr; a.pair_edge = c->pair_edge; a.fixed = c->fixed_mask; a.N = c->N; a.n_pairs = c->n_pairs;
  a.dense = c->dense_loaded ? c->Hd : nullptr;
  a.g = c->g; a.rhs = c->rhs; a.ysol = c->ysol; a.Dfac = c->Dfac; a.Dinv = c->Dinv; a.tau = c->tau;
  a.lambda = c->prm.lm_lambda; a.eps0 = c->prm.eps0; a.max_attempts = c->prm.max_attempts;
  a.status = c->fail_flag; a.eps_used = c->d_eps_used; a.bar = c->bar;
  cudaError_t e = cudaMemsetAsync(c->bar, 0, sizeof(unsigned int), c->stream);
  if (e != cudaSuccess) return e;
  void* args[] = {&a};
  e = cudaLaunchCooperativeKernel((const void*)k_solve, dim3(G), dim3(kSolveThreads), args, smem, c->stream);
  ++c->launches;
  return e;
}

}  // namespace sim3ba
