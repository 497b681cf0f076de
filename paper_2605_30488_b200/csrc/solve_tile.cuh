// Device building blocks of the tiled FP64 Cholesky (a7), shared by the persistent solve kernels
// (k_solve.cu: tile plans of the whole system; k_solve_bb.cu: the border system of the band + border
// plan): grid barrier, 64x64 POTRF / TRSM by 8-column micro-panels, DMMA trailing update, backward step.
#pragma once
#include <cooperative_groups.h>

#include "assemble_tile.cuh"
#include "sim3ba_internal.cuh"

namespace sim3ba {
namespace {

constexpr int NB = kNB;          // 64
constexpr int LDD = NB + 4;      // diagonal tile / TRSM tile in shared memory.  LDD % 16 == 4: the DMMA fragment loads of the rank-8
                                 // updates (address = (row block + lane / 4) * LDD + lane % 4) are conflict-free; the one-thread-per-row
                                 // walks of the row solves take a 4-way conflict instead.  Measured (8 warps, one rank-8 task each):
                                 // 390 cycles a task with the odd stride NB + 1, 200 with NB + 4
constexpr int LDT = NB + 4;      // DMMA operand tiles (LDT % 16 == 4: fragment loads are conflict-free)
constexpr int kSolveThreads = 256;

struct SolveArgs {
  AsmArgs as;
  double* L; int npad, n, nb;
  const int32_t *col_ptr, *col_rows, *row_ptr, *row_cols, *tiles; int n_tiles;
  double *rhs, *ysol, *Dinv, *tau;
  double eps0; int max_attempts;
  int32_t* status;               // [0] failure flag of the running attempt, [1] attempts used, [2] ok
  double* eps_used;
  unsigned int* bar;
};

struct Smem {
  double D[NB * LDD];            // diagonal tile L_kk
  double A[(NB + 1) * LDT];      // TRSM tile + right-hand-side row (stride LDD) / DMMA operand A (stride LDT)
  double B[NB * LDT];            // DMMA operand B
  double y[NB];
  double dinv[NB];               // 1 / diag(L_kk)
  double red[256];
  int flag;
};

__device__ __forceinline__ unsigned int ld_acquire(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ int ld_flag(const int32_t* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ void grid_barrier(unsigned int* bar, unsigned int G, unsigned int& gen) {
  __syncthreads();
  gen += 1;
  if (G > 1 && threadIdx.x == 0) {
    __threadfence();
    atomicAdd(bar, 1u);
    const unsigned int target = gen * G;
    while (ld_acquire(bar) < target) { }
    __threadfence();
  }
  __syncthreads();
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// 1 / sqrt(p) and 1 / p to full double precision from the FP64 MUFU estimates (rsqrt / rcp.approx.ftz.f64 = MUFU.RSQ64H /
// RCP64H on the high word, relative error e ~ 2^-22) and ONE third-order correction each: with e = 1 - p y0^2 the root is
// y0 (1 + e / 2 + 3 e^2 / 8 + O(e^3)), with e = 1 - p r0 the reciprocal is r0 (1 + e + e^2 + O(e^3)) -- e^3 ~ 1e-20 is below
// the rounding.  Dependent FP64 operations behind the MUFU: four for the root, three for the reciprocal (two Newton steps
// are six and four; an FP64 operation that waits for its operand costs ~28 cycles here, and these sit on the pivot chains).
// Pivots outside a comfortable range take the library routines.
__device__ __forceinline__ double mufu_rsqrt(double p) {        // p inside (1e-30, 1e30)
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(p));
  const double e = fma(-(p * y), y, 1.0);
  return fma(y * e, fma(e, 0.375, 0.5), y);
}
__device__ __forceinline__ double mufu_rcp(double p) {          // p inside (1e-30, 1e30)
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(p));
  const double e = fma(-p, r, 1.0);
  return fma(r * e, 1.0 + e, r);
}
__device__ __forceinline__ double fast_rsqrt(double p) { return (p > 1e-30 && p < 1e30) ? mufu_rsqrt(p) : rsqrt(p); }
__device__ __forceinline__ double fast_rcp(double p) { return (p > 1e-30 && p < 1e30) ? mufu_rcp(p) : 1.0 / p; }

// Cholesky of an N x N block (N <= 8, row stride ld) by one warp: lane r holds row r, pivots and columns travel by
// shuffles, the column updates of a pivot run in parallel over the lanes.  The chain from one pivot to the next is
// broadcast -> 1 / pivot -> one FMA: the trailing entries take a_rp a_tp / d_p from the UNSCALED column (the products and
// the shuffles do not wait for the reciprocal), and the scaling of the column by 1 / sqrt(d_p), which only the output
// needs, happens beside it.  Leaves L in the lower triangle (the strict upper triangle is zeroed) and the reciprocal
// pivots 1 / L_pp in inv[]; returns false on a pivot that is <= 0 or not finite.  kMufu: the MUFU-seeded root and
// reciprocal, valid for pivots inside (1e-30, 1e30); a block with a pivot outside is redone with the library routines
// (one warp-uniform branch per block, out of line, instead of a fallback inside every step of the chain).
template <int N, bool kMufu>
__device__ __forceinline__ int potrf_warp_impl(double* blk, int ld, double* inv, int lane) {
  double v[N];
#pragma unroll
  for (int k = 0; k < N; ++k) v[k] = (lane < N) ? blk[lane * ld + k] : 0.0;
  bool good = true, in_range = true;
#pragma unroll
  for (int p = 0; p < N; ++p) {
    const double piv = __shfl_sync(0xffffffffu, v[p], p);
    const bool gd = (piv > 0.0) && (piv < 1.0e300);           // false for NaN, <= 0, inf
    good = good && gd;
    in_range = in_range && (piv > 1e-30) && (piv < 1e30);
    const double ps = gd ? piv : 1.0;
    const double rp = kMufu ? mufu_rcp(ps) : 1.0 / ps;
    const double ap = v[p];                                    // a_rp of this lane's row, unscaled
#pragma unroll
    for (int t = p + 1; t < N; ++t) {
      const double at = __shfl_sync(0xffffffffu, ap, t);
      v[t] = fma(-(ap * at), rp, v[t]);
    }
    const double iv = kMufu ? mufu_rsqrt(ps) : rsqrt(ps);
    v[p] = ap * iv;
    if (lane == 0) inv[p] = iv;
  }
  if (kMufu && good && !in_range) return 2;                    // nothing has been written to blk yet
  if (lane < N) {
#pragma unroll
    for (int k = 0; k < N; ++k) blk[lane * ld + k] = (k <= lane) ? v[k] : 0.0;
  }
  return good ? 0 : 1;
}
template <int N>
__device__ __noinline__ int potrf_warp_lib(double* blk, int ld, double* inv, int lane) {
  return potrf_warp_impl<N, false>(blk, ld, inv, lane);
}
template <int N>
__device__ __forceinline__ bool potrf_warp(double* blk, int ld, double* inv, int lane) {
  int r = potrf_warp_impl<N, true>(blk, ld, inv, lane);
  if (r == 2) r = potrf_warp_lib<N>(blk, ld, inv, lane);
  return r == 0;
}

// ---- rank-8 update on the FP64 tensor pipe ----------------------------------------------------------
// C[rb + i][cb + j] -= sum_{s<8} X[rb + i][c0 + s] * D[cb + j][c0 + s], i, j < 8: one warp, two DMMA.8x8x4.
// X (stride ldx) holds the rows being updated, D (stride LDD) the factorised panel; C lives in X.
__device__ __forceinline__ void rank8_dmma(double* X, int ldx, const double* D, int c0, int rb, int cb, int lane) {
  const int gid = lane >> 2, tig = lane & 3;
  double* cp = X + (rb + gid) * ldx + cb + 2 * tig;
  double v0 = cp[0], v1 = cp[1];
  const double* ap = X + (rb + gid) * ldx + c0 + tig;
  const double* bp = D + (cb + gid) * LDD + c0 + tig;
  dmma884(v0, v1, -ap[0], bp[0]);
  dmma884(v0, v1, -ap[4], bp[4]);
  cp[0] = v0;
  cp[1] = v1;
}

// ---- Cholesky of the 64x64 tile in sm.D (lower triangle; the upper triangle is scratch), fused with the triangular
// solve X L_kk^T = A of the tile in sm.A (rows 0 .. nrows - 1, nrows = 0 or NB; stride LDD) and of the right-hand-side
// row NB of sm.A (if with_rhs) ---------
// Returns false (uniformly) on a pivot that is <= 0 or not finite.  Only the first npan 8-column micro-panels are
// factorised: the rows behind them are identity padding (pivot 1, nothing to eliminate; X stays 0 in those columns).
// Per micro-panel: the 8x8 diagonal block by one warp (lane = row), then every row under it -- of L_kk, of the tile and
// the right-hand side -- against that block, one thread per row, then the trailing columns of all of them by rank-8
// DMMA updates spread over the warps (the right-hand side by plain FMAs).  The rows of the tile ride along in the
// phases the factorisation has anyway: a separate triangular solve after it would pay the sixteen block barriers and
// the short task lists of the eight micro-panels a second time.
__device__ bool panel64(Smem& sm, int nrows, bool with_rhs, int tid, int npan) {
  const int lane = tid & 31, warp = tid >> 5;
  if (tid == 0) sm.flag = 0;
  if (tid >= 8 * npan && tid < NB) sm.dinv[tid] = 1.0;
  __syncthreads();
  const int nra = nrows >> 3;
  // rank-8 updates with the factor columns cf .. cf + 7 onto the column blocks jb .. jb + nj - 1: task t < nd = a lower
  // block pair (bi >= bj) of L_kk's trailing matrix, relative to block jb; the others the blocks (row block r, column
  // block jb + jj) of the tile
  auto task = [&](int cf, int jb, int nj, int t) {
    const int nd = nj * (nj + 1) / 2;
    if (t < nd) {
      int bi = 0, rem = t;
      while (rem > bi) { rem -= bi + 1; ++bi; }          // t -> (bi, bj = rem), bj <= bi
      rank8_dmma(sm.D, LDD, sm.D, cf, 8 * (jb + bi), 8 * (jb + rem), lane);
    } else {
      const int u = t - nd, r = u / nj;
      rank8_dmma(sm.A, LDD, sm.D, cf, 8 * r, 8 * (jb + u - r * nj), lane);
    }
  };
  auto rhs_update = [&](int cf, int c) {                 // right-hand-side entry c against the factor columns cf .. cf + 7
    double acc = sm.A[NB * LDD + c];
#pragma unroll
    for (int s = 0; s < 8; ++s) acc = fma(-sm.A[NB * LDD + cf + s], sm.D[c * LDD + cf + s], acc);
    sm.A[NB * LDD + c] = acc;
  };
  for (int pb = 0; pb < npan; ++pb) {
    const int c0 = 8 * pb;
    // (1) warp 0: the diagonal block.  Warps 1 .. 7 meanwhile: the updates of micro-panel pb - 1 that were not urgent --
    //     onto the column blocks behind pb (pb itself got them before the barrier) -- in the shadow of the pivot chain
    if (warp == 0) {
      if (!potrf_warp<8>(sm.D + c0 * LDD + c0, LDD, sm.dinv + c0, lane) && lane == 0) sm.flag = 1;
    } else if (pb > 0) {
      const int nj = 7 - pb, nt = nj * (nj + 1) / 2 + nra * nj;
      for (int t = warp - 1; t < nt; t += kSolveThreads / 32 - 1) task(c0 - 8, pb + 1, nj, t);
      if (with_rhs && tid >= 192 && tid < 192 + 8 * nj) rhs_update(c0 - 8, c0 + 8 + (tid - 192));
    }
    __syncthreads();
    const int below = NB - c0 - 8;                       // rows of L_kk under the diagonal block
    {                                                    // (2) x L11^T = a, one row per thread: threads 0 .. below - 1 the rows of
      double* row = nullptr;                             //     L_kk, 64 .. 64 + nrows - 1 the tile, 128 the right-hand side
      if (tid < below) row = sm.D + (c0 + 8 + tid) * LDD + c0;
      else if (tid >= NB && tid < NB + nrows) row = sm.A + (tid - NB) * LDD + c0;
      else if (tid == 2 * NB && with_rhs) row = sm.A + NB * LDD + c0;
      if (row != nullptr) {
        double x[8];
#pragma unroll
        for (int t = 0; t < 8; ++t) x[t] = row[t];
#pragma unroll
        for (int s = 0; s < 8; ++s) {
#pragma unroll
          for (int m = 0; m < s; ++m) x[s] = fma(-x[m], sm.D[(c0 + s) * LDD + c0 + m], x[s]);
          x[s] *= sm.dinv[c0 + s];
        }
#pragma unroll
        for (int t = 0; t < 8; ++t) row[t] = x[t];
      }
    }
    __syncthreads();
    // (3) the urgent updates: column block pb + 1, the next to be factorised (blocks (i, pb + 1) of L_kk, i > pb, and of
    //     the tile; eight entries of the right-hand side)
    if (pb < 7) {
      const int ni = 7 - pb, nt = ni + nra;
      for (int t = warp; t < nt; t += kSolveThreads / 32) {
        if (t < ni) rank8_dmma(sm.D, LDD, sm.D, c0, c0 + 8 + 8 * t, c0 + 8, lane);
        else rank8_dmma(sm.A, LDD, sm.D, c0, 8 * (t - ni), c0 + 8, lane);
      }
      if (with_rhs && tid >= 248) rhs_update(c0, c0 + 8 + (tid - 248));
      __syncthreads();
    }
  }
  return sm.flag == 0;
}

// ---- X L_kk^T = A for the tile in sm.A (stride LDD), rows 0..nrows-1 plus, if with_rhs, row NB -----
// Per micro-panel: every row against the 8x8 diagonal block of L_kk (one thread per row), then the remaining columns of
// the rows by rank-8 DMMA updates (the right-hand-side row by plain FMAs).
__device__ void trsm64(Smem& sm, int nrows, bool with_rhs, int tid, int npan) {
  const int lane = tid & 31, warp = tid >> 5;
  const bool row_thread = (tid < nrows) || (with_rhs && tid == NB);
  for (int pb = 0; pb < npan; ++pb) {   // the columns behind the first npan micro-panels belong to padding rows: X stays 0 there
    const int c0 = 8 * pb;
    if (row_thread) {
      double* row = sm.A + tid * LDD + c0;
      double x[8];
#pragma unroll
      for (int t = 0; t < 8; ++t) x[t] = row[t];
#pragma unroll
      for (int s = 0; s < 8; ++s) {
#pragma unroll
        for (int m = 0; m < s; ++m) x[s] = fma(-x[m], sm.D[(c0 + s) * LDD + c0 + m], x[s]);
        x[s] *= sm.dinv[c0 + s];
      }
#pragma unroll
      for (int t = 0; t < 8; ++t) row[t] = x[t];
    }
    __syncthreads();
    const int nc8 = (NB - c0 - 8) >> 3;                  // 8-column blocks still to update
    if (nrows > 0)
      for (int t = warp; t < (NB / 8) * nc8; t += kSolveThreads / 32)
        rank8_dmma(sm.A, LDD, sm.D, c0, 8 * (t / nc8), c0 + 8 + 8 * (t % nc8), lane);
    if (with_rhs && tid >= 192 && tid < 192 + 8 * nc8) {  // the right-hand-side row (warps 6, 7: last in the DMMA round-robin)
      const int c = c0 + 8 + (tid - 192);
      double acc = sm.A[NB * LDD + c];
#pragma unroll
      for (int s = 0; s < 8; ++s) acc = fma(-sm.A[NB * LDD + c0 + s], sm.D[c * LDD + c0 + s], acc);
      sm.A[NB * LDD + c] = acc;
    }
    __syncthreads();
  }
}

// ---- phase A of block column k --------------------------------------------------------------------
// Every CTA that owns a tile of the column (and CTA 0) factorises the diagonal tile for itself, its first tile riding
// along (panel64); CTA 0 stores L_kk and y_k.  A CTA with more than one tile (more tile rows than CTAs) takes the others
// by trsm64.
__device__ void panel_phase(const SolveArgs& a, Smem& sm, int k, int G) {
  const int tid = threadIdx.x;
  const size_t ld = (size_t)a.npad;
  const int cbeg = a.col_ptr[k], c = a.col_ptr[k + 1] - cbeg;
  if (blockIdx.x != 0 && (int)blockIdx.x >= c) return;
  double* Lkk = a.L + (size_t)k * NB * ld + (size_t)k * NB;
  for (int idx = tid; idx < NB * NB; idx += kSolveThreads) {
    const int r = idx >> 6, cc = idx & 63;
    sm.D[r * LDD + cc] = __ldcg(Lkk + r * ld + cc);
  }
  auto load_tile = [&](int t) -> double* {               // tile t of the column -> sm.A
    const int i = a.col_rows[cbeg + t];
    double* Aik = a.L + (size_t)i * NB * ld + (size_t)k * NB;
    for (int idx = tid; idx < NB * NB; idx += kSolveThreads) {
      const int r = idx >> 6, cc = idx & 63;
      sm.A[r * LDD + cc] = __ldcg(Aik + r * ld + cc);
    }
    return Aik;
  };
  auto store_tile = [&](int t, double* Aik) {            // X back in place; b_i -= L_ik y_k: four threads per row, 16 columns each
    const int i = a.col_rows[cbeg + t];
    for (int idx = tid; idx < NB * NB; idx += kSolveThreads) {
      const int r = idx >> 6, cc = idx & 63;
      Aik[r * ld + cc] = sm.A[r * LDD + cc];
    }
    const int r = tid >> 2, g = tid & 3;
    double dot = 0.0;
#pragma unroll
    for (int cc = 0; cc < 16; ++cc) dot = fma(sm.A[r * LDD + 16 * g + cc], sm.y[16 * g + cc], dot);
    dot += __shfl_xor_sync(0xffffffffu, dot, 1);
    dot += __shfl_xor_sync(0xffffffffu, dot, 2);
    if (g == 0) a.rhs[i * NB + r] = __ldcg(a.rhs + i * NB + r) - dot;
  };
  int t = blockIdx.x;
  const bool has_first = t < c;
  double* Aik = has_first ? load_tile(t) : nullptr;
  if (tid < NB) sm.A[NB * LDD + tid] = __ldcg(a.rhs + k * NB + tid);
  __syncthreads();
  const int npan = min(8, max(0, (a.n - k * NB + 7) / 8));   // micro-panels holding rows of the system (the rest is padding)
  if (!panel64(sm, has_first ? NB : 0, true, tid, npan)) {
    if (blockIdx.x == 0 && tid == 0) a.status[0] = 1;
    return;
  }
  if (blockIdx.x == 0) {   // the factorised diagonal tile goes back in place (strict upper triangle zero)
    for (int idx = tid; idx < NB * NB; idx += kSolveThreads) {
      const int r = idx >> 6, cc = idx & 63;
      Lkk[r * ld + cc] = (cc <= r) ? sm.D[r * LDD + cc] : 0.0;
    }
    if (tid < NB) a.Dinv[k * NB + tid] = sm.dinv[tid];
  }
  if (tid < NB) {
    const double yv = sm.A[NB * LDD + tid];
    sm.y[tid] = yv;
    if (blockIdx.x == 0) a.ysol[k * NB + tid] = yv;
  }
  __syncthreads();
  if (has_first) store_tile(t, Aik);
  for (t += G; t < c; t += G) {
    __syncthreads();
    Aik = load_tile(t);
    __syncthreads();
    trsm64(sm, NB, false, tid, npan);
    store_tile(t, Aik);
  }
  __syncthreads();
}

// ---- phase B of block column k: C_ij -= L_ik L_jk^T on the FP64 tensor pipe --------------------
__device__ void update_phase(const SolveArgs& a, Smem& sm, int k, int G) {
  const int cbeg = a.col_ptr[k], c = a.col_ptr[k + 1] - cbeg;
  const int ntasks = c * (c + 1) / 2;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gid = lane >> 2, tig = lane & 3;
  const int wm = warp & 3, wn = warp >> 2;   // rows 16 wm .. +15, columns 32 wn .. +31
  const size_t ld = (size_t)a.npad;
  for (int t = blockIdx.x; t < ntasks; t += G) {
    int ta = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((ta + 1) * (ta + 2) / 2 <= t) ++ta;
    while (ta * (ta + 1) / 2 > t) --ta;
    const int tb = t - ta * (ta + 1) / 2;
    const int i = a.col_rows[cbeg + ta], j = a.col_rows[cbeg + tb];
    const double* Ag = a.L + (size_t)i * NB * ld + (size_t)k * NB;
    const double* Bg = a.L + (size_t)j * NB * ld + (size_t)k * NB;
    for (int idx = tid; idx < NB * NB / 2; idx += kSolveThreads) {
      const int r = idx >> 5, c2 = (idx & 31) * 2;
      const double2 va = __ldcg(reinterpret_cast<const double2*>(Ag + r * ld + c2));
      *reinterpret_cast<double2*>(&sm.A[r * LDT + c2]) = va;
      if (i != j) {
        const double2 vb = __ldcg(reinterpret_cast<const double2*>(Bg + r * ld + c2));
        *reinterpret_cast<double2*>(&sm.B[r * LDT + c2]) = vb;
      }
    }
    __syncthreads();
    const double* Bs = (i != j) ? sm.B : sm.A;
    double acc[2][4][2];
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
      for (int ni = 0; ni < 4; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;
#pragma unroll 4
    for (int kk = 0; kk < NB; kk += 4) {
      double af[2], bf[4];
#pragma unroll
      for (int mi = 0; mi < 2; ++mi) af[mi] = sm.A[(16 * wm + 8 * mi + gid) * LDT + kk + tig];
#pragma unroll
      for (int ni = 0; ni < 4; ++ni) bf[ni] = Bs[(32 * wn + 8 * ni + gid) * LDT + kk + tig];
#pragma unroll
      for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) dmma884(acc[mi][ni][0], acc[mi][ni][1], af[mi], bf[ni]);
    }
    double* Cg = a.L + (size_t)i * NB * ld + (size_t)j * NB;
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
      for (int ni = 0; ni < 4; ++ni) {
        double2* p = reinterpret_cast<double2*>(Cg + (size_t)(16 * wm + 8 * mi + gid) * ld + 32 * wn + 8 * ni + 2 * tig);
        double2 v = __ldcg(p);
        v.x -= acc[mi][ni][0];
        v.y -= acc[mi][ni][1];
        *p = v;
      }
    __syncthreads();
  }
}

// backward step for block kb: tau_kb = L_kk^-T y_kb (each participating CTA, redundantly), then
// y_jb -= L[kb, jb]^T tau_kb for the non-zero tiles of row kb this CTA owns; CTA 0 stores tau_kb.
__device__ void back_phase(const SolveArgs& a, Smem& sm, int kb, int G) {
  const int tid = threadIdx.x;
  const int rbeg = a.row_ptr[kb], rc = a.row_ptr[kb + 1] - rbeg;
  if (blockIdx.x != 0 && (int)blockIdx.x >= rc) return;
  const size_t ld = (size_t)a.npad;
  const double* Lkk = a.L + (size_t)kb * NB * ld + (size_t)kb * NB;
  for (int idx = tid; idx < NB * NB; idx += kSolveThreads) {
    const int r = idx >> 6, cc = idx & 63;
    sm.D[r * LDD + cc] = __ldcg(Lkk + r * ld + cc);
  }
  if (tid < NB) { sm.y[tid] = __ldcg(a.ysol + kb * NB + tid); sm.dinv[tid] = __ldcg(a.Dinv + kb * NB + tid); }
  __syncthreads();
  // D^T x = y, warp 0: lane owns x[lane], x[lane+32]; c from NB-1 down to 0.  The entries are kept divided by their
  // own pivot (b_r / d_r, with the column entries L(c, r) / d_r: products that do not wait for anything), so that the chain
  // from one column to the next is a broadcast and one FMA
  if (tid < 32) {
    const double d0 = sm.dinv[tid], d1 = sm.dinv[tid + 32];
    double b0 = sm.y[tid] * d0, b1 = sm.y[tid + 32] * d1;
#pragma unroll 4
    for (int c = NB - 1; c >= 0; --c) {
      const double xc = __shfl_sync(0xffffffffu, (c < 32) ? b0 : b1, c & 31);
      if (tid < c) b0 = fma(-(sm.D[c * LDD + tid] * d0), xc, b0);
      if (tid + 32 < c) b1 = fma(-(sm.D[c * LDD + tid + 32] * d1), xc, b1);
    }
    sm.y[tid] = b0;
    sm.y[tid + 32] = b1;
  }
  __syncthreads();
  if (blockIdx.x == 0 && tid < NB) a.tau[kb * NB + tid] = sm.y[tid];
  // 256 threads: column c = tid & 63, a quarter of the rows each; the 4 partial sums meet in shared memory
  const int c = tid & 63, part = tid >> 6;
  for (int t = blockIdx.x; t < rc; t += G) {
    const int jb = a.row_cols[rbeg + t];
    const double* Lkj = a.L + (size_t)kb * NB * ld + (size_t)jb * NB;
    double acc = 0.0;
#pragma unroll 4
    for (int rr = part * 16; rr < part * 16 + 16; ++rr) acc = fma(__ldcg(Lkj + rr * ld + c), sm.y[rr], acc);
    __syncthreads();
    sm.red[part * 64 + c] = acc;
    __syncthreads();
    if (tid < NB)
      a.ysol[jb * NB + tid] = __ldcg(a.ysol + jb * NB + tid) - ((sm.red[tid] + sm.red[64 + tid]) + (sm.red[128 + tid] + sm.red[192 + tid]));
  }
}

}  // namespace
}  // namespace sim3ba
