// Kernels 3+4 of the Sim(3) GN step, band + border variant (solver mode 2): ONE persistent cooperative
// kernel for damped assembly (a6), block Cholesky, both triangular solves (a7) and the epsilon escalation.
//
//   Eq. (7)  PAPER.md:120   (H + lambda diag(H) + eps_r I) tau = -g
//   PAPER.md:122            eps_r = eps0 * 100^r on factorisation failure, r < max_attempts, else tau = 0
//   PAPER.md:118            "sparse Cholesky": the pose graph is temporal chains plus a few long links
//
// The free keyframes are split on the host (bb_plan.cu) into interior keyframes -- independent
// SEGMENTS of a chain whose coupling stays inside a block band of kBand -- and BORDER keyframes
// (one endpoint of every long link, separator triples between segments).  With H = [[A, F^T], [F, C]]
// (interior first):
//   phase 0  gather the 7x7 blocks of every interior block column [D | band | border | rhs] and the dense
//            border block C from the per-edge blocks (no atomics, fixed order), damping fused;
//   phase 1  one CTA per segment: right-looking block Cholesky at 7x7 granularity, the block columns
//            streaming through a shared-memory window (cp.async), the right-hand side riding along:
//            A = L L^T, F <- F L^-T, y = L^-1 b;
//   phase 2  one CTA per border keyframe: S = C - F F^T (its block row), b_B <- b_B - F y;
//   phase 3  tiled FP64 Cholesky of the dense S (solve_tile.cuh) -> tau_B;
//   phase 4  one CTA per segment: tau_A = L^-T (y - F^T tau_B) by block back-substitution.
// A pivot <= 0 or not finite anywhere fails the attempt; the retry re-assembles with eps * 100.
#include <stdio.h>

#include <stdlib.h>

#include "solve_tile.cuh"

namespace sim3ba {

namespace {

constexpr int kWin = 8;            // block columns resident in shared memory per segment (needs > kBand + prefetch distance)
constexpr int kBackRing = 8;       // [D | band] parts in flight during the back-substitution
static_assert(kBand == 3, "the trailing update of the border blocks is written out for three band blocks");

// phase time stamps of the persistent kernel (only with sim3ba_set_profiling: a.stamps is NULL otherwise), read back by
// sim3ba_get_solve_phase_us: [0] start, [1] assembled, [2] segments eliminated, [3] barrier passed, [4] Schur rows done,
// [5] border system solved, [6] back-substitution done by the LAST CTA (stamps of the last attempt; [0..5] are CTA 0's,
// each taken behind a grid barrier or timing a phase that ends in one)
#define BB_STAMP(i)                                                                  \
  do {                                                                               \
    if (a.stamps != nullptr && blockIdx.x == 0 && threadIdx.x == 0) {                \
      unsigned long long t_;                                                         \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                         \
      a.stamps[i] = t_;                                                              \
    }                                                                                \
  } while (0)
#define BB_STAMP_LAST(i)                                                             \
  do {                                                                               \
    if (a.stamps != nullptr && threadIdx.x == 0) {                                   \
      unsigned long long t_;                                                         \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                         \
      atomicMax(a.stamps + (i), t_);                                                 \
    }                                                                                \
  } while (0)

struct BBArgs {
  unsigned long long* stamps;
  const double *blocks35, *g;
  const int32_t *kf_ptr, *kf_edge, *pair_ptr, *pair_edge;
  double lambda;
  int n_int, n_seg, n_bord, npadB, slot_doubles, max_len;
  const int32_t *seg_ptr, *seg_bptr, *seg_bord, *col_kf, *col_nb, *col_band, *col_bpair, *bord_kf, *bord_sptr, *bord_seg, *bord_slot, *bb_pair;
  const long long *col_ofs, *col_bofs;
  double *colbuf, *seg_rhs;
  SolveArgs B;                     // border system (dense tile plan); B.as is unused
  double* tau;                     // [7 N] of the whole system
  const uint8_t* fixed; int N;
  double eps0; int max_attempts;
  int32_t* status; double* eps_used; unsigned int* bar;
};

struct BBLevels {
  int n;                           // further levels behind the first (0: the border system of the first is solved densely)
  BBArgs lv[BBPlan::kMaxLevels];
};

__device__ __forceinline__ int col_stride(int nb) { return ((1 + kBand + nb) * 49 + 7 + 1) & ~1; }
__device__ __forceinline__ int tri77(int r, int c) { return r <= c ? r * 7 - r * (r - 1) / 2 + (c - r) : c * 7 - c * (c - 1) / 2 + (r - c); }

__device__ __forceinline__ void cp16(void* dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }

// element (r, c) of the 7x7 block of H between two keyframes joined by pair `pair` (H_ij = -sum A_e), 0 if no pair
__device__ __forceinline__ double pair_elem(const BBArgs& a, int pair, int r, int c) {
  if (pair < 0) return 0.0;
  const int idx = tri77(r, c);
  double v = 0.0;
  for (int q = a.pair_ptr[pair]; q < a.pair_ptr[pair + 1]; ++q) v += a.blocks35[(size_t)a.pair_edge[q] * 35 + idx];
  return -v;
}
// element (r, c) of the damped diagonal block of keyframe kf (H_kk = sum over incident edges of A_e)
__device__ __forceinline__ double diag_elem(const BBArgs& a, int kf, int r, int c, double eps) {
  const int idx = tri77(r, c);
  double v = 0.0;
  for (int p = a.kf_ptr[kf]; p < a.kf_ptr[kf + 1]; ++p) v += a.blocks35[(size_t)a.kf_edge[p] * 35 + idx];
  if (r == c) v = v * (1.0 + a.lambda) + eps;
  return v;
}

// ---- phase 0 ---------------------------------------------------------------------------------------
__device__ void bb_assemble(const BBArgs& a, double eps, int G) {
  const int tid = threadIdx.x;
  for (int c = blockIdx.x; c < a.n_int; c += G) {            // interior block columns, one CTA each
    const int nb = a.col_nb[c];
    const int nel = (1 + kBand + nb) * 49 + 7;
    const int kf = a.col_kf[c];
    double* col = a.colbuf + a.col_ofs[c];
    const int32_t* bp = a.col_bpair + a.col_bofs[c];
    for (int idx = tid; idx < nel; idx += kSolveThreads) {
      const int blk = idx / 49, e = idx - blk * 49, r = e / 7, cc = e - r * 7;
      double v;
      if (blk == 0) v = diag_elem(a, kf, r, cc, eps);
      else if (blk <= kBand) v = pair_elem(a, a.col_band[c * kBand + blk - 1], r, cc);
      else if (blk < 1 + kBand + nb) v = pair_elem(a, bp[blk - 1 - kBand], r, cc);
      else v = -a.g[7 * kf + e];                              // rhs = -g
      col[idx] = v;
    }
  }
  const int nB = a.npadB, n7 = 7 * a.n_bord;                  // dense border block C (lower tiles, full diagonal tiles)
  for (long long idx = (long long)blockIdx.x * kSolveThreads + tid; idx < (long long)nB * nB; idx += (long long)G * kSolveThreads) {
    const int R = (int)(idx / nB), C = (int)(idx - (long long)R * nB);
    if (C / kNB > R / kNB) continue;
    double v = 0.0;
    if (R >= n7 || C >= n7) v = (R == C) ? 1.0 : 0.0;
    else if (C <= R) {
      const int kr = R / 7, kc = C / 7, r = R - 7 * kr, cc = C - 7 * kc;
      v = (kr == kc) ? diag_elem(a, a.bord_kf[kr], r, cc, eps) : pair_elem(a, a.bb_pair[(size_t)kr * a.n_bord + kc], r, cc);
    }
    a.B.L[(size_t)R * nB + C] = v;
    if (C == 0) a.B.rhs[R] = (R < n7) ? -a.g[7 * a.bord_kf[R / 7] + R % 7] : 0.0;
  }
}

// ---- phase 2b: the columns of the second level, read out of S (the level-1 border system after the Schur rows) ----------
// a2's "keyframes" are border indices of the level before (a).  Column c of a2 = separator keyframe b: D = S(b, b) (the lower triangle of
// S is the valid one), band block t = S(b', b) for the next members b' of the same group, border block q = S(q, b) -- or
// S(b, q)^T where q precedes b in S -- and the right-hand side b_B(b); then the dense system of the keyframes that stay.
// the columns of group s of a2, by the calling CTA (which then eliminates them: no grid barrier in between)
__device__ void bb_assemble2_cols(const BBArgs& a, const BBArgs& a2, int s) {
  const int tid = threadIdx.x;
  const size_t nB = (size_t)a.npadB;
  const double* S = a.B.L;
  const int last = a2.seg_ptr[s + 1] - 1;                     // last column of the group
  const int32_t* sb = a2.seg_bord + a2.seg_bptr[s];
  for (int c = a2.seg_ptr[s]; c <= last; ++c) {
    const int nb = a2.col_nb[c];
    const int nel = (1 + kBand + nb) * 49 + 7;
    const int b = a2.col_kf[c];
    double* col = a2.colbuf + a2.col_ofs[c];
    for (int idx = tid; idx < nel; idx += kSolveThreads) {
      const int blk = idx / 49, e = idx - blk * 49, r = e / 7, cc = e - r * 7;
      double v = 0.0;
      if (blk == 0) {
        v = __ldcg(S + (size_t)(7 * b + max(r, cc)) * nB + 7 * b + min(r, cc));
      } else if (blk <= kBand) {
        if (c + blk <= last) v = __ldcg(S + (size_t)(7 * a2.col_kf[c + blk] + r) * nB + 7 * b + cc);
      } else if (blk < 1 + kBand + nb) {
        const int q = a2.bord_kf[sb[blk - 1 - kBand]];        // index, in the level before, of this level's border keyframe
        v = (q > b) ? __ldcg(S + (size_t)(7 * q + r) * nB + 7 * b + cc) : __ldcg(S + (size_t)(7 * b + cc) * nB + 7 * q + r);
      } else {
        v = __ldcg(a.B.rhs + 7 * b + e);
      }
      col[idx] = v;
    }
  }
  __syncthreads();                                            // the CTA's own cp.async reads follow
}

// the border system of a2 before its Schur rows: the blocks of S between the keyframes that stay (all CTAs)
__device__ void bb_assemble2_rest(const BBArgs& a, const BBArgs& a2, int G) {
  const int tid = threadIdx.x;
  const size_t nB = (size_t)a.npadB;
  const double* S = a.B.L;
  const int nB2 = a2.npadB, n72 = 7 * a2.n_bord;
  for (long long idx = (long long)blockIdx.x * kSolveThreads + tid; idx < (long long)nB2 * nB2; idx += (long long)G * kSolveThreads) {
    const int R = (int)(idx / nB2), C = (int)(idx - (long long)R * nB2);
    if (C / kNB > R / kNB) continue;
    double v = 0.0;
    if (R >= n72 || C >= n72) v = (R == C) ? 1.0 : 0.0;
    else if (C <= R) v = __ldcg(S + (size_t)(7 * a2.bord_kf[R / 7] + R % 7) * nB + 7 * a2.bord_kf[C / 7] + C % 7);
    a2.B.L[(size_t)R * nB2 + C] = v;
    if (C == 0) a2.B.rhs[R] = (R < n72) ? __ldcg(a.B.rhs + 7 * a2.bord_kf[R / 7] + R % 7) : 0.0;
  }
}

// ---- phase 1: block Cholesky of one segment -----------------------------------------------------------
struct SegSmem {
  double inv[2][8];     // 1 / diag(L_cc) of the column being eliminated (parity of the column) and of the next one
  int fail;
};

// Right-looking block Cholesky of segment s with one column of look-ahead: while warps 1..7 apply the trailing update of
// column l and write it back, warp 0 finishes the diagonal block of column l + 1 and factorises it, so the serial chain
// per column is  TRSM(l) -> max(update(l), POTRF(l + 1)).
__device__ void bb_segment(const BBArgs& a, double* win, double* brhs, SegSmem& ss, int s) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c0 = a.seg_ptr[s], len = a.seg_ptr[s + 1] - c0;
  const int nb = a.seg_bptr[s + 1] - a.seg_bptr[s];
  const int stride = col_stride(nb), chunks = stride / 2;
  const int oB = (1 + kBand) * 49, oR = oB + nb * 49;        // offsets of the border blocks and of the rhs in a column
  auto slot = [&](int l) -> double* { return win + (size_t)(l % kWin) * a.slot_doubles; };
  auto load_col = [&](int l) {                                // global -> window slot l % kWin (all threads; caller commits)
    if (l < len) {
      const double* src = a.colbuf + a.col_ofs[c0 + l];
      double* dst = slot(l);
      for (int q = tid; q < chunks; q += kSolveThreads) cp16(dst + 2 * q, src + 2 * q);
    }
  };
  for (int q = tid; q < 7 * nb; q += kSolveThreads) brhs[q] = 0.0;
  if (tid == 0) ss.fail = 0;
  for (int l = 0; l < kWin - 1; ++l) { load_col(l); cp_commit(); }
  cp_wait<kWin - 2>();                                        // column 0 has landed
  __syncthreads();
  if (warp == 0 && !potrf_warp<7>(slot(0), 7, ss.inv[0], lane) && lane == 0) ss.fail = 1;
  __syncthreads();
  for (int l = 0; l < len; ++l) {
    if (ss.fail) break;                                       // uniform: the attempt has failed
    double* col = slot(l);
    const double* inv = ss.inv[l & 1];
    const int nbnd = min(kBand, len - 1 - l);
    // (b) TRSM: every row x of [band blocks; border blocks; rhs^T] becomes x L_cc^-T (one thread per row); seven more
    //     threads do the same to the rows of the identity: row k of L_cc^-T, kept in the strict upper triangle of the
    //     diagonal block (its diagonal, 1 / L_kk, goes there at write-back) for the back-substitution
    {
      const int nrows = 7 * (nbnd + nb) + 1;
      if (tid < nrows) {
        double* row = (tid < 7 * nbnd) ? col + 49 + tid * 7 : (tid < nrows - 1) ? col + oB + (tid - 7 * nbnd) * 7 : col + oR;
        double x[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) x[k] = row[k];
#pragma unroll
        for (int k = 0; k < 7; ++k) {
#pragma unroll
          for (int m = 0; m < k; ++m) x[k] = fma(-x[m], col[k * 7 + m], x[k]);
          x[k] *= inv[k];
        }
#pragma unroll
        for (int k = 0; k < 7; ++k) row[k] = x[k];
      } else if (tid < nrows + 7) {
        const int j = tid - nrows;
        double x[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) {
          x[k] = (k == j) ? 1.0 : 0.0;
#pragma unroll
          for (int m = 0; m < k; ++m) x[k] = fma(-x[m], col[k * 7 + m], x[k]);
          x[k] *= inv[k];
        }
#pragma unroll
        for (int k = 0; k < 7; ++k) if (k > j) col[j * 7 + k] = x[k];
      }
    }
    load_col(l + kWin - 1);                                   // into the slot of column l - 1 (written back, barrier passed)
    cp_commit();
    cp_wait<kWin - 1 - kBand>();                              // columns l .. l + kBand have landed (this thread's part)
    __syncthreads();
    // (c) trailing update of the next nbnd block columns (all in the window)
    if (warp == 0) {
      if (nbnd > 0) {                                         // D(l + 1) -= L(l + 1, l) L(l + 1, l)^T, then its Cholesky
        double* tc = slot(l + 1);
        const double* Xa = col + 49;
        for (int e = lane; e < 49; e += 32) {
          const int r = e / 7, cc = e - r * 7;
          double acc = 0.0;
#pragma unroll
          for (int k = 0; k < 7; ++k) acc = fma(Xa[r * 7 + k], Xa[cc * 7 + k], acc);
          tc[e] -= acc;
        }
        __syncwarp();
        if (!potrf_warp<7>(tc, 7, ss.inv[(l + 1) & 1], lane) && lane == 0) ss.fail = 1;
      }
    } else {
      const int wt = tid - 32;                                // 0 .. 223
      constexpr int kWT = kSolveThreads - 32;
      // the few diagonal / band blocks (all but D(l + 1)) and the right-hand sides, by general indexing
      const int nbt = nbnd * (nbnd + 1) / 2;
      for (int idx = 49 + wt; idx < nbt * 49 + 7 * nbnd; idx += kWT) {
        if (idx < nbt * 49) {
          const int bt = idx / 49, e = idx - bt * 49, r = e / 7, cc = e - r * 7;
          int t = 0, blk = bt;
          while (blk >= nbnd - t) { blk -= nbnd - t; ++t; }
          double* tc = slot(l + 1 + t);
          const double* Xa = col + 49 + t * 49;               // L(l + 1 + t, l)
          const double* Xr = (blk == 0) ? Xa : col + 49 + (t + blk) * 49;   // the block whose row r meets row cc of Xa
          double* dst = (blk == 0) ? tc : tc + 49 + (blk - 1) * 49;
          double acc = 0.0;
#pragma unroll
          for (int k = 0; k < 7; ++k) acc = fma(Xr[r * 7 + k], Xa[cc * 7 + k], acc);
          dst[e] -= acc;
        } else {
          const int j = idx - nbt * 49, t = j / 7, r = j - 7 * t;
          const double* Xa = col + 49 + t * 49;
          double acc = 0.0;
#pragma unroll
          for (int k = 0; k < 7; ++k) acc = fma(Xa[r * 7 + k], col[oR + k], acc);
          slot(l + 1 + t)[oR + r] -= acc;
        }
      }
      // the border blocks F(p, l + 1 + t) -= F(p, l) L(l + 1 + t, l)^T: four blocks at a time, thread = one element
      // (r, cc) of a block, the rows of the nbnd band blocks it meets held in registers
      if (wt < 196 && nb > 0 && nbnd > 0) {
        const int grp = wt / 49, e = wt - grp * 49, r = e / 7, cc = e - r * 7;
        double xa[kBand][7];
#pragma unroll
        for (int t = 0; t < kBand; ++t)
#pragma unroll
          for (int k = 0; k < 7; ++k) xa[t][k] = (t < nbnd) ? col[49 + t * 49 + cc * 7 + k] : 0.0;
        double* t0 = slot(l + 1) + oB + e;
        double* t1 = slot(l + 2) + oB + e;
        double* t2 = slot(l + 3) + oB + e;
        for (int p = grp; p < nb; p += 4) {
          const double* F = col + oB + p * 49 + r * 7;
          double f[7];
#pragma unroll
          for (int k = 0; k < 7; ++k) f[k] = F[k];
          double a0 = 0.0, a1 = 0.0, a2 = 0.0;
#pragma unroll
          for (int k = 0; k < 7; ++k) { a0 = fma(f[k], xa[0][k], a0); a1 = fma(f[k], xa[1][k], a1); a2 = fma(f[k], xa[2][k], a2); }
          t0[p * 49] -= a0;
          if (nbnd > 1) t1[p * 49] -= a1;
          if (nbnd > 2) t2[p * 49] -= a2;
        }
      }
      for (int q = wt; q < 7 * nb; q += kWT) {                // sum_c F_c y_c, in column order
        double acc = 0.0;
#pragma unroll
        for (int k = 0; k < 7; ++k) acc = fma(col[oB + q * 7 + k], col[oR + k], acc);
        brhs[q] += acc;
      }
      // (d) the finished column goes back: L_cc (reciprocal pivots on its diagonal, L_cc^-T above it), L band, F L^-T, y
      double* dstg = a.colbuf + a.col_ofs[c0 + l];
      for (int q = wt; q < stride; q += kWT) {
        double v = col[q];
        if (q < 49 && (q % 8) == 0) v = inv[q / 8];
        dstg[q] = v;
      }
    }
    __syncthreads();
  }
  cp_wait<0>();
  __syncthreads();
  if (ss.fail) { if (tid == 0) a.status[0] = 1; return; }
  double* out = a.seg_rhs + (size_t)a.seg_bptr[s] * 7;
  for (int q = tid; q < 7 * nb; q += kSolveThreads) out[q] = brhs[q];
  __syncthreads();
}

// ---- phase 2: block row of the Schur complement on one border keyframe ---------------------------------
// For every segment (s, slot p) touching the keyframe: S(b, q) -= sum_c F_c(p) F_c(q)^T for the border keyframes q <= p of
// the segment, b_B(b) -= sum_c F_c(p) y_c.  The border parts of the block columns stream through shared memory in chunks
// of kSchurCols columns (cp.async, double-buffered).  A 7x7 block product F_c(p) F_c(q)^T is two DMMA.8x8x4 (rows and
// k padded to 8 with zeros); warp w owns the blocks q = w, w + 8, ... and sums over the columns in order.
constexpr int kSchurCols = 4;
constexpr int kSchurPairs = (kMaxSegBorder + 7) / 8;        // blocks per warp
constexpr int kSchurPart = (kMaxSegBorder * 49 + 1) & ~1;   // doubles of one column's border part in the buffer

__device__ void bb_schur_row(const BBArgs& a, double* buf, int b) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gid = lane >> 2, tig = lane & 3;
  const int nB = a.npadB;
  const int oB = (1 + kBand) * 49;
  const bool v0 = gid < 7, v1 = gid < 7 && tig < 3;           // fragment elements inside the 7x7 block
  const int f0 = gid * 7 + tig, f1 = gid * 7 + 4 + tig;
  for (int t = a.bord_sptr[b]; t < a.bord_sptr[b + 1]; ++t) {
    const int s = a.bord_seg[t], p = a.bord_slot[t];
    const int c0 = a.seg_ptr[s], len = a.seg_ptr[s + 1] - c0;
    const int32_t* sb = a.seg_bord + a.seg_bptr[s];
    const int chunks16 = ((p + 1) * 49 + 1) / 2;              // 16-byte chunks of a column's blocks 0 .. p
    const int part = 2 * chunks16;                            // doubles of one column in the buffer
    const int ccols = min(64, (kSchurCols * kSchurPart) / part);   // columns per chunk: the narrower the row, the more
    double acc[kSchurPairs][2];
#pragma unroll
    for (int j = 0; j < kSchurPairs; ++j) acc[j][0] = acc[j][1] = 0.0;
    auto stage = [&](int ch) {                                // columns ch * kSchurCols ... -> buffer ch & 1
      double* dst = buf + (size_t)(ch & 1) * kSchurCols * kSchurPart;
      const int l0 = ch * ccols, nl = min(ccols, len - l0);
      for (int q = tid; q < nl * chunks16; q += kSolveThreads) {
        const int w = q / chunks16, qq = q - w * chunks16;
        cp16(dst + w * part + 2 * qq, a.colbuf + a.col_ofs[c0 + l0 + w] + oB + 2 * qq);
      }
    };
    const int nch = (len + ccols - 1) / ccols;
    stage(0);
    cp_commit();
    for (int ch = 0; ch < nch; ++ch) {
      if (ch + 1 < nch) stage(ch + 1);
      cp_commit();
      cp_wait<1>();
      __syncthreads();
      const double* src = buf + (size_t)(ch & 1) * kSchurCols * kSchurPart;
      const int ncol = min(ccols, len - ch * ccols);
      for (int w = 0; w < ncol; ++w) {
        const double* F = src + w * part;
        const double a0 = v0 ? F[p * 49 + f0] : 0.0, a1 = v1 ? F[p * 49 + f1] : 0.0;
#pragma unroll
        for (int j = 0; j < kSchurPairs; ++j) {
          const int q = warp + 8 * j;
          if (q <= p) {
            const double b0 = v0 ? F[q * 49 + f0] : 0.0, b1 = v1 ? F[q * 49 + f1] : 0.0;
            dmma884(acc[j][0], acc[j][1], a0, b0);
            dmma884(acc[j][0], acc[j][1], a1, b1);
          }
        }
      }
      __syncthreads();                                        // the buffer is restaged two chunks later
    }
#pragma unroll
    for (int j = 0; j < kSchurPairs; ++j) {
      const int q = warp + 8 * j;
      if (q <= p && gid < 7) {
        double* dst = a.B.L + (size_t)(7 * b + gid) * nB + 7 * sb[q] + 2 * tig;
        dst[0] = __ldcg(dst) - acc[j][0];
        if (tig < 3) dst[1] = __ldcg(dst + 1) - acc[j][1];
      }
    }
    if (tid < 7) a.B.rhs[7 * b + tid] = __ldcg(a.B.rhs + 7 * b + tid) - __ldcg(a.seg_rhs + (size_t)(a.seg_bptr[s] + p) * 7 + tid);
    __syncthreads();                                          // a later segment may map the same block to another warp
  }
}

// ---- phase 3, border system of at most one tile (7 n_bord <= 64): unblocked LDL^T and both solves in shared memory
// by CTA 0 (the tiled path costs two grid barriers and a 64-pivot tile for what is here a 14 x 14 .. 63 x 63 system).
// S = L~ D L~^T with l_rc = a_rc / d_c: column c of the lower triangle keeps the UNSCALED a_rc (nothing touches it after
// pivot c), so there is no square root and no scaling pass.  One barrier per pivot, and the pivot chain is taken off
// the update: thread 0 alone produces d_{p+1} and 1 / d_{p+1} (its Newton chain) while warps 2..7 apply pivot p to the
// rest of the trailing matrix and warp 1 takes column p of the forward solve.  1 / d = 0 marks a pivot that is <= 0 or not finite.
__device__ void bb_small_border(const BBArgs& a, Smem& sm, int n7) {
  const int tid = threadIdx.x;
  const int nB = a.npadB;
  double* ipv = sm.red;                                        // [n7] 1 / d_p
  for (int idx = tid; idx < n7 * n7; idx += kSolveThreads) {
    const int r = idx / n7, c = idx - r * n7;
    if (c <= r) sm.D[r * LDD + c] = __ldcg(a.B.L + (size_t)r * nB + c);
  }
  if (tid < n7) sm.y[tid] = __ldcg(a.B.rhs + tid);
  __syncthreads();
  if (tid == 0) {
    const double d0 = sm.D[0];
    ipv[0] = ((d0 > 0.0) && (d0 < 1.0e300)) ? fast_rcp(d0) : 0.0;
  }
  __syncthreads();
  bool good = true;
  constexpr int kRows = (kSolveThreads - 64) / 16;             // update threads: warps 2.., kRows x 16
  constexpr int kRowIt = (NB + kRows - 1) / kRows, kColIt = NB / 16;
  const int ty = (tid - 64) >> 4, tx = tid & 15;
  const int lane = tid & 31;
  // warp 1 carries the forward solve L~ y = b one column per pivot, as z_c = y_c / d_c (b_r -= a_rc z_c): lanes own rows
  // lane, lane + 32
  double b0 = 0.0, b1 = 0.0;
  if (tid >= 32 && tid < 64) { b0 = lane < n7 ? sm.y[lane] : 0.0; b1 = lane + 32 < n7 ? sm.y[lane + 32] : 0.0; }
  for (int p = 0; p < n7; ++p) {
    const double ipiv = ipv[p];                                // everybody reads the same value: uniform control flow
    if (ipiv == 0.0) { good = false; break; }
    if (tid == 0) {
      if (p + 1 < n7) {                                        // the next pivot, one step ahead of its row
        const double ap = sm.D[(p + 1) * LDD + p];
        const double d = fma(-(ap * ipiv), ap, sm.D[(p + 1) * LDD + p + 1]);
        sm.D[(p + 1) * LDD + p + 1] = d;
        ipv[p + 1] = ((d > 0.0) && (d < 1.0e300)) ? fast_rcp(d) : 0.0;
      }
    } else if (tid >= 64) {                                    // all loads of a thread are independent: fully unrolled
      double lc[kColIt];
#pragma unroll
      for (int j = 0; j < kColIt; ++j) {
        const int c = p + 1 + tx + 16 * j;
        lc[j] = c < n7 ? sm.D[c * LDD + p] : 0.0;
      }
#pragma unroll
      for (int i = 0; i < kRowIt; ++i) {
        const int r = p + 1 + ty + kRows * i;
        if (r > p + 1 && r < n7) {                             // row p + 1 is its diagonal only: thread 0's
          const double arp = sm.D[r * LDD + p] * ipiv;
#pragma unroll
          for (int j = 0; j < kColIt; ++j) {
            const int c = p + 1 + tx + 16 * j;
            if (c <= r) sm.D[r * LDD + c] = fma(-arp, lc[j], sm.D[r * LDD + c]);
          }
        }
      }
    } else if (tid >= 32) {
      const double zc = __shfl_sync(0xffffffffu, p < 32 ? b0 * ipiv : b1 * ipiv, p & 31);
      if (lane == (p & 31)) { if (p < 32) b0 = zc; else b1 = zc; }
      if (lane > p && lane < n7) b0 = fma(-sm.D[lane * LDD + p], zc, b0);
      if (lane + 32 > p && lane + 32 < n7) b1 = fma(-sm.D[(lane + 32) * LDD + p], zc, b1);
    }
    __syncthreads();
  }
  if (!good) { if (tid == 0) a.status[0] = 1; return; }
  if (tid >= 32 && tid < 64) {
    const double i0 = lane < n7 ? ipv[lane] : 0.0, i1 = lane + 32 < n7 ? ipv[lane + 32] : 0.0;
    double s0 = 0.0, s1 = 0.0;                                 // L~^T x = z: x_c = z_c - (1 / d_c) sum_{r > c} a_rc x_r
    for (int c = n7 - 1; c >= 0; --c) {
      const double xc = __shfl_sync(0xffffffffu, c < 32 ? fma(-i0, s0, b0) : fma(-i1, s1, b1), c & 31);
      if (lane == (c & 31)) { if (c < 32) b0 = xc; else b1 = xc; }
      if (lane < c) s0 = fma(sm.D[c * LDD + lane], xc, s0);
      if (lane + 32 < c) s1 = fma(sm.D[c * LDD + lane + 32], xc, s1);
    }
    if (lane < n7) a.B.tau[lane] = b0;
    if (lane + 32 < n7) a.B.tau[lane + 32] = b1;
  }
  __syncthreads();
}

// ---- phase 4: back-substitution of one segment ------------------------------------------------------------
__device__ void bb_back(const BBArgs& a, double* ring, double* z, double* tb, int s) {
  const int tid = threadIdx.x, lane = tid & 31;
  const int c0 = a.seg_ptr[s], len = a.seg_ptr[s + 1] - c0;
  const int nb = a.seg_bptr[s + 1] - a.seg_bptr[s];
  const int oB = (1 + kBand) * 49, oR = oB + nb * 49;
  const int32_t* sb = a.seg_bord + a.seg_bptr[s];
  for (int q = tid; q < 7 * nb; q += kSolveThreads) tb[q] = __ldcg(a.B.tau + 7 * sb[q / 7] + q % 7);
  __syncthreads();
  for (int q = tid; q < 7 * len; q += kSolveThreads) {        // z_c = y_c - F_c^T tau_B, all columns at once
    const int l = q / 7, k = q - 7 * l;
    const double* col = a.colbuf + a.col_ofs[c0 + l];
    double acc = __ldcg(col + oR + k);
    for (int pr = 0; pr < 7 * nb; ++pr) acc = fma(-__ldcg(col + oB + pr * 7 + k), tb[pr], acc);
    z[q] = acc;
  }
  __syncthreads();
  if (tid < 32) {                                             // the chain itself: one warp, lane k owns component k
    constexpr int part = (1 + kBand) * 49;                    // [D | band] doubles of a column (even: 16-byte chunks)
    auto load = [&](int l) {
      if (l >= 0) {
        const double* src = a.colbuf + a.col_ofs[c0 + l];
        double* dst = ring + (size_t)(l % kBackRing) * part;
        for (int q = lane; q < part / 2; q += 32) cp16(dst + 2 * q, src + 2 * q);
      }
    };
    for (int l = len - 1; l > len - kBackRing; --l) { load(l); cp_commit(); }
    for (int l = len - 1; l >= 0; --l) {
      load(l - kBackRing + 1);
      cp_commit();
      cp_wait<kBackRing - 1>();
      __syncwarp();
      const double* col = ring + (size_t)(l % kBackRing) * part;
      const int nbnd = min(kBand, len - 1 - l);
      // s = z_l - sum_t L(l+1+t, l)^T tau_{l+1+t}: lane 8 t + k takes band block t, component k
      const int t = lane >> 3, k = lane & 7;
      double part_sum = 0.0;
      if (t < nbnd && k < 7) {
        const double* X = col + 49 + t * 49;
        const double* tn = z + 7 * (l + 1 + t);               // tau of column l + 1 + t (already final)
#pragma unroll
        for (int r = 0; r < 7; ++r) part_sum = fma(X[r * 7 + k], tn[r], part_sum);
      }
      const double p1 = __shfl_down_sync(0xffffffffu, part_sum, 8), p2 = __shfl_down_sync(0xffffffffu, part_sum, 16);
      double sk = (lane < 7) ? z[7 * l + lane] - ((part_sum + p1) + p2) : 0.0;
      // x = L_cc^-T s: row k of L_cc^-T sits in row k of the diagonal block, columns k .. 6
      double xk = 0.0;
#pragma unroll
      for (int m = 0; m < 7; ++m) {
        const double sm_ = __shfl_sync(0xffffffffu, sk, m);
        if (lane < 7 && m >= lane) xk = fma(col[lane * 7 + m], sm_, xk);
      }
      sk = xk;
      __syncwarp();
      if (lane < 7) {
        z[7 * l + lane] = sk;
        a.tau[7 * a.col_kf[c0 + l] + lane] = sk;
      }
      __syncwarp();
    }
    cp_wait<0>();
  }
  __syncthreads();
}

// ---- phase 3: the dense border system of t (tiled Cholesky with the forward solve riding along, then the backward
// solve; a system of one tile directly by CTA 0).  Returns true (uniformly) if a pivot failed; otherwise tau_B is final and
// a grid barrier has been passed since it was written.
__device__ bool bb_border_solve(const BBArgs& t, Smem& sm, int G, unsigned int& gen) {
  const int nbB = t.npadB / kNB;
  if (nbB == 0) return false;
  bool failed = false;
  if (nbB == 1) {                                             // one tile: direct solve by CTA 0
    if (blockIdx.x == 0) bb_small_border(t, sm, 7 * t.n_bord);
    grid_barrier(t.bar, G, gen);
    return ld_flag(t.status) != 0;
  }
  for (int k = 0; k < nbB; ++k) {                             // tiled Cholesky of S, forward solve riding along
    panel_phase(t.B, sm, k, G);
    if (t.B.col_ptr[k + 1] > t.B.col_ptr[k]) {
      grid_barrier(t.bar, G, gen);
      if (ld_flag(t.status) != 0) { failed = true; break; }
      update_phase(t.B, sm, k, G);
      grid_barrier(t.bar, G, gen);
    }
  }
  if (!failed) {
    grid_barrier(t.bar, G, gen);
    failed = ld_flag(t.status) != 0;
  }
  if (failed) return true;
  for (int kb = nbB - 1; kb >= 0; --kb) {
    back_phase(t.B, sm, kb, G);
    if (t.B.row_ptr[kb + 1] > t.B.row_ptr[kb]) grid_barrier(t.bar, G, gen);
  }
  grid_barrier(t.bar, G, gen);                                // tau_B is final
  return false;
}

// a: the graph's band + border plan.  L: its further levels: each eliminates an independent set of separator groups from
// the border system the level before left, with the same phases on columns read out of that system; the dense solve
// takes what the last level leaves.
__global__ void __launch_bounds__(kSolveThreads, 1)
k_solve_bb(const __grid_constant__ BBArgs a, const __grid_constant__ BBLevels L) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);              // phase 3 view
  double* win = reinterpret_cast<double*>(smem_raw);          // phase 1 / 4 view
  const int G = gridDim.x, tid = threadIdx.x;
  double* brhs = win + (size_t)kWin * a.slot_doubles;         // [7 kMaxSegBorder]
  SegSmem& ss = *reinterpret_cast<SegSmem*>(brhs + 7 * kMaxSegBorder);
  double* ring = win;                                         // phase 4 view
  double* z = win + (size_t)kBackRing * (1 + kBand) * 49;
  unsigned int gen = 0;
  bool solved = false;
  double eps = a.eps0;
  const int nbB = a.npadB / kNB;
  int r = 0;
  for (; r < a.max_attempts; ++r, eps *= 100.0) {
    BB_STAMP(0);
    bb_assemble(a, eps, G);
    if (blockIdx.x == 0 && tid == 0) a.status[0] = 0;
    grid_barrier(a.bar, G, gen);
    BB_STAMP(1);
    for (int s = blockIdx.x; s < a.n_seg; s += G) bb_segment(a, win, brhs, ss, s);
    BB_STAMP(2);
    grid_barrier(a.bar, G, gen);
    BB_STAMP(3);
    bool failed = ld_flag(a.status) != 0;
    if (!failed && nbB > 0) {
      for (int b = blockIdx.x; b < a.n_bord; b += G) bb_schur_row(a, win, b);
      grid_barrier(a.bar, G, gen);
      BB_STAMP(4);
      const BBArgs* prev = &a;
      for (int k = 0; k < L.n && !failed; ++k) {              // further levels: groups out of the border system of the level before
        const BBArgs& cur = L.lv[k];
        bb_assemble2_rest(*prev, cur, G);
        for (int s = blockIdx.x; s < cur.n_seg; s += G) {
          bb_assemble2_cols(*prev, cur, s);
          bb_segment(cur, win, brhs, ss, s);
        }
        grid_barrier(a.bar, G, gen);
        failed = ld_flag(a.status) != 0;
        if (!failed && cur.n_bord > 0) {
          for (int b = blockIdx.x; b < cur.n_bord; b += G) bb_schur_row(cur, win, b);
          grid_barrier(a.bar, G, gen);
        }
        prev = &cur;
      }
      if (!failed) failed = bb_border_solve(*prev, sm, G, gen);
      if (!failed) {
        for (int k = L.n - 1; k >= 0; --k) {                   // back through the levels: tau_B of the level before
          const BBArgs& cur = L.lv[k];
          const BBArgs& upper = (k > 0) ? L.lv[k - 1] : a;
          for (int s = blockIdx.x; s < cur.n_seg; s += G) bb_back(cur, ring, z, z + 7 * cur.max_len, s);
          for (int q = blockIdx.x * kSolveThreads + tid; q < 7 * cur.n_bord; q += G * kSolveThreads)
            upper.B.tau[7 * cur.bord_kf[q / 7] + q % 7] = __ldcg(cur.B.tau + q);
          grid_barrier(a.bar, G, gen);
        }
      }
    }
    if (failed) {
      grid_barrier(a.bar, G, gen);   // everybody has seen the flag before it is cleared again
      continue;
    }
    BB_STAMP(5);
    {
      for (int s = blockIdx.x; s < a.n_seg; s += G) bb_back(a, ring, z, z + 7 * a.max_len, s);
      for (int q = blockIdx.x * kSolveThreads + tid; q < 7 * a.n_bord; q += G * kSolveThreads)
        a.tau[7 * a.bord_kf[q / 7] + q % 7] = __ldcg(a.B.tau + q);
    }
    BB_STAMP_LAST(6);
    solved = true;
    break;
  }
  if (!solved) {   // all attempts failed: zero update
    for (int idx = blockIdx.x * kSolveThreads + tid; idx < 7 * a.N; idx += G * kSolveThreads) a.tau[idx] = 0.0;
  }
  if (blockIdx.x == 0 && tid == 0) {
    a.status[1] = solved ? r + 1 : a.max_attempts;
    a.status[2] = solved ? 1 : 0;
    a.status[0] = solved ? 0 : 1;
    *a.eps_used = solved ? eps : nan("");
  }
}

}  // namespace

static size_t bb_smem_bytes(const BBPlan& P, int* slot_out) {
  int max_nb = P.max_nb;
  for (int k = 0; k < P.n_lv; ++k) max_nb = std::max(max_nb, P.lv[k].max_nb);
  const int slot = ((1 + kBand + max_nb) * 49 + 7 + 1) & ~1;   // one window slot size for all levels
  const size_t smem_seg = ((size_t)kWin * slot + 7 * kMaxSegBorder) * sizeof(double) + sizeof(SegSmem);
  const size_t smem_back = ((size_t)kBackRing * (1 + kBand) * 49 + 7 * (size_t)P.max_len + 7 * kMaxSegBorder) * sizeof(double);
  const size_t smem_schur = (size_t)2 * kSchurCols * kSchurPart * sizeof(double);
  if (slot_out) *slot_out = slot;
  return std::max({sizeof(Smem), smem_seg, smem_back, smem_schur});
}

cudaError_t prepare_solve_bb(Ctx* c) {
  const size_t smem = bb_smem_bytes(c->plan_bb, nullptr);
  if (c->bb_bpsm >= 0 && smem <= c->bb_smem) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(k_solve_bb, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int bpsm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bpsm, k_solve_bb, kSolveThreads, smem);
  if (e != cudaSuccess) return e;
  if (bpsm < 1) return cudaErrorLaunchOutOfResources;
  c->bb_bpsm = bpsm;
  c->bb_smem = smem;
  return cudaSuccess;
}

cudaError_t launch_solve_bb(Ctx* c) {
  BBPlan& P = c->plan_bb;
  {
    cudaError_t e = prepare_solve_bb(c);
    if (e != cudaSuccess) return e;
  }
  int slot = 0;
  const size_t smem = bb_smem_bytes(P, &slot);
  const int num_sms = c->num_sms, max_blocks_per_sm = c->bb_bpsm;
  const SolvePlan& D = P.dense;
  // enough CTAs for the widest phase: one block column each in the assembly (its loads are a chain of L2 round trips),
  // one per segment / border keyframe / tile task
  long long want = std::max<long long>({(long long)P.n_seg, (long long)P.n_bord, (long long)D.max_upd, (long long)D.max_col,
                                        (long long)P.n_int, 1LL});
  for (int k = 0; k < P.n_lv; ++k) want = std::max<long long>(want, (long long)P.lv[k].n_int);
  if (P.n_lv > 0) want = std::max<long long>({want, (long long)P.lv[P.n_lv - 1].dense.max_upd, (long long)P.lv[P.n_lv - 1].dense.max_col});
  int G = (int)std::min<long long>(want, (long long)num_sms * std::min(max_blocks_per_sm, 1));
  if (const char* cap = getenv("SIM3BA_SOLVE_MAX_CTAS")) G = std::max(1, std::min(G, atoi(cap)));   // tests: several segments / tiles / tasks per CTA
  BBArgs a{};
  a.stamps = c->profiling ? c->solve_stamps : nullptr;
  a.blocks35 = c->blocks35; a.g = c->g; a.kf_ptr = c->kf_ptr; a.kf_edge = c->kf_edge; a.pair_ptr = c->pair_ptr; a.pair_edge = c->pair_edge;
  a.lambda = c->prm.lm_lambda;
  a.n_int = P.n_int; a.n_seg = P.n_seg; a.n_bord = P.n_bord; a.npadB = P.npadB; a.slot_doubles = slot; a.max_len = P.max_len;
  a.seg_ptr = P.seg_ptr; a.seg_bptr = P.seg_bptr; a.seg_bord = P.seg_bord; a.col_kf = P.col_kf; a.col_nb = P.col_nb; a.col_band = P.col_band;
  a.col_bpair = P.col_bpair; a.bord_kf = P.bord_kf; a.bord_sptr = P.bord_sptr; a.bord_seg = P.bord_seg; a.bord_slot = P.bord_slot;
  a.bb_pair = P.bb_pair; a.col_ofs = reinterpret_cast<const long long*>(P.col_ofs); a.col_bofs = reinterpret_cast<const long long*>(P.col_bofs);
  a.colbuf = P.colbuf; a.seg_rhs = P.seg_rhs;
  SolveArgs& B = a.B;
  B.L = P.LB; B.npad = P.npadB; B.n = 7 * P.n_bord; B.nb = P.npadB / kNB;
  B.col_ptr = D.col_ptr; B.col_rows = D.col_rows; B.row_ptr = D.row_ptr; B.row_cols = D.row_cols; B.tiles = D.tiles; B.n_tiles = D.n_tiles;
  B.rhs = P.rhsB; B.ysol = P.ysolB; B.Dinv = P.DinvB; B.tau = P.tauB;
  B.eps0 = c->prm.eps0; B.max_attempts = c->prm.max_attempts; B.status = c->fail_flag; B.eps_used = c->d_eps_used; B.bar = c->bar;
  a.tau = c->tau; a.fixed = c->fixed_mask; a.N = c->N;
  a.eps0 = c->prm.eps0; a.max_attempts = c->prm.max_attempts; a.status = c->fail_flag; a.eps_used = c->d_eps_used; a.bar = c->bar;
  BBLevels L{};
  L.n = P.n_lv;
  for (int k = 0; k < P.n_lv; ++k) {
    const BBLevel2& Q = P.lv[k];
    BBArgs& a2 = L.lv[k];
    a2.n_int = Q.n_int; a2.n_seg = Q.n_seg; a2.n_bord = Q.n_bord; a2.npadB = Q.npadB; a2.slot_doubles = slot; a2.max_len = Q.max_len;
    a2.seg_ptr = Q.seg_ptr; a2.seg_bptr = Q.seg_bptr; a2.seg_bord = Q.seg_bord; a2.col_kf = Q.col_kf; a2.col_nb = Q.col_nb;
    a2.bord_kf = Q.bord_kf; a2.bord_sptr = Q.bord_sptr; a2.bord_seg = Q.bord_seg; a2.bord_slot = Q.bord_slot;
    a2.col_ofs = reinterpret_cast<const long long*>(Q.col_ofs); a2.colbuf = Q.colbuf; a2.seg_rhs = Q.seg_rhs;
    SolveArgs& B2 = a2.B;
    const SolvePlan& D2 = Q.dense;                            // filled for the last level only: the others are never solved densely
    B2.L = Q.LB; B2.npad = Q.npadB; B2.n = 7 * Q.n_bord; B2.nb = Q.npadB / kNB;
    B2.col_ptr = D2.col_ptr; B2.col_rows = D2.col_rows; B2.row_ptr = D2.row_ptr; B2.row_cols = D2.row_cols; B2.tiles = D2.tiles; B2.n_tiles = D2.n_tiles;
    B2.rhs = Q.rhsB; B2.ysol = Q.ysolB; B2.Dinv = Q.DinvB; B2.tau = Q.tauB;
    B2.eps0 = c->prm.eps0; B2.max_attempts = c->prm.max_attempts; B2.status = c->fail_flag; B2.eps_used = c->d_eps_used; B2.bar = c->bar;
    a2.tau = (k > 0) ? P.lv[k - 1].tauB : P.tauB;             // the columns of a level are border keyframes of the level before
    a2.N = (k > 0) ? P.lv[k - 1].n_bord : P.n_bord;
    a2.eps0 = c->prm.eps0; a2.max_attempts = c->prm.max_attempts; a2.status = c->fail_flag; a2.eps_used = c->d_eps_used; a2.bar = c->bar;
  }
  cudaError_t e = cudaMemsetAsync(c->bar, 0, sizeof(unsigned int), c->stream);
  if (e != cudaSuccess) return e;
  if (c->profiling) {
    cudaMemsetAsync(c->solve_stamps, 0, 16 * sizeof(unsigned long long), c->stream);
    cudaEventRecord(c->ev[4], c->stream);
  }
  void* args[] = {&a, &L};
  e = cudaLaunchCooperativeKernel((const void*)k_solve_bb, dim3(G), dim3(kSolveThreads), args, smem, c->stream);
  c->launches += 1;
  c->last_solve_grid = G;
  return e;
}

}  // namespace sim3ba
