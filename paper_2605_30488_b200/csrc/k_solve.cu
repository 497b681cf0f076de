// Kernels 3+4 of the Sim(3) GN step: damped tile assembly (a6) and ONE persistent cooperative kernel
// for the blocked FP64 Cholesky, the forward and backward triangular solves (a7) and the epsilon
// escalation of PAPER.md:122 -- all on the device, no host round trip between attempts.
//
//   Eq. (7)  PAPER.md:120   (H + lambda diag(H) + eps_r I) tau = -g
//   PAPER.md:122            eps_r = eps0 * 100^r on factorisation failure, r < max_attempts, else tau = 0
//
// Layout: L is npad x npad row-major (npad multiple of NB = 64, identity padding), lower triangle,
// addressed in 64x64 tiles.  The kernel walks the tile plan built at create (solve_plan.cu): only the
// non-zero tiles of L (fill included) are assembled, factorised and used; the dense plan lists all.
// Right-looking, per block column k:
//   phase A  every CTA that owns a tile (i, k) re-factorises the diagonal tile L_kk in shared memory
//            (redundant work instead of one more grid-wide dependency): 8-column micro-panels by one
//            warp in registers (pivots and column broadcasts by warp shuffles), rank-8 trailing
//            updates by all warps; then X L_kk^T = A_ik by the same micro-panel scheme, with the
//            right-hand side riding along as a 65th row (y_k = L_kk^-1 b_k) and b_i -= L_ik y_k.
//   phase B  trailing update C_ij -= L_ik L_jk^T over the pairs of non-zero tiles of column k, on the
//            FP64 tensor pipe (mma.sync.m8n8k4.f64 = DMMA.8x8x4).
//   back     L^T tau = y block by block, last to first, over the row lists.
// Grid-wide barriers are a monotonically increasing global counter (all CTAs are co-resident: the
// kernel is launched with cudaLaunchCooperativeKernel, with no more CTAs than the widest phase needs).
#include <stdlib.h>

#include "solve_tile.cuh"

namespace sim3ba {

namespace {

__global__ void __launch_bounds__(kSolveThreads)
k_assemble_tiles(AsmArgs a, const int32_t* __restrict__ tiles, double eps, int32_t* __restrict__ status) {
  assemble_tile(a, tiles[2 * blockIdx.x], tiles[2 * blockIdx.x + 1], eps, threadIdx.x);
  if (blockIdx.x == 0 && threadIdx.x == 0) status[0] = 0;
}

__global__ void __launch_bounds__(kSolveThreads, 2)
k_solve(SolveArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
  const int G = gridDim.x;
  unsigned int gen = 0;
  bool solved = false;
  double eps = a.eps0;
  int r = 0;
  for (; r < a.max_attempts; ++r, eps *= 100.0) {
    if (r > 0) {   // retry: damped re-assembly of the non-zero tiles (the first attempt was assembled by k_assemble_tiles)
      for (int t = blockIdx.x; t < a.n_tiles; t += G) assemble_tile(a.as, a.tiles[2 * t], a.tiles[2 * t + 1], eps, threadIdx.x);
      if (blockIdx.x == 0 && threadIdx.x == 0) a.status[0] = 0;
      grid_barrier(a.bar, G, gen);
    }
    // ---- factorisation with the forward solve riding along ----
    bool failed = false;
    for (int k = 0; k < a.nb; ++k) {
      panel_phase(a, sm, k, G);
      if (a.col_ptr[k + 1] > a.col_ptr[k]) {
        grid_barrier(a.bar, G, gen);
        if (ld_flag(a.status) != 0) { failed = true; break; }
        update_phase(a, sm, k, G);
        grid_barrier(a.bar, G, gen);
      }
    }
    if (!failed) {   // block columns without sub-diagonal tiles are factorised by CTA 0 alone
      grid_barrier(a.bar, G, gen);
      failed = ld_flag(a.status) != 0;
    }
    if (failed) {
      grid_barrier(a.bar, G, gen);   // everybody has seen the flag before it is cleared again
      continue;
    }
    // ---- backward substitution ----
    for (int kb = a.nb - 1; kb >= 0; --kb) {
      back_phase(a, sm, kb, G);
      if (a.row_ptr[kb + 1] > a.row_ptr[kb]) grid_barrier(a.bar, G, gen);
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

cudaError_t prepare_solve(Ctx* c) {
  const size_t smem = sizeof(Smem);
  if (c->solve_bpsm < 0) {
    cudaError_t e = cudaFuncSetAttribute(k_solve, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int bpsm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bpsm, k_solve, kSolveThreads, smem);
    if (e != cudaSuccess) return e;
    if (bpsm < 1) return cudaErrorLaunchOutOfResources;
    c->solve_bpsm = bpsm;
  }
  const bool dense = c->dense_loaded || c->solver_mode == 1;
  SolvePlan& plan = dense ? c->plan_dense : c->plan_sparse;
  if (!plan.ready) {
    std::string err;
    if (!build_plan(c, dense, plan, err)) { c->err = err; return cudaErrorUnknown; }
  }
  return ensure_dense(c, false, true);
}

cudaError_t launch_solve(Ctx* c) {
  const size_t smem = sizeof(Smem);
  {
    cudaError_t e = prepare_solve(c);
    if (e != cudaSuccess) return e;
  }
  const int num_sms = c->num_sms, max_blocks_per_sm = c->solve_bpsm;
  const bool dense = c->dense_loaded || c->solver_mode == 1;
  SolvePlan& plan = dense ? c->plan_dense : c->plan_sparse;
  long long want = std::max<long long>({(long long)plan.max_upd, (long long)plan.max_col, (long long)plan.max_row, 1LL});
  int G = (int)std::min<long long>(want, (long long)num_sms * std::min(max_blocks_per_sm, 2));
  if (const char* cap = getenv("SIM3BA_SOLVE_MAX_CTAS")) G = std::max(1, std::min(G, atoi(cap)));   // tests: several tiles / tasks per CTA
  SolveArgs a;
  AsmArgs& s = a.as;
  s.L = c->L; s.npad = c->npad; s.n = c->n; s.N = c->N; s.blocks35 = c->blocks35;
  s.kf_ptr = c->kf_ptr; s.kf_edge = c->kf_edge; s.pair_kf = c->pair_kf; s.pairhi_ptr = c->pairhi_ptr;
  s.pair_ptr = c->pair_ptr; s.pair_edge = c->pair_edge; s.fixed = c->fixed_mask;
  s.dense = c->dense_loaded ? c->Hd : nullptr; s.g = c->g; s.rhs = c->rhs; s.lambda = c->prm.lm_lambda;
  a.L = c->L; a.npad = c->npad; a.n = c->n; a.nb = plan.nb;
  a.col_ptr = plan.col_ptr; a.col_rows = plan.col_rows; a.row_ptr = plan.row_ptr; a.row_cols = plan.row_cols;
  a.tiles = plan.tiles; a.n_tiles = plan.n_tiles;
  a.rhs = c->rhs; a.ysol = c->ysol; a.Dinv = c->Dinv; a.tau = c->tau;
  a.eps0 = c->prm.eps0; a.max_attempts = c->prm.max_attempts;
  a.status = c->fail_flag; a.eps_used = c->d_eps_used; a.bar = c->bar;
  cudaError_t e = cudaMemsetAsync(c->bar, 0, sizeof(unsigned int), c->stream);
  if (e != cudaSuccess) return e;
  k_assemble_tiles<<<plan.n_tiles, kSolveThreads, 0, c->stream>>>(s, plan.tiles, c->prm.eps0, c->fail_flag);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (c->profiling) cudaEventRecord(c->ev[4], c->stream);
  void* args[] = {&a};
  e = cudaLaunchCooperativeKernel((const void*)k_solve, dim3(G), dim3(kSolveThreads), args, smem, c->stream);
  c->launches += 2;
  c->last_solve_grid = G;
  return e;
}

}  // namespace sim3ba
