// a0 (host): symbolic tile-level Cholesky of the keyframe graph.  The 7x7 blocks of H sit on the
// 64x64 tile grid of the padded 7N system; a tile of L is non-zero if it holds a block of H or is
// created by fill-in.  Fill is computed exactly at tile level with the elimination-tree recurrence
// struct(L_{*p}) >= struct(L_{*k}) \ {p}, p = min struct(L_{*k}) (keyframes stay in their natural,
// i.e. temporal, order: loop closures and inter-agent links then cost a few dense tile rows instead
// of a dense band).  Integer bookkeeping only.
#include <algorithm>

#include "sim3ba_internal.cuh"

namespace sim3ba {

namespace {
template <class T>
cudaError_t up(T** dst, const std::vector<T>& src, cudaStream_t s) {
  cudaError_t e = dmalloc(reinterpret_cast<void**>(dst), std::max<size_t>(src.size(), 1) * sizeof(T));
  if (e != cudaSuccess || src.empty()) return e;
  return cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s);
}
}  // namespace

void free_plan(SolvePlan& p) {
  dfree(p.col_ptr); dfree(p.col_rows); dfree(p.row_ptr); dfree(p.row_cols); dfree(p.tiles);
  p = SolvePlan();
}

namespace {
// column lists (rows i > k with a non-zero tile (i, k)) -> row lists, tile list, flop count; upload
bool finish_plan(int nb, const std::vector<std::vector<int32_t>>& col, SolvePlan& plan, cudaStream_t stream, std::string& err) {
  plan.nb = nb;
  plan.h_col_ptr.assign(nb + 1, 0);
  plan.h_col_rows.clear();
  std::vector<std::vector<int32_t>> row(nb);
  plan.max_col = plan.max_row = plan.max_upd = 0;
  const double t3 = (double)kNB * kNB * kNB;
  plan.flops = 0.0;
  for (int k = 0; k < nb; ++k) {
    for (int32_t i : col[k]) { plan.h_col_rows.push_back(i); row[i].push_back(k); }
    plan.h_col_ptr[k + 1] = (int32_t)plan.h_col_rows.size();
    const int ck = (int)col[k].size();
    plan.max_col = std::max(plan.max_col, ck);
    plan.max_upd = std::max(plan.max_upd, ck * (ck + 1) / 2);
    plan.flops += t3 / 3.0 + ck * t3 + (double)ck * (ck + 1) / 2 * 2.0 * t3 + 4.0 * ck * kNB * kNB + 2.0 * kNB * kNB;
  }
  plan.n_off = (int)plan.h_col_rows.size();
  plan.h_row_ptr.assign(nb + 1, 0);
  plan.h_row_cols.clear();
  plan.h_tiles.clear();
  for (int k = 0; k < nb; ++k) {
    for (int32_t j : row[k]) { plan.h_row_cols.push_back(j); plan.h_tiles.push_back(k); plan.h_tiles.push_back(j); }
    plan.h_tiles.push_back(k); plan.h_tiles.push_back(k);
    plan.h_row_ptr[k + 1] = (int32_t)plan.h_row_cols.size();
    plan.max_row = std::max(plan.max_row, (int)row[k].size());
  }
  plan.n_tiles = (int)plan.h_tiles.size() / 2;
  cudaError_t e;
  if ((e = up(&plan.col_ptr, plan.h_col_ptr, stream)) != cudaSuccess || (e = up(&plan.col_rows, plan.h_col_rows, stream)) != cudaSuccess ||
      (e = up(&plan.row_ptr, plan.h_row_ptr, stream)) != cudaSuccess || (e = up(&plan.row_cols, plan.h_row_cols, stream)) != cudaSuccess ||
      (e = up(&plan.tiles, plan.h_tiles, stream)) != cudaSuccess || (e = cudaStreamSynchronize(stream)) != cudaSuccess) {
    err = std::string("build_plan: ") + cudaGetErrorString(e);
    return false;
  }
  plan.ready = true;
  return true;
}

}  // namespace

bool build_plan(Ctx* c, bool dense, SolvePlan& plan, std::string& err) {
  const int nb = c->npad / kNB;
  std::vector<std::vector<int32_t>> col(nb);
  if (dense) {
    for (int k = 0; k < nb; ++k)
      for (int i = k + 1; i < nb; ++i) col[k].push_back(i);
  } else {
    auto add = [&](int ti, int tj) { if (ti > tj) col[tj].push_back(ti); };
    for (int k = 0; k < c->N; ++k) {                       // a diagonal block may straddle two tiles
      if (c->h_fixed[k]) continue;
      add((7 * k + 6) / kNB, (7 * k) / kNB);
    }
    const int P = (int)c->h_pair_kf.size() / 2;
    for (int p = 0; p < P; ++p) {
      const int hi = c->h_pair_kf[2 * p], lo = c->h_pair_kf[2 * p + 1];
      if (c->h_fixed[hi] || c->h_fixed[lo]) continue;
      for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) add((7 * hi + 6 * a) / kNB, (7 * lo + 6 * b) / kNB);
    }
    for (int k = 0; k < nb; ++k) {                         // symbolic factorisation (fill-in)
      auto& v = col[k];
      std::sort(v.begin(), v.end());
      v.erase(std::unique(v.begin(), v.end()), v.end());
      if (v.size() > 1) col[v[0]].insert(col[v[0]].end(), v.begin() + 1, v.end());
    }
  }
  return finish_plan(nb, col, plan, c->stream, err);
}

bool build_dense_plan(int nb, SolvePlan& plan, cudaStream_t stream, std::string& err) {
  std::vector<std::vector<int32_t>> col(nb);
  for (int k = 0; k < nb; ++k)
    for (int i = k + 1; i < nb; ++i) col[k].push_back(i);
  return finish_plan(nb, col, plan, stream, err);
}

}  // namespace sim3ba
