// a0 (host): band + border analysis of the keyframe graph for the block (7x7) Cholesky of a7
// (solver mode 2; layout and roles in sim3ba_internal.cuh, kernel in k_solve_bb.cu).
//
// The Sim(3) graph of PAPER.md:108 is, per agent, a temporal chain (edges (k, k+1..k+3)) plus a few
// long links: loop closures and inter-agent edges.  One endpoint of every long link becomes a BORDER
// keyframe (greedy vertex cover, the endpoint with more long links first); a chain longer than
// `lmax` (about 2 sqrt(N)) interior keyframes is cut by making the next kBand keyframes border as well (substructuring:
// the pieces are then independent and are eliminated in parallel).  Integer bookkeeping only.
#include <math.h>
#include <stdlib.h>

#include <algorithm>
#include <utility>

#include "sim3ba_internal.cuh"

namespace sim3ba {

namespace {
template <class T>
cudaError_t up(T** dst, const std::vector<T>& src, cudaStream_t s) {
  cudaError_t e = dmalloc(reinterpret_cast<void**>(dst), std::max<size_t>(src.size(), 1) * sizeof(T));
  if (e != cudaSuccess || src.empty()) return e;
  return cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s);
}
template <class T>
cudaError_t dalloc(T** p, size_t count) {
  return dmalloc(reinterpret_cast<void**>(p), std::max<size_t>(count, 1) * sizeof(T));
}
}  // namespace

void free_bb_plan(BBPlan& p) {
  dfree(p.seg_ptr); dfree(p.seg_bptr); dfree(p.seg_bord); dfree(p.col_kf); dfree(p.col_nb); dfree(p.col_ofs);
  dfree(p.col_band); dfree(p.col_bpair); dfree(p.col_bofs); dfree(p.bord_kf); dfree(p.bord_sptr);
  dfree(p.bord_seg); dfree(p.bord_slot); dfree(p.bb_pair); dfree(p.colbuf); dfree(p.seg_rhs);
  dfree(p.LB); dfree(p.rhsB); dfree(p.ysolB); dfree(p.DinvB); dfree(p.tauB);
  free_plan(p.dense);
  for (BBLevel2& q : p.lv) {
    dfree(q.seg_ptr); dfree(q.seg_bptr); dfree(q.seg_bord); dfree(q.col_kf); dfree(q.col_nb); dfree(q.bord_kf);
    dfree(q.bord_sptr); dfree(q.bord_seg); dfree(q.bord_slot); dfree(q.col_ofs);
    dfree(q.colbuf); dfree(q.seg_rhs); dfree(q.LB); dfree(q.rhsB); dfree(q.ysolB); dfree(q.DinvB); dfree(q.tauB);
    free_plan(q.dense);
  }
  p = BBPlan();
}

bool build_bb_plan(Ctx* c, std::string& err, int lmax_hint) {
  BBPlan& P = c->plan_bb;
  P.ready = true;
  P.valid = false;
  const int N = c->N;
  const int n_pairs = (int)c->h_pair_kf.size() / 2;
  // Longest segment.  A segment costs ~1.4 us per keyframe, sequentially; every cut adds kBand keyframes to the border
  // system, of which the further levels (below) take most out again before the dense solve at ~32 us per 64 rows: the two
  // balance near lmax ~ 0.9 sqrt(free keyframes) (measured on the BASELINE graphs, flat around the optimum: 200 keyframes
  // 12-28, 1000 16-36, 2000 28-56; it was 2 sqrt before the levels existed).  SIM3BA_BB_LMAX overrides (tests,
  // experiments); lmax_hint is this function calling itself with longer segments after too many border keyframes.
  int n_free = 0;
  for (int k = 0; k < N; ++k) n_free += c->h_fixed[k] ? 0 : 1;
  int lmax = std::max(12, std::min(160, (int)(0.9 * sqrt((double)n_free) + 0.5)));
  if (lmax_hint > 0) lmax = lmax_hint;
  const char* lmax_env = getenv("SIM3BA_BB_LMAX");
  if (lmax_env) lmax = std::max(4, atoi(lmax_env));

  enum { FIXED = 0, INTERIOR = 1, BORDER = 2 };
  std::vector<int> role(N, INTERIOR);
  for (int k = 0; k < N; ++k) if (c->h_fixed[k]) role[k] = FIXED;
  // adjacency over the pairs with both endpoints free
  std::vector<std::vector<std::pair<int32_t, int32_t>>> adj(N);   // (other keyframe, pair index)
  std::vector<int> longdeg(N, 0);
  for (int p = 0; p < n_pairs; ++p) {
    const int hi = c->h_pair_kf[2 * p], lo = c->h_pair_kf[2 * p + 1];
    if (role[hi] == FIXED || role[lo] == FIXED) continue;
    adj[hi].push_back({lo, p});
    adj[lo].push_back({hi, p});
    if (hi - lo > kBand) { ++longdeg[hi]; ++longdeg[lo]; }
  }
  // vertex cover of the long links (pairs are sorted by (hi, lo))
  for (int p = 0; p < n_pairs; ++p) {
    const int hi = c->h_pair_kf[2 * p], lo = c->h_pair_kf[2 * p + 1];
    if (role[hi] == FIXED || role[lo] == FIXED || hi - lo <= kBand) continue;
    if (role[hi] == BORDER || role[lo] == BORDER) continue;
    role[longdeg[lo] > longdeg[hi] ? lo : hi] = BORDER;
  }
  // segments: runs of interior keyframes in index order; natural cut where no band pair reaches on; forced
  // cut after lmax keyframes by turning the interior keyframes of the next kBand indices into border
  std::vector<int32_t> col_kf, seg_ptr(1, 0);
  std::vector<int> sep_group(N, -1);                          // cut c of the chains -> its <= kBand separator keyframes
  int n_groups = 0;
  {
    int reach = -1, run = 0, sep_until = -1;
    for (int u = 0; u < N; ++u) {
      if (role[u] != INTERIOR) continue;
      if (u <= sep_until) { role[u] = BORDER; sep_group[u] = n_groups - 1; continue; }
      if (run > 0 && reach < u) { seg_ptr.push_back((int32_t)col_kf.size()); run = 0; }
      col_kf.push_back(u);
      ++run;
      for (auto& nb : adj[u])
        if (nb.first > u && nb.first - u <= kBand && role[nb.first] == INTERIOR) reach = std::max(reach, (int)nb.first);
      if (run >= lmax && reach > u) {   // the chain goes on: cut it
        sep_until = u + kBand;
        ++n_groups;
        seg_ptr.push_back((int32_t)col_kf.size());
        run = 0;
        reach = -1;
      }
    }
    if (run > 0) seg_ptr.push_back((int32_t)col_kf.size());
  }
  const int n_int = (int)col_kf.size(), n_seg = (int)seg_ptr.size() - 1;
  std::vector<int32_t> bord_kf, bidx(N, -1), seg_of(N, -1), pos_of(N, -1);
  for (int k = 0; k < N; ++k) if (role[k] == BORDER) { bidx[k] = (int32_t)bord_kf.size(); bord_kf.push_back(k); }
  const int n_bord = (int)bord_kf.size();
  for (int s = 0; s < n_seg; ++s)
    for (int q = seg_ptr[s]; q < seg_ptr[s + 1]; ++q) { seg_of[col_kf[q]] = s; pos_of[col_kf[q]] = q; }

  // border keyframes of every segment; structure checks
  std::vector<int32_t> seg_bptr(1, 0), seg_bord;
  int max_nb = 0, max_len = 0;
  for (int s = 0; s < n_seg; ++s) {
    std::vector<int32_t> b;
    for (int q = seg_ptr[s]; q < seg_ptr[s + 1]; ++q)
      for (auto& nb : adj[col_kf[q]]) {
        const int v = nb.first;
        if (role[v] == BORDER) b.push_back(bidx[v]);
        else if (seg_of[v] != s || std::abs(pos_of[v] - q) > kBand) return true;   // not band + border: plan not used
      }
    std::sort(b.begin(), b.end());
    b.erase(std::unique(b.begin(), b.end()), b.end());
    max_nb = std::max(max_nb, (int)b.size());
    max_len = std::max(max_len, seg_ptr[s + 1] - seg_ptr[s]);
    seg_bord.insert(seg_bord.end(), b.begin(), b.end());
    seg_bptr.push_back((int32_t)seg_bord.size());
  }
  if (7 * n_bord > 2048 && !lmax_env && lmax < 640) return build_bb_plan(c, err, 2 * lmax);   // fewer, longer segments
  if (max_nb > kMaxSegBorder || 7 * n_bord > 2048) return true;   // too much border: the tile plan is the better tool

  // per-column block sources
  std::vector<int64_t> col_ofs(n_int), col_bofs(n_int);
  std::vector<int32_t> col_nb(n_int, 0);
  std::vector<int32_t> col_band((size_t)n_int * kBand, -1), col_bpair;
  size_t ofs = 0;
  for (int s = 0; s < n_seg; ++s) {
    const int nb = seg_bptr[s + 1] - seg_bptr[s];
    for (int q = seg_ptr[s]; q < seg_ptr[s + 1]; ++q) {
      const int u = col_kf[q];
      col_ofs[q] = (int64_t)ofs;
      col_nb[q] = nb;
      ofs += ((size_t)(1 + kBand + nb) * 49 + 7 + 1) & ~(size_t)1;   // 16-byte granules
      col_bofs[q] = (int64_t)col_bpair.size();
      col_bpair.resize(col_bpair.size() + nb, -1);
      for (auto& a : adj[u]) {
        const int v = a.first;
        if (role[v] == BORDER) {
          const int slot = (int)(std::lower_bound(seg_bord.begin() + seg_bptr[s], seg_bord.begin() + seg_bptr[s + 1], bidx[v]) -
                                 (seg_bord.begin() + seg_bptr[s]));
          col_bpair[(size_t)col_bofs[q] + slot] = a.second;
        } else if (pos_of[v] > q) {
          col_band[(size_t)q * kBand + (pos_of[v] - q - 1)] = a.second;
        }
      }
    }
  }
  // border side: segments touching a border keyframe, border-border pairs
  std::vector<int32_t> bord_sptr(n_bord + 1, 0), bord_seg, bord_slot, bb_pair((size_t)n_bord * n_bord, -1);
  {
    std::vector<std::vector<std::pair<int32_t, int32_t>>> touch(n_bord);
    for (int s = 0; s < n_seg; ++s)
      for (int q = seg_bptr[s]; q < seg_bptr[s + 1]; ++q) touch[seg_bord[q]].push_back({s, q - seg_bptr[s]});
    for (int b = 0; b < n_bord; ++b) {
      for (auto& t : touch[b]) { bord_seg.push_back(t.first); bord_slot.push_back(t.second); }
      bord_sptr[b + 1] = (int32_t)bord_seg.size();
    }
    for (int b = 0; b < n_bord; ++b)
      for (auto& a : adj[bord_kf[b]])
        if (role[a.first] == BORDER && a.first < bord_kf[b]) bb_pair[(size_t)b * n_bord + bidx[a.first]] = a.second;
  }

  // flop count of the plan itself (FMA = 2), at 7x7 granularity: per interior column with B = band + border blocks below
  // the diagonal -- POTRF 7^3/3, TRSM of 7 B + 1 rows (49 each), trailing update B (B + 1) / 2 block products (2 * 7^3) plus
  // the right-hand side (B * 2 * 49; the border x border part of it is the Schur complement), back-substitution
  // (B + 1) * 2 * 49 -- and the dense Cholesky + two triangular solves of the border system
  double flops = 0.0;
  for (int s = 0; s < n_seg; ++s) {
    const int nb = seg_bptr[s + 1] - seg_bptr[s], len = seg_ptr[s + 1] - seg_ptr[s];
    for (int q = 0; q < len; ++q) {
      const double B = (double)std::min(kBand, len - 1 - q) + nb;
      flops += 343.0 / 3.0 + (7.0 * B + 1.0) * 49.0 + B * (B + 1.0) / 2.0 * 686.0 + B * 98.0 + (B + 1.0) * 98.0;
    }
  }
  {
    const double nB = 7.0 * n_bord;
    flops += nB * nB * nB / 3.0 + 2.0 * nB * nB;
  }
  P.flops = flops;
  P.n_int = n_int; P.n_seg = n_seg; P.n_bord = n_bord; P.max_nb = max_nb; P.max_len = max_len;
  P.npadB = (7 * n_bord + kNB - 1) / kNB * kNB;
  P.col_doubles = ofs;
  P.h_seg_ptr = seg_ptr; P.h_seg_bptr = seg_bptr;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; return e == cudaSuccess; };
  ok(up(&P.seg_ptr, seg_ptr, c->stream)); ok(up(&P.seg_bptr, seg_bptr, c->stream)); ok(up(&P.seg_bord, seg_bord, c->stream));
  ok(up(&P.col_kf, col_kf, c->stream)); ok(up(&P.col_nb, col_nb, c->stream)); ok(up(&P.col_ofs, col_ofs, c->stream)); ok(up(&P.col_band, col_band, c->stream));
  ok(up(&P.col_bpair, col_bpair, c->stream)); ok(up(&P.col_bofs, col_bofs, c->stream)); ok(up(&P.bord_kf, bord_kf, c->stream));
  ok(up(&P.bord_sptr, bord_sptr, c->stream)); ok(up(&P.bord_seg, bord_seg, c->stream)); ok(up(&P.bord_slot, bord_slot, c->stream));
  ok(up(&P.bb_pair, bb_pair, c->stream));
  ok(dalloc(&P.colbuf, ofs)); ok(dalloc(&P.seg_rhs, seg_bord.size() * 7));
  const size_t nB = (size_t)P.npadB;
  ok(dalloc(&P.LB, nB * nB)); ok(dalloc(&P.rhsB, nB)); ok(dalloc(&P.ysolB, nB)); ok(dalloc(&P.DinvB, nB)); ok(dalloc(&P.tauB, nB));
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);   // the host vectors go out of scope
  if (e != cudaSuccess) { err = std::string("build_bb_plan: ") + cudaGetErrorString(e); return false; }
  if (P.npadB > 0 && !build_dense_plan(P.npadB / kNB, P.dense, c->stream, err)) return false;
  P.valid = true;

  // ---- further levels: independent sets of separator groups are eliminated from S before the dense solve ----
  // A level is used where it removes at least two 64-row tile columns from the dense system (a tile column costs ~32 us,
  // the four extra phases and barriers of a level ~45 us).  SIM3BA_BB_LEVELS = 1 switches the levels off, = 2 forces
  // one wherever a group can be eliminated (tests).
  const char* lvs = getenv("SIM3BA_BB_LEVELS");
  const int lv_mode = lvs ? atoi(lvs) : 0;
  if (n_groups == 0 || n_bord == 0 || lv_mode == 1) return true;
  // state of the current level: its border keyframes 0 .. cur_n - 1, their coupling in the current S, their group
  int cur_n = n_bord, cur_npad = P.npadB;
  std::vector<std::vector<int32_t>> adjS(n_bord);              // coupling in S: same segment, or a direct pair
  for (int s = 0; s < n_seg; ++s)
    for (int x = seg_bptr[s]; x < seg_bptr[s + 1]; ++x)
      for (int y = seg_bptr[s]; y < seg_bptr[s + 1]; ++y)
        if (x != y) adjS[seg_bord[x]].push_back(seg_bord[y]);
  for (int b = 0; b < n_bord; ++b)
    for (int b2 = 0; b2 < b; ++b2)
      if (bb_pair[(size_t)b * n_bord + b2] >= 0) { adjS[b].push_back(b2); adjS[b2].push_back(b); }
  std::vector<int> grp_of(n_bord, -1);
  for (int b = 0; b < n_bord; ++b) grp_of[b] = sep_group[bord_kf[b]];
  for (int level = 0; level < BBPlan::kMaxLevels; ++level) {
    for (auto& v : adjS) { std::sort(v.begin(), v.end()); v.erase(std::unique(v.begin(), v.end()), v.end()); }
    std::vector<std::vector<int32_t>> grp(n_groups);          // members of a group as current border indices, ascending
    for (int b = 0; b < cur_n; ++b) if (grp_of[b] >= 0) grp[grp_of[b]].push_back(b);
    std::vector<char> picked(n_groups, 0);
    for (int gI = 0; gI < n_groups; ++gI) {                   // greedy independent set, in chain order
      if (grp[gI].empty()) continue;
      bool free_of_picked = true;
      std::vector<int32_t> ext;
      for (int32_t b : grp[gI])
        for (int32_t v : adjS[b]) {
          if (grp_of[v] == gI) continue;
          if (grp_of[v] >= 0 && picked[grp_of[v]]) free_of_picked = false;
          ext.push_back(v);
        }
      std::sort(ext.begin(), ext.end());
      ext.erase(std::unique(ext.begin(), ext.end()), ext.end());
      if (free_of_picked && (int)ext.size() <= kMaxSegBorder) picked[gI] = 1;
    }
    std::vector<int32_t> l2_bord_kf, b2idx(cur_n, -1), l2_col_kf, l2_seg_ptr(1, 0);
    for (int b = 0; b < cur_n; ++b)
      if (!(grp_of[b] >= 0 && picked[grp_of[b]])) { b2idx[b] = (int32_t)l2_bord_kf.size(); l2_bord_kf.push_back(b); }
    for (int gI = 0; gI < n_groups; ++gI)
      if (picked[gI]) { for (int32_t b : grp[gI]) l2_col_kf.push_back(b); l2_seg_ptr.push_back((int32_t)l2_col_kf.size()); }
    const int n_int2 = (int)l2_col_kf.size(), n_seg2 = (int)l2_seg_ptr.size() - 1, n_bord2 = (int)l2_bord_kf.size();
    const int npadB2 = (7 * n_bord2 + kNB - 1) / kNB * kNB;
    if (n_seg2 == 0 || (lv_mode != 2 && npadB2 + kNB >= cur_npad) || (lv_mode == 2 && level > 0 && npadB2 >= cur_npad)) break;
    BBLevel2& Q = P.lv[level];
    std::vector<int32_t> l2_seg_bptr(1, 0), l2_seg_bord, l2_col_nb(n_int2, 0);
    std::vector<int64_t> l2_col_ofs(n_int2);
    std::vector<std::vector<int32_t>> seg_ext(n_seg2);       // external neighbours of a group, as current border indices
    int max_nb2 = 0, max_len2 = 0;
    size_t ofs2 = 0;
    for (int s = 0; s < n_seg2; ++s) {
      std::vector<int32_t> ext;
      for (int q = l2_seg_ptr[s]; q < l2_seg_ptr[s + 1]; ++q)
        for (int32_t v : adjS[l2_col_kf[q]])
          if (b2idx[v] >= 0) { ext.push_back(b2idx[v]); seg_ext[s].push_back(v); }
      std::sort(ext.begin(), ext.end());
      ext.erase(std::unique(ext.begin(), ext.end()), ext.end());
      std::sort(seg_ext[s].begin(), seg_ext[s].end());
      seg_ext[s].erase(std::unique(seg_ext[s].begin(), seg_ext[s].end()), seg_ext[s].end());
      const int nb = (int)ext.size();
      max_nb2 = std::max(max_nb2, nb);
      max_len2 = std::max(max_len2, l2_seg_ptr[s + 1] - l2_seg_ptr[s]);
      l2_seg_bord.insert(l2_seg_bord.end(), ext.begin(), ext.end());
      l2_seg_bptr.push_back((int32_t)l2_seg_bord.size());
      for (int q = l2_seg_ptr[s]; q < l2_seg_ptr[s + 1]; ++q) {
        l2_col_nb[q] = nb;
        l2_col_ofs[q] = (int64_t)ofs2;
        ofs2 += ((size_t)(1 + kBand + nb) * 49 + 7 + 1) & ~(size_t)1;
      }
    }
    std::vector<int32_t> l2_bord_sptr(n_bord2 + 1, 0), l2_bord_seg, l2_bord_slot;
    {
      std::vector<std::vector<std::pair<int32_t, int32_t>>> touch(n_bord2);
      for (int s = 0; s < n_seg2; ++s)
        for (int q = l2_seg_bptr[s]; q < l2_seg_bptr[s + 1]; ++q) touch[l2_seg_bord[q]].push_back({s, q - l2_seg_bptr[s]});
      for (int b = 0; b < n_bord2; ++b) {
        for (auto& t : touch[b]) { l2_bord_seg.push_back(t.first); l2_bord_slot.push_back(t.second); }
        l2_bord_sptr[b + 1] = (int32_t)l2_bord_seg.size();
      }
    }
    Q.n_int = n_int2; Q.n_seg = n_seg2; Q.n_bord = n_bord2; Q.max_nb = max_nb2; Q.max_len = max_len2; Q.npadB = npadB2;
    ok(up(&Q.seg_ptr, l2_seg_ptr, c->stream)); ok(up(&Q.seg_bptr, l2_seg_bptr, c->stream)); ok(up(&Q.seg_bord, l2_seg_bord, c->stream));
    ok(up(&Q.col_kf, l2_col_kf, c->stream)); ok(up(&Q.col_nb, l2_col_nb, c->stream)); ok(up(&Q.col_ofs, l2_col_ofs, c->stream));
    ok(up(&Q.bord_kf, l2_bord_kf, c->stream)); ok(up(&Q.bord_sptr, l2_bord_sptr, c->stream)); ok(up(&Q.bord_seg, l2_bord_seg, c->stream));
    ok(up(&Q.bord_slot, l2_bord_slot, c->stream));
    ok(dalloc(&Q.colbuf, ofs2)); ok(dalloc(&Q.seg_rhs, l2_seg_bord.size() * 7));
    const size_t nB2 = (size_t)npadB2;
    ok(dalloc(&Q.LB, nB2 * nB2)); ok(dalloc(&Q.rhsB, nB2)); ok(dalloc(&Q.ysolB, nB2)); ok(dalloc(&Q.DinvB, nB2)); ok(dalloc(&Q.tauB, nB2));
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);   // the host vectors go out of scope
    if (e != cudaSuccess) { err = std::string("build_bb_plan (further level): ") + cudaGetErrorString(e); return false; }
    {   // flop count: the dense system shrinks, the groups are eliminated at 7x7 granularity
      const double nB1 = 7.0 * cur_n, nBn = 7.0 * n_bord2;
      double f2 = nBn * nBn * nBn / 3.0 + 2.0 * nBn * nBn;
      for (int s = 0; s < n_seg2; ++s) {
        const int nb = l2_seg_bptr[s + 1] - l2_seg_bptr[s], len = l2_seg_ptr[s + 1] - l2_seg_ptr[s];
        for (int q = 0; q < len; ++q) {
          const double B = (double)std::min(kBand, len - 1 - q) + nb;
          f2 += 343.0 / 3.0 + (7.0 * B + 1.0) * 49.0 + B * (B + 1.0) / 2.0 * 686.0 + B * 98.0 + (B + 1.0) * 98.0;
        }
      }
      Q.flops_saved = (nB1 * nB1 * nB1 / 3.0 + 2.0 * nB1 * nB1) - f2;
      P.flops -= Q.flops_saved;
    }
    Q.valid = true;
    P.n_lv = level + 1;
    // the next level sees the keyframes that stayed; eliminating a group couples all its neighbours with one another (fill)
    std::vector<std::vector<int32_t>> adj_next(n_bord2);
    std::vector<int> grp_next(n_bord2, -1);
    for (int b = 0; b < cur_n; ++b) {
      if (b2idx[b] < 0) continue;
      grp_next[b2idx[b]] = grp_of[b];
      for (int32_t v : adjS[b]) if (b2idx[v] >= 0) adj_next[b2idx[b]].push_back(b2idx[v]);
    }
    for (int s = 0; s < n_seg2; ++s)
      for (int32_t x : seg_ext[s])
        for (int32_t y : seg_ext[s])
          if (x != y) adj_next[b2idx[x]].push_back(b2idx[y]);
    adjS.swap(adj_next);
    grp_of.swap(grp_next);
    cur_n = n_bord2;
    cur_npad = npadB2;
  }
  if (P.n_lv > 0) {
    BBLevel2& last = P.lv[P.n_lv - 1];
    if (last.npadB > 0 && !build_dense_plan(last.npadB / kNB, last.dense, c->stream, err)) return false;
  }
  return true;
}

}  // namespace sim3ba
