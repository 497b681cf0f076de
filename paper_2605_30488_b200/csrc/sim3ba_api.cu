// C ABI of libsim3ba (include/sim3ba.h): argument checking, memory, a0 bookkeeping, and the
// sequencing of kernels 1-5.  Host code only; every step of the hot path runs in the kernels.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <new>
#include <numeric>
#include <utility>

#include "sim3ba_internal.cuh"

using namespace sim3ba;

namespace sim3ba {

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_pool_mutex;
cudaMemPool_t g_pools[kMaxDevices] = {};
}  // namespace

cudaError_t lib_pool(cudaMemPool_t* pool) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (!g_pools[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    e = cudaMemPoolCreate(&g_pools[dev], &props);
    if (e != cudaSuccess) { g_pools[dev] = nullptr; return e; }
    uint64_t keep = UINT64_MAX;   // freed blocks stay in the library's pool until sim3ba_release_memory
    cudaMemPoolSetAttribute(g_pools[dev], cudaMemPoolAttrReleaseThreshold, &keep);
  }
  *pool = g_pools[dev];
  return cudaSuccess;
}

// Hd (undamped dense system: sim3ba_build_system read-back, sim3ba_load_system) and L (work matrix of the tile plans,
// solver modes 0 / 1) are npad^2 doubles each -- 1.57 GB at N = 2000: allocated when first needed, never by the
// default path (sim3ba_step with the band + border plan)
cudaError_t ensure_dense(Ctx* c, bool want_Hd, bool want_L) {
  const size_t bytes = (size_t)c->npad * c->npad * sizeof(double);
  if (want_Hd && !c->Hd) {
    cudaError_t e = dmalloc(reinterpret_cast<void**>(&c->Hd), bytes);
    if (e != cudaSuccess) return e;
  }
  if (want_L && !c->L) {
    cudaError_t e = dmalloc(reinterpret_cast<void**>(&c->L), bytes);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace sim3ba

struct sim3ba_ctx {
  Ctx c;
};

namespace {

thread_local std::string g_create_error;

int fail(Ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}

int cuda_fail(Ctx* c, cudaError_t e, const char* what) {
  return fail(c, SIM3BA_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define CU(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(c, e_, #call);    \
  } while (0)

template <class T>
cudaError_t dev_alloc(T** p, size_t count) {
  return dmalloc(reinterpret_cast<void**>(p), std::max<size_t>(count, 1) * sizeof(T));
}

bool params_ok(const sim3ba_params* p) {
  return p && p->sigma_ray > 0.f && p->sigma_dist > 0.f && p->huber_k > 0.f && p->lm_lambda >= 0.0 &&
         p->eps0 >= 0.0 && p->max_attempts >= 1 && p->max_attempts <= 16 && isfinite(p->sigma_ray) &&
         isfinite(p->sigma_dist) && isfinite(p->huber_k) && isfinite(p->conf_min);
}

// a0: keyframe -> incident-edge CSR, unique unordered pairs -> edge CSR, processing order.
void build_bookkeeping(Ctx* c) {
  const int N = c->N, E = c->E;
  const std::vector<int32_t>& ed = c->h_edges;
  c->h_kf_ptr.assign(N + 1, 0);
  for (int e = 0; e < E; ++e) { ++c->h_kf_ptr[ed[2 * e] + 1]; ++c->h_kf_ptr[ed[2 * e + 1] + 1]; }
  for (int k = 0; k < N; ++k) c->h_kf_ptr[k + 1] += c->h_kf_ptr[k];
  c->h_kf_edge.assign(2 * (size_t)E, 0);
  std::vector<int32_t> cur(c->h_kf_ptr.begin(), c->h_kf_ptr.end() - 1);
  for (int e = 0; e < E; ++e) {  // ascending e inside every keyframe's list
    c->h_kf_edge[cur[ed[2 * e]]++] = e;
    c->h_kf_edge[cur[ed[2 * e + 1]]++] = e;
  }
  std::map<std::pair<int32_t, int32_t>, std::vector<int32_t>> pairs;  // key (hi, lo), sorted
  for (int e = 0; e < E; ++e) {
    const int32_t a = ed[2 * e], b = ed[2 * e + 1];
    pairs[{std::max(a, b), std::min(a, b)}].push_back(e);
  }
  c->n_pairs = (int)pairs.size();
  c->h_pair_kf.clear(); c->h_pair_ptr.assign(1, 0); c->h_pair_edge.clear();
  c->h_pairhi_ptr.assign(N + 1, 0);
  for (const auto& kv : pairs) {
    c->h_pair_kf.push_back(kv.first.first);
    c->h_pair_kf.push_back(kv.first.second);
    ++c->h_pairhi_ptr[kv.first.first + 1];
    for (int32_t e : kv.second) c->h_pair_edge.push_back(e);
    c->h_pair_ptr.push_back((int32_t)c->h_pair_edge.size());
  }
  for (int k = 0; k < N; ++k) c->h_pairhi_ptr[k + 1] += c->h_pairhi_ptr[k];
}

template <class T>
cudaError_t upload(T** dst, const std::vector<T>& src, cudaStream_t s) {
  cudaError_t e = dev_alloc(dst, src.size());
  if (e != cudaSuccess || src.empty()) return e;
  return cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s);
}

void free_all(Ctx* c) {
  dfree(c->pm); dfree(c->pm0); dfree(c->edges); dfree(c->grp_kf); dfree(c->grp_ptr); dfree(c->grp_edge); dfree(c->edgeT); dfree(c->fixed_mask); dfree(c->poses);
  dfree(c->kf_ptr); dfree(c->kf_edge); dfree(c->pair_kf); dfree(c->pair_ptr); dfree(c->pair_edge);
  dfree(c->partials); dfree(c->def_sums); dfree(c->def_masks); dfree(c->def_flag); dfree(c->blocks35); dfree(c->edge_cost); dfree(c->n_valid); dfree(c->checksum);
  dfree(c->Hd); dfree(c->L); dfree(c->g); dfree(c->rhs); dfree(c->ysol); dfree(c->Dinv); dfree(c->pairhi_ptr);
  free_plan(c->plan_sparse); free_plan(c->plan_dense); free_bb_plan(c->plan_bb);
  dfree(c->tau); dfree(c->total_cost); dfree(c->fail_flag); dfree(c->d_eps_used); dfree(c->bar); dfree(c->solve_stamps);
  if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
  if (c->h_flag) cudaFreeHost(c->h_flag);
  if (c->h_scalar) cudaFreeHost(c->h_scalar);
  for (auto& ev : c->ev) if (ev) cudaEventDestroy(ev);
}

inline void mark(Ctx* c, int i) { if (c->profiling) cudaEventRecord(c->ev[i], c->stream); }

void drop_graph(Ctx* c) {
  if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
  c->graph_exec = nullptr;
  c->graph_steps = 0;
}

// a1-a5 (+ gradient and total cost): the block-sparse system at the current poses
int build_blocks(Ctx* c) {
  mark(c, 0);
  CU(launch_accumulate(c));   // records ev[1] between kernel 1 and kernel 2 when profiling
  CU(launch_gradient(c));
  mark(c, 2);
  c->built = true; c->solved = false; c->dense_loaded = false;
  return SIM3BA_OK;
}

// a6 (damped, into L) + a7 with the escalation of PAPER.md:122: one persistent kernel, no host sync
int solve_impl(Ctx* c) {
  mark(c, 3);
  // mode 2 (default): band + border block Cholesky where the graph has that shape, else the tile-sparse plan;
  // a caller-supplied dense system (sim3ba_load_system) always takes the dense tile plan
  if (c->solver_mode == 2 && !c->dense_loaded && c->plan_bb.valid) CU(launch_solve_bb(c));
  else CU(launch_solve(c));
  mark(c, 5);
  c->solved = true;
  c->status_stale = true;
  return SIM3BA_OK;
}

// attempts / eps of the last solve live on the device until somebody asks for them
int fetch_status(Ctx* c) {
  if (!c->status_stale) return SIM3BA_OK;
  CU(cudaMemcpyAsync(c->h_flag, c->fail_flag, 4 * sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaMemcpyAsync(c->h_scalar + 1, c->d_eps_used, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  c->attempts = c->h_flag[1];
  c->eps_used = c->h_scalar[1];
  c->status_stale = false;
  return SIM3BA_OK;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

int sim3ba_default_params(sim3ba_params* p) {
  if (!p) return SIM3BA_ERR_INVALID_ARG;
  p->sigma_ray = 0.003f; p->sigma_dist = 10.0f; p->huber_k = 1.345f; p->conf_min = 0.0f;
  p->lm_lambda = 0.0; p->eps0 = 1e-6; p->max_attempts = 6; p->reserved = 0;
  return SIM3BA_OK;
}

int sim3ba_create(sim3ba_ctx** out, int32_t n_kf, int32_t height, int32_t width, int32_t n_edges,
                  const float* d_points, const float* d_conf, const int32_t* d_edges, const int32_t* d_match,
                  const int32_t* h_fixed_kf, int32_t n_fixed, const sim3ba_params* params, void* cuda_stream) {
  Ctx* c = nullptr;
  if (!out) return fail(c, SIM3BA_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (n_kf <= 0 || height <= 0 || width <= 0 || n_edges < 0 || n_fixed < 0 || (int64_t)height * width > (1 << 28) ||
      (int64_t)n_kf * 7 > (1 << 20))
    return fail(c, SIM3BA_ERR_INVALID_ARG, "non-positive or oversized dimensions");
  if (!d_points || !d_conf || (n_edges > 0 && (!d_edges || !d_match)) || (n_fixed > 0 && !h_fixed_kf))
    return fail(c, SIM3BA_ERR_INVALID_ARG, "NULL input pointer");
  if (!params_ok(params)) return fail(c, SIM3BA_ERR_INVALID_ARG, "invalid params (sigmas, kappa > 0; lambda, eps0 >= 0; 1 <= attempts <= 16)");
  int ndev = 0;
  cudaError_t de = cudaGetDeviceCount(&ndev);
  if (de != cudaSuccess || ndev == 0) return fail(c, SIM3BA_ERR_CUDA, "no CUDA device (libsim3ba has no CPU fallback)");

  tl_stream = (cudaStream_t)cuda_stream;
  sim3ba_ctx* h = new (std::nothrow) sim3ba_ctx();
  if (!h) return fail(c, SIM3BA_ERR_ALLOC, "host allocation failed");
  c = &h->c;
  c->N = n_kf; c->H = height; c->W = width; c->HW = height * width; c->E = n_edges;
  c->n = 7 * n_kf; c->npad = (c->n + kNB - 1) / kNB * kNB;
  c->chunks = (c->HW + kTilePx - 1) / kTilePx;
  c->stream = (cudaStream_t)cuda_stream;
  c->prm = *params;

  auto bail = [&](int code, const std::string& msg) {
    free_all(c);
    delete h;
    return fail(nullptr, code, msg);
  };
#define CUB(call)                                                                                 \
  do {                                                                                            \
    cudaError_t e_ = (call);                                                                      \
    if (e_ != cudaSuccess)                                                                        \
      return bail(e_ == cudaErrorMemoryAllocation ? SIM3BA_ERR_ALLOC : SIM3BA_ERR_CUDA,           \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                            \
  } while (0)

  // edge list -> host, validation (i != j, endpoints in range)
  c->h_edges.resize(2 * (size_t)n_edges);
  if (n_edges > 0) {
    CUB(cudaMemcpyAsync(c->h_edges.data(), d_edges, c->h_edges.size() * sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
    CUB(cudaStreamSynchronize(c->stream));
  }
  for (int e = 0; e < n_edges; ++e) {
    const int32_t i = c->h_edges[2 * e], j = c->h_edges[2 * e + 1];
    if (i < 0 || i >= n_kf || j < 0 || j >= n_kf || i == j)
      return bail(SIM3BA_ERR_INVALID_ARG, "edge " + std::to_string(e) + " has an endpoint out of range or i == j");
  }
  c->h_fixed.assign(n_kf, 0);
  for (int k = 0; k < n_fixed; ++k) {
    if (h_fixed_kf[k] < 0 || h_fixed_kf[k] >= n_kf) return bail(SIM3BA_ERR_INVALID_ARG, "fixed keyframe out of range");
    c->h_fixed[h_fixed_kf[k]] = 1;
  }
  build_bookkeeping(c);
  // kernel-1 schedule: edges grouped by their first endpoint i (the tile of X_i is staged once per group)
  std::vector<int32_t> grp_edge(n_edges), grp_kf, grp_ptr(1, 0);
  std::iota(grp_edge.begin(), grp_edge.end(), 0);
  std::stable_sort(grp_edge.begin(), grp_edge.end(), [&](int32_t a, int32_t b) {
    return std::make_pair(c->h_edges[2 * a], c->h_edges[2 * a + 1]) < std::make_pair(c->h_edges[2 * b], c->h_edges[2 * b + 1]);
  });
  for (int k = 0; k < n_edges; ++k) {
    const int32_t i = c->h_edges[2 * grp_edge[k]];
    if (grp_kf.empty() || grp_kf.back() != i) { grp_kf.push_back(i); if (k) grp_ptr.push_back(k); }
  }
  grp_ptr.push_back(n_edges);
  if (n_edges == 0) grp_ptr.assign(1, 0);
  c->n_groups = (int)grp_kf.size();

  const size_t NHW = (size_t)c->N * c->HW;
  {
    int dev = 0;
    CUB(cudaGetDevice(&dev));
    CUB(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev));
  }
  CUB(dev_alloc(&c->pm, NHW));
  CUB(upload(&c->edges, c->h_edges, c->stream));
  CUB(upload(&c->grp_kf, grp_kf, c->stream));
  CUB(upload(&c->grp_ptr, grp_ptr, c->stream));
  CUB(upload(&c->grp_edge, grp_edge, c->stream));
  CUB(dev_alloc(&c->edgeT, (size_t)c->E * 12));
  CUB(upload(&c->fixed_mask, c->h_fixed, c->stream));
  CUB(upload(&c->kf_ptr, c->h_kf_ptr, c->stream));
  CUB(upload(&c->kf_edge, c->h_kf_edge, c->stream));
  CUB(upload(&c->pair_kf, c->h_pair_kf, c->stream));
  CUB(upload(&c->pair_ptr, c->h_pair_ptr, c->stream));
  CUB(upload(&c->pair_edge, c->h_pair_edge, c->stream));
  CUB(upload(&c->pairhi_ptr, c->h_pairhi_ptr, c->stream));
  CUB(dev_alloc(&c->poses, (size_t)8 * c->N));
  CUB(dev_alloc(&c->partials, (size_t)c->E * c->chunks * (kAccThreads / 32) * kPartialStride));
  CUB(dev_alloc(&c->blocks35, (size_t)c->E * 35));
  CUB(dev_alloc(&c->def_sums, (size_t)c->E * 40));
  CUB(dev_alloc(&c->def_masks, (size_t)c->E * c->chunks * (kAccThreads / 32) * 32));
  CUB(dev_alloc(&c->def_flag, (size_t)c->E));
  CUB(dev_alloc(&c->edge_cost, (size_t)c->E));
  CUB(dev_alloc(&c->n_valid, (size_t)c->E));
  CUB(dev_alloc(&c->checksum, (size_t)c->E));
  CUB(dev_alloc(&c->g, (size_t)c->npad));
  CUB(dev_alloc(&c->rhs, (size_t)c->npad));
  CUB(dev_alloc(&c->ysol, (size_t)c->npad));
  CUB(dev_alloc(&c->tau, (size_t)c->npad));
  CUB(dev_alloc(&c->Dinv, (size_t)c->npad));
  CUB(dev_alloc(&c->total_cost, 1));
  CUB(dev_alloc(&c->fail_flag, 4));
  CUB(dev_alloc(&c->d_eps_used, 1));
  CUB(dev_alloc(&c->bar, 1));
  CUB(dev_alloc(&c->solve_stamps, 16));
  CUB(cudaMemsetAsync(c->solve_stamps, 0, 16 * sizeof(unsigned long long), c->stream));
  CUB(cudaMallocHost(reinterpret_cast<void**>(&c->h_flag), 4 * sizeof(int32_t)));
  CUB(cudaMallocHost(reinterpret_cast<void**>(&c->h_scalar), 4 * sizeof(double)));
  for (auto& ev : c->ev) CUB(cudaEventCreate(&ev));
  CUB(cudaMemsetAsync(c->g, 0, (size_t)c->npad * sizeof(double), c->stream));
  CUB(cudaMemsetAsync(c->tau, 0, (size_t)c->npad * sizeof(double), c->stream));
  CUB(cudaMemsetAsync(c->total_cost, 0, sizeof(double), c->stream));
  CUB(cudaMemsetAsync(c->fail_flag, 0, 4 * sizeof(int32_t), c->stream));
  {
    std::vector<double> id(8 * (size_t)c->N, 0.0);
    for (int k = 0; k < c->N; ++k) { id[8 * k + 6] = 1.0; id[8 * k + 7] = 1.0; }
    CUB(cudaMemcpyAsync(c->poses, id.data(), id.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CUB(cudaStreamSynchronize(c->stream));
  }
  c->match = d_match;
  {
    std::string perr;
    if (!build_plan(c, false, c->plan_sparse, perr)) return bail(SIM3BA_ERR_CUDA, perr);
    if (!build_bb_plan(c, perr)) return bail(SIM3BA_ERR_CUDA, perr);
  }
  CUB(launch_pack(c, d_points, d_conf));
  CUB(cudaStreamSynchronize(c->stream));
#undef CUB
  *out = h;
  return SIM3BA_OK;
}

int sim3ba_destroy(sim3ba_ctx* h) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  tl_stream = h->c.stream;
  cudaStreamSynchronize(h->c.stream);
  free_all(&h->c);
  delete h;
  return SIM3BA_OK;
}

int sim3ba_set_params(sim3ba_ctx* h, const sim3ba_params* p) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!params_ok(p)) return fail(c, SIM3BA_ERR_INVALID_ARG, "invalid params");
  if (p->conf_min != c->prm.conf_min)
    return fail(c, SIM3BA_ERR_INVALID_ARG, "conf_min is fixed at sim3ba_create (the validity mask is baked into the packed pointmap)");
  c->prm = *p;
  drop_graph(c);   // the constants are kernel arguments of the captured launches
  return SIM3BA_OK;
}

int sim3ba_set_poses(sim3ba_ctx* h, const double* d_poses) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!d_poses) return fail(c, SIM3BA_ERR_INVALID_ARG, "d_poses is NULL");
  CU(cudaMemcpyAsync(c->poses, d_poses, (size_t)8 * c->N * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  return SIM3BA_OK;
}

int sim3ba_get_poses(sim3ba_ctx* h, double* d_poses) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!d_poses) return fail(c, SIM3BA_ERR_INVALID_ARG, "d_poses is NULL");
  CU(cudaMemcpyAsync(d_poses, c->poses, (size_t)8 * c->N * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  return SIM3BA_OK;
}

int sim3ba_build_system(sim3ba_ctx* h) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  int rc = build_blocks(c);
  if (rc) return rc;
  CU(ensure_dense(c, true, false));
  CU(launch_assemble(c, c->Hd, 0.0, 0.0, false));
  mark(c, 3);
  c->hd_valid = true;
  if (c->profiling) {
    CU(cudaStreamSynchronize(c->stream));
    cudaEventElapsedTime(&c->phase_ms[0], c->ev[0], c->ev[1]);
    cudaEventElapsedTime(&c->phase_ms[1], c->ev[1], c->ev[2]);
    cudaEventElapsedTime(&c->phase_ms[2], c->ev[2], c->ev[3]);
    c->phase_ms[3] = c->phase_ms[4] = 0.f;
  }
  return SIM3BA_OK;
}

int sim3ba_solve(sim3ba_ctx* h) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!c->built && !c->dense_loaded) return fail(c, SIM3BA_ERR_BAD_STATE, "sim3ba_solve before sim3ba_build_system");
  return solve_impl(c);
}

int sim3ba_retract(sim3ba_ctx* h) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!c->solved) return fail(c, SIM3BA_ERR_BAD_STATE, "sim3ba_retract before sim3ba_solve");
  CU(launch_retract(c));
  c->built = false; c->solved = false;
  return SIM3BA_OK;
}

int sim3ba_step(sim3ba_ctx* h) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  int rc = build_blocks(c);
  if (rc) return rc;
  c->hd_valid = false;
  rc = solve_impl(c);
  if (rc) return rc;
  mark(c, 6);
  CU(launch_retract(c));
  if (c->profiling) {
    mark(c, 7);
    CU(cudaStreamSynchronize(c->stream));
    cudaEventElapsedTime(&c->phase_ms[0], c->ev[0], c->ev[1]);
    cudaEventElapsedTime(&c->phase_ms[1], c->ev[1], c->ev[2]);
    cudaEventElapsedTime(&c->phase_ms[2], c->ev[3], c->ev[4]);   // damped tile assembly
    cudaEventElapsedTime(&c->phase_ms[3], c->ev[4], c->ev[5]);   // persistent factor + solves
    cudaEventElapsedTime(&c->phase_ms[4], c->ev[6], c->ev[7]);
  }
  c->built = false; c->solved = false;
  return SIM3BA_OK;
}

int sim3ba_step_graph(sim3ba_ctx* h, int32_t n_steps) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (n_steps < 1 || n_steps > 4096) return fail(c, SIM3BA_ERR_INVALID_ARG, "n_steps must be in 1..4096");
  if (!c->graph_exec || c->graph_steps != n_steps) {
    drop_graph(c);
    // everything that is not a stream operation (function attributes, occupancy, lazily allocated buffers) first
    c->dense_loaded = false;
    CU(prepare_accumulate(c));
    if (c->solver_mode == 2 && c->plan_bb.valid) CU(prepare_solve_bb(c)); else CU(prepare_solve(c));
    const bool prof = c->profiling;
    c->profiling = false;                               // no event records inside the capture
    const int64_t l0 = c->launches;
    cudaGraph_t graph = nullptr;
    // captured on a stream of the library's own (the caller's may be the legacy default stream, which cannot be
    // captured); the launchers enqueue on c->stream, so it is swapped for the duration of the capture
    cudaStream_t user_stream = c->stream, cap = nullptr;
    cudaError_t e = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking);
    int rc = SIM3BA_OK;
    if (e == cudaSuccess) e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
      c->stream = cap;
      for (int it = 0; it < n_steps && rc == SIM3BA_OK; ++it) {
        rc = build_blocks(c);
        if (rc == SIM3BA_OK) rc = solve_impl(c);
        if (rc == SIM3BA_OK && launch_retract(c) != cudaSuccess) rc = fail(c, SIM3BA_ERR_CUDA, "launch_retract during capture");
      }
      c->stream = user_stream;
      cudaError_t e2 = cudaStreamEndCapture(cap, &graph);
      if (e2 != cudaSuccess && rc == SIM3BA_OK) e = e2;
    }
    if (cap) cudaStreamDestroy(cap);
    c->profiling = prof;
    c->graph_launches = c->launches - l0;
    c->launches = l0;
    if (rc != SIM3BA_OK) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return rc; }
    if (e != cudaSuccess || !graph) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return cuda_fail(c, e, "stream capture of the GN step"); }
    e = cudaGraphInstantiate(&c->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { c->graph_exec = nullptr; return cuda_fail(c, e, "cudaGraphInstantiate"); }
    c->graph_steps = n_steps;
  }
  CU(cudaGraphLaunch(c->graph_exec, c->stream));
  c->launches += c->graph_launches;
  c->hd_valid = false; c->built = false; c->solved = false;
  c->status_stale = true;
  return SIM3BA_OK;
}

int sim3ba_get_solve_phase_us(sim3ba_ctx* h, float us[8]) {
  if (!h || !us) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  unsigned long long st[16];
  CU(cudaMemcpyAsync(st, c->solve_stamps, sizeof(st), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  for (int k = 0; k < 8; ++k) us[k] = 0.f;
  // a phase the plan does not have (no border keyframes: no Schur rows, no border system) leaves its stamp at zero
  unsigned long long prev = st[0];
  for (int k = 0; k < 6 && st[0] != 0ull; ++k) {
    if (st[k + 1] == 0ull) continue;
    us[k] = st[k + 1] >= prev ? (float)((double)(st[k + 1] - prev) * 1e-3) : 0.f;
    prev = st[k + 1];
  }
  return SIM3BA_OK;
}

int sim3ba_probe_fp64(double* h_dfma_tflops, double* h_dmma_tflops, void* cuda_stream) {
  if (!h_dfma_tflops || !h_dmma_tflops) return SIM3BA_ERR_INVALID_ARG;
  cudaError_t e = run_probe_fp64((cudaStream_t)cuda_stream, h_dfma_tflops, h_dmma_tflops);
  return e == cudaSuccess ? SIM3BA_OK : cuda_fail(nullptr, e, "sim3ba_probe_fp64");
}

int sim3ba_release_memory(void) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return SIM3BA_ERR_CUDA;
  cudaMemPool_t pool;
  if (lib_pool(&pool) != cudaSuccess) return SIM3BA_ERR_CUDA;
  if (cudaDeviceSynchronize() != cudaSuccess) return SIM3BA_ERR_CUDA;
  return cudaMemPoolTrimTo(pool, 0) == cudaSuccess ? SIM3BA_OK : SIM3BA_ERR_CUDA;
}

int sim3ba_step_host(sim3ba_ctx* h, const double* h_in, double* h_out, double* h_cost) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  const size_t bytes = (size_t)8 * c->N * sizeof(double);
  if (h_in) CU(cudaMemcpyAsync(c->poses, h_in, bytes, cudaMemcpyHostToDevice, c->stream));
  int rc = sim3ba_step(h);
  if (rc) return rc;
  if (h_out) CU(cudaMemcpyAsync(h_out, c->poses, bytes, cudaMemcpyDeviceToHost, c->stream));
  if (h_cost) CU(cudaMemcpyAsync(h_cost, c->total_cost, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  return SIM3BA_OK;
}

namespace {

// Device copies of a host graph + a context on them: the common front part of the *_host jobs.  Everything comes from the
// library's stream-ordered pool, kept warm between jobs (no map / unmap per job).
struct HostJob {
  float *d_points = nullptr, *d_conf = nullptr;
  int32_t *d_edges = nullptr, *d_match = nullptr, *d_labels = nullptr;
  double* d_eta = nullptr;
  sim3ba_ctx* h = nullptr;
  cudaStream_t st = nullptr;
  ~HostJob() {
    if (h) sim3ba_destroy(h);                                   // synchronises the stream
    tl_stream = st;
    dfree(d_points); dfree(d_conf); dfree(d_edges); dfree(d_match); dfree(d_labels); dfree(d_eta);
  }
  // returns SIM3BA_OK or a negative status with the message in the thread-local create error
  int open(int32_t n_kf, int32_t height, int32_t width, int32_t n_edges, const float* h_points, const float* h_conf,
           const int32_t* h_edges, const int32_t* h_match, const int32_t* h_fixed_kf, int32_t n_fixed, const sim3ba_params* params,
           const double* h_poses_in, void* cuda_stream) {
    st = (cudaStream_t)cuda_stream;
    tl_stream = st;
    const size_t NHW = (size_t)n_kf * height * width, EHW = (size_t)n_edges * height * width;
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; return e == cudaSuccess; };
    ok(dmalloc(reinterpret_cast<void**>(&d_points), 3 * NHW * sizeof(float)));
    ok(dmalloc(reinterpret_cast<void**>(&d_conf), NHW * sizeof(float)));
    ok(dmalloc(reinterpret_cast<void**>(&d_edges), 2 * (size_t)n_edges * sizeof(int32_t)));
    ok(dmalloc(reinterpret_cast<void**>(&d_match), EHW * sizeof(int32_t)));
    if (e == cudaSuccess) ok(cudaMemcpyAsync(d_points, h_points, 3 * NHW * sizeof(float), cudaMemcpyHostToDevice, st));
    if (e == cudaSuccess) ok(cudaMemcpyAsync(d_conf, h_conf, NHW * sizeof(float), cudaMemcpyHostToDevice, st));
    if (e == cudaSuccess && n_edges > 0) {
      ok(cudaMemcpyAsync(d_edges, h_edges, 2 * (size_t)n_edges * sizeof(int32_t), cudaMemcpyHostToDevice, st));
      ok(cudaMemcpyAsync(d_match, h_match, EHW * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    }
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "host job: graph upload");
    int rc = sim3ba_create(&h, n_kf, height, width, n_edges, d_points, d_conf, d_edges, d_match, h_fixed_kf, n_fixed, params, cuda_stream);
    if (rc) { h = nullptr; return rc; }
    e = cudaMemcpyAsync(h->c.poses, h_poses_in, (size_t)8 * n_kf * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "host job: pose upload");
    return SIM3BA_OK;
  }
};

bool host_graph_args_ok(int32_t n_kf, int32_t height, int32_t width, int32_t n_edges, const float* h_points, const float* h_conf,
                        const int32_t* h_edges, const int32_t* h_match, const double* h_poses_in, const double* h_poses_out) {
  if (n_kf <= 0 || height <= 0 || width <= 0 || n_edges < 0 || (int64_t)height * width > (1 << 28)) return false;
  return h_points && h_conf && (n_edges == 0 || (h_edges && h_match)) && h_poses_in && h_poses_out;
}

}  // namespace

int sim3ba_optimize_host(int32_t n_kf, int32_t height, int32_t width, int32_t n_edges, const float* h_points,
                         const float* h_conf, const int32_t* h_edges, const int32_t* h_match, const int32_t* h_fixed_kf,
                         int32_t n_fixed, const sim3ba_params* params, const double* h_poses_in, int32_t n_iters,
                         double* h_poses_out, double* h_cost, void* cuda_stream) {
  if (n_iters < 0 || !host_graph_args_ok(n_kf, height, width, n_edges, h_points, h_conf, h_edges, h_match, h_poses_in, h_poses_out))
    return fail(nullptr, SIM3BA_ERR_INVALID_ARG, "NULL host pointer, or non-positive / oversized dimensions");
  HostJob job;
  int rc = job.open(n_kf, height, width, n_edges, h_points, h_conf, h_edges, h_match, h_fixed_kf, n_fixed, params, h_poses_in, cuda_stream);
  if (rc) return rc;
  Ctx* c = &job.h->c;
  cudaStream_t st = job.st;
  cudaError_t ce = cudaSuccess;
  for (int it = 0; it < n_iters && ce == cudaSuccess && rc == SIM3BA_OK; ++it) {
    rc = sim3ba_step(job.h);
    if (rc == SIM3BA_OK && h_cost) ce = cudaMemcpyAsync(h_cost + it, c->total_cost, sizeof(double), cudaMemcpyDeviceToHost, st);
  }
  if (ce == cudaSuccess && rc == SIM3BA_OK) ce = cudaMemcpyAsync(h_poses_out, c->poses, (size_t)8 * n_kf * sizeof(double), cudaMemcpyDeviceToHost, st);
  if (ce == cudaSuccess && rc == SIM3BA_OK) ce = cudaStreamSynchronize(st);
  if (rc != SIM3BA_OK) { g_create_error = c->err; return rc; }
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "sim3ba_optimize_host");
  return SIM3BA_OK;
}

int sim3ba_refine_host(int32_t n_kf, int32_t height, int32_t width, int32_t n_edges, const float* h_points, const float* h_conf,
                       const int32_t* h_edges, const int32_t* h_match, const int32_t* h_fixed_kf, int32_t n_fixed,
                       const sim3ba_params* params, const int32_t* h_labels, int32_t n_seg, const int32_t* h_pairs, const double* h_delta,
                       int32_t n_pairs, const sim3ba_depth_params* depth_params, int32_t n_rounds, int32_t n_depth_iters,
                       int32_t n_pose_iters, const double* h_poses_in, double* h_poses_out, double* h_eta, double* h_pose_cost,
                       double* h_depth_cost, void* cuda_stream) {
  if (n_rounds < 0 || n_depth_iters < 0 || n_pose_iters < 0 || !h_labels || !h_eta || !depth_params || n_seg < 1 ||
      !host_graph_args_ok(n_kf, height, width, n_edges, h_points, h_conf, h_edges, h_match, h_poses_in, h_poses_out))
    return fail(nullptr, SIM3BA_ERR_INVALID_ARG, "NULL host pointer, negative count, or non-positive / oversized dimensions");
  HostJob job;
  int rc = job.open(n_kf, height, width, n_edges, h_points, h_conf, h_edges, h_match, h_fixed_kf, n_fixed, params, h_poses_in, cuda_stream);
  if (rc) return rc;
  Ctx* c = &job.h->c;
  cudaStream_t st = job.st;
  const size_t NHW = (size_t)n_kf * height * width, M = (size_t)n_kf * n_seg;
  cudaError_t ce = dmalloc(reinterpret_cast<void**>(&job.d_labels), NHW * sizeof(int32_t));
  if (ce == cudaSuccess) ce = dmalloc(reinterpret_cast<void**>(&job.d_eta), M * sizeof(double));
  if (ce == cudaSuccess) ce = cudaMemcpyAsync(job.d_labels, h_labels, NHW * sizeof(int32_t), cudaMemcpyHostToDevice, st);
  if (ce == cudaSuccess) ce = cudaMemcpyAsync(job.d_eta, h_eta, M * sizeof(double), cudaMemcpyHostToDevice, st);
  for (int r = 0; r < n_rounds && ce == cudaSuccess && rc == SIM3BA_OK; ++r) {
    // structure pass with the poses fixed (anchor = gauge keyframes), then the pose passes on X(eta)
    rc = sim3ba_depth_refine(job.h, job.d_labels, n_seg, h_pairs, h_delta, n_pairs, h_fixed_kf, n_fixed, depth_params, n_depth_iters, job.d_eta,
                             h_depth_cost ? h_depth_cost + (size_t)r * n_depth_iters : nullptr);
    if (rc == SIM3BA_OK) rc = sim3ba_apply_depth(job.h, job.d_points, job.d_conf, job.d_labels, n_seg, job.d_eta);
    for (int it = 0; it < n_pose_iters && ce == cudaSuccess && rc == SIM3BA_OK; ++it) {
      rc = sim3ba_step(job.h);
      if (rc == SIM3BA_OK && h_pose_cost)
        ce = cudaMemcpyAsync(h_pose_cost + (size_t)r * n_pose_iters + it, c->total_cost, sizeof(double), cudaMemcpyDeviceToHost, st);
    }
  }
  if (ce == cudaSuccess && rc == SIM3BA_OK) ce = cudaMemcpyAsync(h_poses_out, c->poses, (size_t)8 * n_kf * sizeof(double), cudaMemcpyDeviceToHost, st);
  if (ce == cudaSuccess && rc == SIM3BA_OK) ce = cudaMemcpyAsync(h_eta, job.d_eta, M * sizeof(double), cudaMemcpyDeviceToHost, st);
  if (ce == cudaSuccess && rc == SIM3BA_OK) ce = cudaStreamSynchronize(st);
  if (rc != SIM3BA_OK) { g_create_error = c->err; return rc; }
  if (ce != cudaSuccess) return cuda_fail(nullptr, ce, "sim3ba_refine_host");
  return SIM3BA_OK;
}

int sim3ba_gauge_sync(sim3ba_ctx* h, int32_t edge, const int32_t* h_moving_kf, int32_t n_moving, int32_t moving_is_i,
                      int32_t n_c_min, double* h_T, int32_t* h_n_c, int32_t* h_fallback) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (edge < 0 || edge >= c->E) return fail(c, SIM3BA_ERR_INVALID_ARG, "edge index out of range");
  if (n_moving < 0 || (n_moving > 0 && !h_moving_kf) || n_c_min < 1) return fail(c, SIM3BA_ERR_INVALID_ARG, "bad moving list or n_c_min");
  for (int k = 0; k < n_moving; ++k)
    if (h_moving_kf[k] < 0 || h_moving_kf[k] >= c->N) return fail(c, SIM3BA_ERR_INVALID_ARG, "moving keyframe out of range");
  const int grid = gauge_sync_grid(c->HW);
  double* d_work = nullptr;
  int32_t* d_moving = nullptr;
  CU(dev_alloc(&d_work, (size_t)gauge_sync_work_doubles(grid)));
  cudaError_t e = dev_alloc(&d_moving, (size_t)n_moving);
  if (e == cudaSuccess && n_moving > 0)
    e = cudaMemcpyAsync(d_moving, h_moving_kf, (size_t)n_moving * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess) e = launch_gauge_sync(c, edge, d_moving, n_moving, moving_is_i != 0, n_c_min, d_work, grid);
  double res[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(res, d_work + (size_t)gauge_sync_work_doubles(grid) - 10, sizeof(res), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);   // also keeps h_moving_kf / the temporaries alive long enough
  dfree(d_work);
  dfree(d_moving);
  if (e != cudaSuccess) return cuda_fail(c, e, "sim3ba_gauge_sync");
  if (h_T) memcpy(h_T, res, 8 * sizeof(double));
  if (h_n_c) *h_n_c = (int32_t)res[8];
  if (h_fallback) *h_fallback = (int32_t)res[9];
  c->built = false; c->solved = false;   // the poses changed
  return SIM3BA_OK;
}

int sim3ba_gauge_sync_static(sim3ba_ctx* h, int32_t edge, const int32_t* d_moving_kf, int32_t n_moving, int32_t moving_is_i,
                             int32_t n_c_min, double* d_result) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (edge < 0 || edge >= c->E) return fail(c, SIM3BA_ERR_INVALID_ARG, "edge index out of range");
  if (n_moving < 0 || (n_moving > 0 && !d_moving_kf) || n_c_min < 1 || !d_result)
    return fail(c, SIM3BA_ERR_INVALID_ARG, "bad moving list, n_c_min < 1 or NULL result buffer");
  if (c->HW > gauge_sync_static_max_pixels()) {
    char msg[200];
    snprintf(msg, sizeof(msg), "sim3ba_gauge_sync_static: image of %d pixels exceeds the static scratch array (at most %d pixels); "
             "use sim3ba_gauge_sync", c->HW, gauge_sync_static_max_pixels());
    return fail(c, SIM3BA_ERR_INVALID_ARG, msg);
  }
  const cudaError_t e = launch_gauge_sync_static(c, edge, d_moving_kf, n_moving, moving_is_i != 0, n_c_min, d_result);
  if (e != cudaSuccess) return cuda_fail(c, e, "sim3ba_gauge_sync_static");
  c->built = false; c->solved = false;   // the poses changed
  return SIM3BA_OK;
}

int sim3ba_depth_default_params(sim3ba_depth_params* p) {
  if (!p) return SIM3BA_ERR_INVALID_ARG;
  p->sigma_point = 0.05f; p->huber_k = 1.345f; p->lambda_smooth = 1.0; p->lambda_prior = 1.0; p->lambda_lm = 0.05; p->eta_max = 0.5;
  return SIM3BA_OK;
}

int sim3ba_depth_refine(sim3ba_ctx* h, const int32_t* d_labels, int32_t n_seg, const int32_t* h_pairs, const double* h_delta,
                        int32_t n_pairs, const int32_t* h_anchor_kf, int32_t n_anchor, const sim3ba_depth_params* p, int32_t n_iters,
                        double* d_eta, double* h_cost) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!d_labels || !d_eta || !p || n_seg < 1 || n_seg > depth_max_segments() || n_iters < 0 || n_pairs < 0 || n_anchor < 0 ||
      (n_pairs > 0 && (!h_pairs || !h_delta)) || (n_anchor > 0 && !h_anchor_kf))
    return fail(c, SIM3BA_ERR_INVALID_ARG, "NULL pointer, or n_seg outside 1..512, or a negative count");
  if (!(p->sigma_point > 0.f) || !(p->huber_k > 0.f) || p->lambda_smooth < 0.0 || !(p->lambda_prior > 0.0) || p->lambda_lm < 0.0 ||
      !(p->eta_max > 0.0))
    return fail(c, SIM3BA_ERR_INVALID_ARG, "invalid depth params (sigma, kappa, lambda_prior, eta_max > 0; lambda_smooth, lambda_lm >= 0)");
  const int n_total = c->N * n_seg;
  for (int q = 0; q < 2 * n_pairs; ++q)
    if (h_pairs[q] < 0 || h_pairs[q] >= n_total) return fail(c, SIM3BA_ERR_INVALID_ARG, "segment id of a boundary pair out of range");
  for (int k = 0; k < n_anchor; ++k)
    if (h_anchor_kf[k] < 0 || h_anchor_kf[k] >= c->N) return fail(c, SIM3BA_ERR_INVALID_ARG, "anchor keyframe out of range");
  CU(run_depth_refine(c, d_labels, n_seg, h_pairs, h_delta, n_pairs, h_anchor_kf, n_anchor, *p, n_iters, d_eta, h_cost));
  return SIM3BA_OK;
}

int sim3ba_apply_depth(sim3ba_ctx* h, const float* d_points, const float* d_conf, const int32_t* d_labels, int32_t n_seg,
                       const double* d_eta) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!d_points || !d_conf || !d_labels || !d_eta || n_seg < 1) return fail(c, SIM3BA_ERR_INVALID_ARG, "NULL pointer or n_seg < 1");
  CU(launch_depth_apply(c, d_points, d_conf, d_labels, n_seg, d_eta));
  c->built = false; c->solved = false;   // the pointmaps changed
  return SIM3BA_OK;
}

int sim3ba_get_edge_stats(sim3ba_ctx* h, const int32_t** nv, const uint64_t** chk, const double** cost) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (nv) *nv = c->n_valid;
  if (chk) *chk = reinterpret_cast<const uint64_t*>(c->checksum);
  if (cost) *cost = c->edge_cost;
  return SIM3BA_OK;
}

int sim3ba_get_edge_blocks(sim3ba_ctx* h, const double** b) {
  if (!h || !b) return SIM3BA_ERR_INVALID_ARG;
  *b = h->c.blocks35;
  return SIM3BA_OK;
}

int sim3ba_get_system(sim3ba_ctx* h, const double** H, int32_t* ld, const double** g) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!c->hd_valid) return fail(c, SIM3BA_ERR_BAD_STATE, "no dense system: call sim3ba_build_system first");
  if (H) *H = c->Hd;
  if (ld) *ld = c->npad;
  if (g) *g = c->g;
  return SIM3BA_OK;
}

int sim3ba_get_update(sim3ba_ctx* h, const double** tau, int32_t* attempts, double* eps_used, double* cost) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (tau) *tau = c->tau;
  if (attempts || eps_used) {
    int rc = fetch_status(c);
    if (rc) return rc;
  }
  if (attempts) *attempts = c->attempts;
  if (eps_used) *eps_used = c->eps_used;
  if (cost) {
    CU(cudaMemcpyAsync(c->h_scalar, c->total_cost, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    *cost = c->h_scalar[0];
  }
  return SIM3BA_OK;
}

int sim3ba_get_bookkeeping(sim3ba_ctx* h, const int32_t** kf_ptr, const int32_t** kf_edge, int32_t* n_pairs,
                           const int32_t** pair_kf, const int32_t** pair_ptr, const int32_t** pair_edge) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (kf_ptr) *kf_ptr = c->h_kf_ptr.data();
  if (kf_edge) *kf_edge = c->h_kf_edge.data();
  if (n_pairs) *n_pairs = c->n_pairs;
  if (pair_kf) *pair_kf = c->h_pair_kf.data();
  if (pair_ptr) *pair_ptr = c->h_pair_ptr.data();
  if (pair_edge) *pair_edge = c->h_pair_edge.data();
  return SIM3BA_OK;
}

int sim3ba_load_system(sim3ba_ctx* h, const double* d_H, const double* d_g) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (!d_H || !d_g) return fail(c, SIM3BA_ERR_INVALID_ARG, "NULL system pointer");
  CU(ensure_dense(c, true, false));
  CU(cudaMemcpyAsync(c->Hd, d_H, (size_t)c->n * c->n * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
  CU(launch_load_gradient(c, d_g));
  c->dense_loaded = true; c->hd_valid = false; c->built = false; c->solved = false;
  drop_graph(c);
  return SIM3BA_OK;
}

int sim3ba_set_solver_mode(sim3ba_ctx* h, int32_t mode) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (mode < 0 || mode > 2) return fail(c, SIM3BA_ERR_INVALID_ARG, "solver mode must be 0 (tile-sparse), 1 (dense) or 2 (band + border)");
  c->solver_mode = mode;
  drop_graph(c);
  return SIM3BA_OK;
}

int sim3ba_get_solver_info(sim3ba_ctx* h, int32_t* n_tiles, int32_t* n_tiles_dense, double* flops, int32_t* grid) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  const bool dense = c->solver_mode == 1;
  const bool bb = c->solver_mode == 2 && c->plan_bb.valid;
  SolvePlan& plan = dense ? c->plan_dense : c->plan_sparse;
  if (!plan.ready) {
    std::string err;
    if (!build_plan(c, dense, plan, err)) return fail(c, SIM3BA_ERR_CUDA, err);
  }
  const int nb = c->npad / kNB;
  if (n_tiles) *n_tiles = plan.n_tiles;
  if (n_tiles_dense) *n_tiles_dense = nb * (nb + 1) / 2;
  if (flops) *flops = bb ? c->plan_bb.flops : plan.flops;
  if (grid) *grid = c->last_solve_grid;
  return SIM3BA_OK;
}

int sim3ba_get_bb_info(sim3ba_ctx* h, int32_t info[8]) {
  if (!h || !info) return SIM3BA_ERR_INVALID_ARG;
  const BBPlan& P = h->c.plan_bb;
  info[0] = P.valid ? 1 : 0; info[1] = P.n_int; info[2] = P.n_seg; info[3] = P.n_bord; info[4] = P.max_len; info[5] = P.max_nb;
  info[6] = 0;
  for (int k = 0; k < P.n_lv; ++k) info[6] += P.lv[k].n_seg;
  info[7] = P.n_lv > 0 ? P.lv[P.n_lv - 1].n_bord : P.n_bord;
  return SIM3BA_OK;
}

int sim3ba_get_launch_count(sim3ba_ctx* h, int64_t* n) {
  if (!h || !n) return SIM3BA_ERR_INVALID_ARG;
  *n = h->c.launches;
  return SIM3BA_OK;
}

int sim3ba_set_profiling(sim3ba_ctx* h, int32_t enable) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  h->c.profiling = enable != 0;
  return SIM3BA_OK;
}

int sim3ba_get_phase_ms(sim3ba_ctx* h, float ms[8]) {
  if (!h || !ms) return SIM3BA_ERR_INVALID_ARG;
  for (int k = 0; k < 8; ++k) ms[k] = h->c.phase_ms[k];
  return SIM3BA_OK;
}

int sim3ba_copy_d2d(sim3ba_ctx* h, void* dst, const void* src, uint64_t bytes) {
  if (!h) return SIM3BA_ERR_INVALID_ARG;
  Ctx* c = &h->c;
  tl_stream = c->stream;
  if (bytes == 0) return SIM3BA_OK;
  if (!dst || !src) return fail(c, SIM3BA_ERR_INVALID_ARG, "NULL pointer in sim3ba_copy_d2d");
  CU(cudaMemcpyAsync(dst, src, (size_t)bytes, cudaMemcpyDeviceToDevice, c->stream));
  return SIM3BA_OK;
}

const char* sim3ba_last_error(const sim3ba_ctx* h) { return h ? h->c.err.c_str() : g_create_error.c_str(); }

const char* sim3ba_version(void) { return "sim3ba 0.1 (sm_100a)"; }

}  // extern "C"
#pragma GCC visibility pop
