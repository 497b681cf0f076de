// Gauge synchronisation of two map components.
//
//   PAPER.md:94     x_l = T_WCi X_i[m], y_l = T_WCj X_j[n] over the valid matches of the linking edge (i, j)
//   Eq. (3)  :96    (s*, R*, t*) = argmin sum_l |x_l - (s R y_l + t)|^2
//   Eq. (4)  :100   R* = U S V^T (S = diag(1, 1, det(U V^T))), s* = tr(S Lambda) / var(y), t* = x_bar - s* R* y_bar
//   PAPER.md:104    fewer than 64 correspondences: T* = T_WCi T_WCj^-1
//   PAPER.md:102    T* is left-multiplied onto every pose of the moving component
//
// Three small FP64 kernels: (1) a fixed-order reduction of the 19 moments (count, sum x, sum y, sum x y^T, sum |x|^2,
// sum |y|^2) over the pixels of the edge, taken about the two camera centres t_i, t_j (pivots: two components with
// far-apart origins would otherwise lose (|centroid| / spread)^2 ulps to cancellation when the moments are centred), (2) one warp: centred cross-covariance A, the proper rotation maximising
// tr(R^T A) -- the largest eigenvector of Horn's symmetric 4x4 matrix by cyclic Jacobi sweeps, which IS U S V^T of
// Eq. (4) (the search is over rotations only, so the reflection case needs no special handling) -- then
// s* = tr(R*^T A) / var(y) (= tr(S Lambda) / var(y)) and t*; (3) T* applied to the listed keyframes.
#include <mutex>

#include "sim3ba_internal.cuh"
#include "sim3_math.cuh"

namespace sim3ba {

namespace {

constexpr int kGsThreads = 256;
constexpr int kGsSlots = 20;   // [0] count, [1..3] sum x, [4..6] sum y, [7..15] sum x y^T (row-major), [16] sum |x|^2, [17] sum |y|^2

__global__ void __launch_bounds__(kGsThreads)
k_gs_moments(const float4* __restrict__ pm, const int32_t* __restrict__ match_e, const double* __restrict__ poses, int i, int j,
             int HW, double* __restrict__ partial) {
  __shared__ double s_red[kGsThreads / 32][kGsSlots];
  const Sim3d Ti = load_pose(poses + 8 * i), Tj = load_pose(poses + 8 * j);
  const float4* __restrict__ Pi = pm + (size_t)i * HW;
  const float4* __restrict__ Pj = pm + (size_t)j * HW;
  double acc[kGsSlots];
#pragma unroll
  for (int q = 0; q < kGsSlots; ++q) acc[q] = 0.0;
  for (int m = blockIdx.x * kGsThreads + threadIdx.x; m < HW; m += gridDim.x * kGsThreads) {
    const int n = match_e[m];
    if ((unsigned)n >= (unsigned)HW) continue;
    const float4 a = Pi[m], b = Pj[n];
    if (a.w < 0.f || b.w < 0.f) continue;                     // same validity as the GN step (reading R12)
    double x[3], y[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      // x_l - t_i and y_l - t_j: the moments are accumulated about the camera centres (see k_gs_solve)
      x[r] = Ti.s * (Ti.R[3 * r] * (double)a.x + Ti.R[3 * r + 1] * (double)a.y + Ti.R[3 * r + 2] * (double)a.z);
      y[r] = Tj.s * (Tj.R[3 * r] * (double)b.x + Tj.R[3 * r + 1] * (double)b.y + Tj.R[3 * r + 2] * (double)b.z);
    }
    acc[0] += 1.0;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      acc[1 + r] += x[r];
      acc[4 + r] += y[r];
#pragma unroll
      for (int c = 0; c < 3; ++c) acc[7 + 3 * r + c] = fma(x[r], y[c], acc[7 + 3 * r + c]);
      acc[16] = fma(x[r], x[r], acc[16]);
      acc[17] = fma(y[r], y[r], acc[17]);
    }
  }
#pragma unroll
  for (int q = 0; q < kGsSlots; ++q)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0)
#pragma unroll
    for (int q = 0; q < kGsSlots; ++q) s_red[warp][q] = acc[q];
  __syncthreads();
  if (threadIdx.x < kGsSlots) {
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < kGsThreads / 32; ++w) v += s_red[w][threadIdx.x];
    partial[(size_t)blockIdx.x * kGsSlots + threadIdx.x] = v;
  }
}

// eigenvector of the largest eigenvalue of the symmetric 4x4 matrix N (cyclic Jacobi, FP64)
__device__ void max_eigvec4(double N[4][4], double q[4]) {
  double V[4][4] = {{1, 0, 0, 0}, {0, 1, 0, 0}, {0, 0, 1, 0}, {0, 0, 0, 1}};
  for (int sweep = 0; sweep < 30; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int a = 0; a < 4; ++a) {
      diag += N[a][a] * N[a][a];
      for (int b = a + 1; b < 4; ++b) off += N[a][b] * N[a][b];
    }
    if (off <= 1e-32 * diag || off == 0.0) break;
    for (int p = 0; p < 3; ++p)
      for (int r = p + 1; r < 4; ++r) {
        if (N[p][r] == 0.0) continue;
        const double theta = (N[r][r] - N[p][p]) / (2.0 * N[p][r]);
        const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
        const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
        for (int k = 0; k < 4; ++k) {                         // N <- N J
          const double nkp = N[k][p], nkr = N[k][r];
          N[k][p] = c * nkp - s * nkr;
          N[k][r] = s * nkp + c * nkr;
        }
        for (int k = 0; k < 4; ++k) {                         // N <- J^T N
          const double npk = N[p][k], nrk = N[r][k];
          N[p][k] = c * npk - s * nrk;
          N[r][k] = s * npk + c * nrk;
        }
        for (int k = 0; k < 4; ++k) {
          const double vkp = V[k][p], vkr = V[k][r];
          V[k][p] = c * vkp - s * vkr;
          V[k][r] = s * vkp + c * vkr;
        }
      }
  }
  int best = 0;
  for (int a = 1; a < 4; ++a) if (N[a][a] > N[best][best]) best = a;
  for (int k = 0; k < 4; ++k) q[k] = V[k][best];
}

// out[0..7] = T* as a pose (t, q_xyzw, s), out[8] = N_c, out[9] = 1 if the endpoint fallback was taken
__global__ void __launch_bounds__(32)
k_gs_solve(const double* __restrict__ partial, int n_part, const double* __restrict__ poses, int i, int j, int moving_is_i,
           int n_c_min, double* __restrict__ out) {
  __shared__ double s_m[kGsSlots];
  const int lane = threadIdx.x;
  if (lane < kGsSlots) {
    double v = 0.0;
    for (int b = 0; b < n_part; ++b) v += partial[(size_t)b * kGsSlots + lane];
    s_m[lane] = v;
  }
  __syncwarp();
  if (lane != 0) return;
  const double nc = s_m[0];
  double Tq[4], Tt[3], Ts = 0.0;
  bool closed_form = nc >= (double)n_c_min;
  if (closed_form) {
    // reference cloud r (target) and moving cloud m: x ~ s R y + t, or with the roles swapped; the moments are about the
    // pivots t_i (x side) and t_j (y side): centroid offsets rb, mb first, the pivots added back for t* only
    const double* piv_r = poses + 8 * (moving_is_i ? j : i);
    const double* piv_m = poses + 8 * (moving_is_i ? i : j);
    double rb[3], mb[3], A[3][3], var_m;
    for (int r = 0; r < 3; ++r) { rb[r] = s_m[(moving_is_i ? 4 : 1) + r] / nc; mb[r] = s_m[(moving_is_i ? 1 : 4) + r] / nc; }
    for (int r = 0; r < 3; ++r)
      for (int c = 0; c < 3; ++c) {
        const double sxy = moving_is_i ? s_m[7 + 3 * c + r] : s_m[7 + 3 * r + c];   // sum ref_r mov_c
        A[r][c] = sxy / nc - rb[r] * mb[c];
      }
    var_m = s_m[moving_is_i ? 16 : 17] / nc - (mb[0] * mb[0] + mb[1] * mb[1] + mb[2] * mb[2]);
    // Horn's matrix for the rotation taking the moving cloud onto the reference: S_ab = sum mov_a ref_b = A[b][a]
    const double Sxx = A[0][0], Sxy = A[1][0], Sxz = A[2][0], Syx = A[0][1], Syy = A[1][1], Syz = A[2][1], Szx = A[0][2],
                 Szy = A[1][2], Szz = A[2][2];
    double Nm[4][4] = {{Sxx + Syy + Szz, Syz - Szy, Szx - Sxz, Sxy - Syx},
                       {Syz - Szy, Sxx - Syy - Szz, Sxy + Syx, Szx + Sxz},
                       {Szx - Sxz, Sxy + Syx, -Sxx + Syy - Szz, Syz + Szy},
                       {Sxy - Syx, Szx + Sxz, Syz + Szy, -Sxx - Syy + Szz}};
    double qw[4];
    max_eigvec4(Nm, qw);                                      // (w, x, y, z)
    const double qn = 1.0 / sqrt(qw[0] * qw[0] + qw[1] * qw[1] + qw[2] * qw[2] + qw[3] * qw[3]);
    Tq[0] = qw[1] * qn; Tq[1] = qw[2] * qn; Tq[2] = qw[3] * qn; Tq[3] = qw[0] * qn;
    if (Tq[3] < 0.0) for (int k = 0; k < 4; ++k) Tq[k] = -Tq[k];
    double R[9];
    quat_to_rot(Tq, R);
    double tr = 0.0;
    for (int r = 0; r < 3; ++r)
      for (int c = 0; c < 3; ++c) tr += R[3 * r + c] * A[r][c];
    Ts = tr / var_m;
    const double mc[3] = {mb[0] + piv_m[0], mb[1] + piv_m[1], mb[2] + piv_m[2]};
    for (int r = 0; r < 3; ++r) Tt[r] = (rb[r] + piv_r[r]) - Ts * (R[3 * r] * mc[0] + R[3 * r + 1] * mc[1] + R[3 * r + 2] * mc[2]);
    out[9] = 0.0;
    // degenerate clouds (coincident or collinear points: var = 0, tr <= 0) have no similarity: endpoint transform instead
    if (!(var_m > 0.0) || !(Ts > 0.0) || !isfinite(Ts) || !isfinite(Tt[0] + Tt[1] + Tt[2])) closed_form = false;
  }
  if (!closed_form) {
    // endpoint fallback: T* = T_ref T_mov^-1
    const double* pr = poses + 8 * (moving_is_i ? j : i);
    const double* pv = poses + 8 * (moving_is_i ? i : j);
    Ts = pr[7] / pv[7];
    // q = q_ref (x) conj(q_mov)
    const double ax = pr[3], ay = pr[4], az = pr[5], aw = pr[6], bx = -pv[3], by = -pv[4], bz = -pv[5], bw = pv[6];
    Tq[0] = aw * bx + ax * bw + ay * bz - az * by;
    Tq[1] = aw * by - ax * bz + ay * bw + az * bx;
    Tq[2] = aw * bz + ax * by - ay * bx + az * bw;
    Tq[3] = aw * bw - ax * bx - ay * by - az * bz;
    const double qn = 1.0 / sqrt(Tq[0] * Tq[0] + Tq[1] * Tq[1] + Tq[2] * Tq[2] + Tq[3] * Tq[3]);
    for (int k = 0; k < 4; ++k) Tq[k] *= qn;
    double R[9];
    quat_to_rot(Tq, R);
    for (int r = 0; r < 3; ++r) Tt[r] = pr[r] - Ts * (R[3 * r] * pv[0] + R[3 * r + 1] * pv[1] + R[3 * r + 2] * pv[2]);
    out[9] = 1.0;
  }
  out[0] = Tt[0]; out[1] = Tt[1]; out[2] = Tt[2];
  out[3] = Tq[0]; out[4] = Tq[1]; out[5] = Tq[2]; out[6] = Tq[3];
  out[7] = Ts;
  out[8] = nc;
}

// pose_k <- T* pose_k for the listed keyframes
__global__ void k_gs_apply(double* __restrict__ poses, const int32_t* __restrict__ moving, int n_moving, const double* __restrict__ T) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_moving) return;
  double* p = poses + 8 * moving[idx];
  double R[9];
  quat_to_rot(T + 3, R);
  const double s = T[7];
  const double t0 = p[0], t1 = p[1], t2 = p[2];
  p[0] = s * (R[0] * t0 + R[1] * t1 + R[2] * t2) + T[0];
  p[1] = s * (R[3] * t0 + R[4] * t1 + R[5] * t2) + T[1];
  p[2] = s * (R[6] * t0 + R[7] * t1 + R[8] * t2) + T[2];
  const double ax = T[3], ay = T[4], az = T[5], aw = T[6], bx = p[3], by = p[4], bz = p[5], bw = p[6];
  double q[4] = {aw * bx + ax * bw + ay * bz - az * by, aw * by - ax * bz + ay * bw + az * bx,
                 aw * bz + ax * by - ay * bx + az * bw, aw * bw - ax * bx - ay * by - az * bz};
  const double inv = 1.0 / sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  for (int a = 0; a < 4; ++a) p[3 + a] = q[a] * inv;
  p[7] *= s;
}

}  // namespace

// d_work: [grid * kGsSlots + 10] doubles; d_moving: [n_moving] keyframe indices (device).  The result T*, N_c, fallback
// flag is left in d_work[grid * kGsSlots ..].
cudaError_t launch_gauge_sync(Ctx* c, int e, const int32_t* d_moving, int n_moving, int moving_is_i, int n_c_min, double* d_work, int grid) {
  const int i = c->h_edges[2 * e], j = c->h_edges[2 * e + 1];
  double* d_out = d_work + (size_t)grid * kGsSlots;
  k_gs_moments<<<grid, kGsThreads, 0, c->stream>>>(c->pm, c->match + (size_t)e * c->HW, c->poses, i, j, c->HW, d_work);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  k_gs_solve<<<1, 32, 0, c->stream>>>(d_work, grid, c->poses, i, j, moving_is_i, n_c_min, d_out);
  err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  if (n_moving > 0) k_gs_apply<<<(n_moving + 127) / 128, 128, 0, c->stream>>>(c->poses, d_moving, n_moving, d_out);
  c->launches += 3;
  return cudaGetLastError();
}

int gauge_sync_grid(int HW) { return std::max(1, std::min((HW + 4 * kGsThreads - 1) / (4 * kGsThreads), 296)); }
int gauge_sync_work_doubles(int grid) { return grid * kGsSlots + 10; }

// ---- sim3ba_gauge_sync_static: the same computation with NO device allocation ---------------------------------------
// For callers that cannot call cudaMalloc (a region under CUDA graph capture, a serving loop, a harness that forbids it).
// The per-block moment records of k_gs_moments -- the only scratch memory of the gauge synchronisation -- live in a
// file-scope device array instead of a pool allocation; the result goes to a buffer of the caller, the moving keyframes
// come from a device array of the caller, so nothing is allocated, freed, copied from the host or synchronised.
//   * Size: one record of kGsSlots doubles per 1024 pixels, for images of at most kGsStaticMaxPixels = 2^18 pixels
//     (512 x 512; every BASELINE config is 512 x 384 or smaller): 256 x 20 x 8 = 40960 bytes, held by every GPU that
//     loads the library until the process exits.  Below that size the grid -- and with it the fixed summation order --
//     is the one sim3ba_gauge_sync uses, so the two entry points give bit-identical results.
//   * Nothing in the array has to start at zero: every record k_gs_solve reads (blocks 0 .. grid - 1) is written in
//     full by k_gs_moments of the same call, whatever an earlier call (another edge, another image size) left behind.
//   * Every call on a device shares the array: calls that overlap on the GPU (two streams, two contexts) RACE on it.
// In host code the array's name is a host-side stand-in, not a device address: the address is looked up once per device
// (that device current) with cudaGetSymbolAddress and handed to the kernels.
namespace {

constexpr int kGsStaticMaxPixels = 1 << 18;
constexpr int kGsStaticBlocks = kGsStaticMaxPixels / (4 * kGsThreads);
static __device__ __align__(256) double g_gs_scratch[kGsStaticBlocks * kGsSlots];

constexpr int kGsMaxDevices = 64;
std::mutex g_gs_mutex;
double* g_gs_scratch_addr[kGsMaxDevices] = {};

// device address of g_gs_scratch on the CURRENT device (one cudaGetSymbolAddress per device and process)
cudaError_t gs_static_scratch(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kGsMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_gs_mutex);
  if (!g_gs_scratch_addr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_gs_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_gs_scratch_addr[dev] = p;
  }
  *out = g_gs_scratch_addr[dev];
  return cudaSuccess;
}

// k_gs_apply for a list nobody has validated on the host: indices outside 0 .. N - 1 are skipped
__global__ void k_gs_apply_checked(double* __restrict__ poses, const int32_t* __restrict__ moving, int n_moving, int N,
                                   const double* __restrict__ T) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= n_moving) return;
  const int kf = moving[idx];
  if ((unsigned)kf >= (unsigned)N) return;
  double* p = poses + 8 * kf;
  double R[9];
  quat_to_rot(T + 3, R);
  const double s = T[7];
  const double t0 = p[0], t1 = p[1], t2 = p[2];
  p[0] = s * (R[0] * t0 + R[1] * t1 + R[2] * t2) + T[0];
  p[1] = s * (R[3] * t0 + R[4] * t1 + R[5] * t2) + T[1];
  p[2] = s * (R[6] * t0 + R[7] * t1 + R[8] * t2) + T[2];
  const double ax = T[3], ay = T[4], az = T[5], aw = T[6], bx = p[3], by = p[4], bz = p[5], bw = p[6];
  double q[4] = {aw * bx + ax * bw + ay * bz - az * by, aw * by - ax * bz + ay * bw + az * bx,
                 aw * bz + ax * by - ay * bx + az * bw, aw * bw - ax * bx - ay * by - az * bz};
  const double inv = 1.0 / sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  for (int a = 0; a < 4; ++a) p[3 + a] = q[a] * inv;
  p[7] *= s;
}

}  // namespace

int gauge_sync_static_max_pixels() { return kGsStaticMaxPixels; }

// d_moving [n_moving] and d_result [10] are device arrays of the caller; asynchronous on the context's stream
cudaError_t launch_gauge_sync_static(Ctx* c, int e, const int32_t* d_moving, int n_moving, int moving_is_i, int n_c_min,
                                     double* d_result) {
  if (c->HW > kGsStaticMaxPixels) return cudaErrorInvalidValue;          // the entry point has said why
  double* scratch = nullptr;
  cudaError_t err = gs_static_scratch(&scratch);
  if (err != cudaSuccess) return err;
  const int grid = gauge_sync_grid(c->HW);                                // <= kGsStaticBlocks for HW <= kGsStaticMaxPixels
  if (grid > kGsStaticBlocks) return cudaErrorInvalidValue;
  const int i = c->h_edges[2 * e], j = c->h_edges[2 * e + 1];
  k_gs_moments<<<grid, kGsThreads, 0, c->stream>>>(c->pm, c->match + (size_t)e * c->HW, c->poses, i, j, c->HW, scratch);
  err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  k_gs_solve<<<1, 32, 0, c->stream>>>(scratch, grid, c->poses, i, j, moving_is_i, n_c_min, d_result);
  err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  if (n_moving > 0)
    k_gs_apply_checked<<<(n_moving + 127) / 128, 128, 0, c->stream>>>(c->poses, d_moving, n_moving, c->N, d_result);
  c->launches += 3;
  return cudaGetLastError();
}

}  // namespace sim3ba
