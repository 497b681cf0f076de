// Device-side FP64 Sim(3) helpers: pose decoding, T_ij, Ad_{T^-1}, Exp-map retraction.
// PAPER.md:71 (pose convention), :114 (left perturbation, tau = (v, omega, zeta)), :118 (adjoints).
// Independent of oracle/: W(omega, zeta) = phi_1([omega]x + zeta I) is evaluated here by a 3x3
// matrix power series with argument halving + the doubling rule, not by scalar closed forms.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace sim3ba {

struct Sim3d {
  double s;
  double R[9];  // row-major
  double t[3];
};

__host__ __device__ inline void quat_to_rot(const double* q, double* R) {
  double x = q[0], y = q[1], z = q[2], w = q[3];
  double nn = x * x + y * y + z * z + w * w;
  double k = nn > 0.0 ? 2.0 / nn : 0.0;
  R[0] = 1.0 - k * (y * y + z * z); R[1] = k * (x * y - z * w);       R[2] = k * (x * z + y * w);
  R[3] = k * (x * y + z * w);       R[4] = 1.0 - k * (x * x + z * z); R[5] = k * (y * z - x * w);
  R[6] = k * (x * z - y * w);       R[7] = k * (y * z + x * w);       R[8] = 1.0 - k * (x * x + y * y);
}

__host__ __device__ inline Sim3d load_pose(const double* p) {
  Sim3d T;
  T.t[0] = p[0]; T.t[1] = p[1]; T.t[2] = p[2];
  quat_to_rot(p + 3, T.R);
  T.s = p[7];
  return T;
}

// T_ij = T_i^-1 T_j : s = s_j/s_i, R = R_i^T R_j, t = R_i^T (t_j - t_i) / s_i
__host__ __device__ inline Sim3d relative_pose(const Sim3d& Ti, const Sim3d& Tj) {
  Sim3d T;
  T.s = Tj.s / Ti.s;
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c)
      T.R[3 * r + c] = Ti.R[0 + r] * Tj.R[0 + c] + Ti.R[3 + r] * Tj.R[3 + c] + Ti.R[6 + r] * Tj.R[6 + c];
  double d[3] = {Tj.t[0] - Ti.t[0], Tj.t[1] - Ti.t[1], Tj.t[2] - Ti.t[2]};
  for (int r = 0; r < 3; ++r) T.t[r] = (Ti.R[0 + r] * d[0] + Ti.R[3 + r] * d[1] + Ti.R[6 + r] * d[2]) / Ti.s;
  return T;
}

// Ad_{T^-1} (7x7 row-major), rows/cols (v, omega, zeta):
//   [[R^T/s, -R^T [t]x / s, R^T t / s], [0, R^T, 0], [0, 0, 1]]
__host__ __device__ inline void adjoint_of_inverse(const Sim3d& T, double* Ad) {
  for (int k = 0; k < 49; ++k) Ad[k] = 0.0;
  const double is = 1.0 / T.s;
  const double* t = T.t;
  // [t]x
  double tx[9] = {0.0, -t[2], t[1], t[2], 0.0, -t[0], -t[1], t[0], 0.0};
  for (int r = 0; r < 3; ++r) {
    double rt = 0.0;
    for (int c = 0; c < 3; ++c) {
      double Rt = T.R[3 * c + r];  // (R^T)[r][c]
      Ad[7 * r + c] = Rt * is;
      Ad[7 * (3 + r) + 3 + c] = Rt;
      double acc = 0.0;
      for (int k = 0; k < 3; ++k) acc += T.R[3 * k + r] * tx[3 * k + c];
      Ad[7 * r + 3 + c] = -acc * is;
      rt += Rt * t[c];
    }
    Ad[7 * r + 6] = rt * is;
  }
  Ad[48] = 1.0;
}

__host__ __device__ inline void mat3_mul(const double* A, const double* B, double* C) {
  for (int r = 0; r < 3; ++r)
    for (int c = 0; c < 3; ++c) C[3 * r + c] = A[3 * r] * B[c] + A[3 * r + 1] * B[3 + c] + A[3 * r + 2] * B[6 + c];
}

// W = phi_1(M), M = [omega]x + zeta I, phi_1(M) = sum_k M^k/(k+1)!.
// Halve M until its norm is <= 0.25, sum the series there, then apply
// phi_1(2M) = (exp(M) + I) phi_1(M) / 2 with exp(M) = I + M phi_1(M).
__host__ __device__ inline void sim3_W(const double* om, double zeta, double* W) {
  double M[9] = {zeta, -om[2], om[1], om[2], zeta, -om[0], -om[1], om[0], zeta};
  double nrm = fabs(zeta) + sqrt(om[0] * om[0] + om[1] * om[1] + om[2] * om[2]);
  int j = 0;
  while (nrm > 0.25 && j < 40) { nrm *= 0.5; ++j; }
  const double sc = ldexp(1.0, -j);
  for (int k = 0; k < 9; ++k) M[k] *= sc;
  double P[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};   // M^k / (k+1)!
  for (int k = 0; k < 9; ++k) W[k] = P[k];
  for (int k = 1; k <= 18; ++k) {
    double Q[9];
    mat3_mul(P, M, Q);
    const double inv = 1.0 / (double)(k + 1);
    for (int a = 0; a < 9; ++a) { P[a] = Q[a] * inv; W[a] += P[a]; }
  }
  for (int it = 0; it < j; ++it) {
    double E[9], Q[9];
    mat3_mul(M, W, E);                 // exp(M) - I
    E[0] += 2.0; E[4] += 2.0; E[8] += 2.0;   // exp(M) + I
    mat3_mul(E, W, Q);
    for (int a = 0; a < 9; ++a) { W[a] = 0.5 * Q[a]; M[a] *= 2.0; }
  }
}

// pose <- Exp(tau) pose;  s' = e^zeta s, R' = Exp(omega) R, t' = e^zeta Exp(omega) t + W v
__host__ __device__ inline void retract_pose(double* p, const double* tau) {
  const double* v = tau;
  const double* om = tau + 3;
  const double zeta = tau[6];
  const double th2 = om[0] * om[0] + om[1] * om[1] + om[2] * om[2];
  const double th = sqrt(th2);
  double k, cw;  // dq = (k*om, cw) = (sin(th/2)/th * om, cos(th/2))
  if (th < 1e-4) {
    k = 0.5 - th2 / 48.0 + th2 * th2 / 3840.0;
    cw = 1.0 - th2 / 8.0 + th2 * th2 / 384.0;
  } else {
    k = sin(0.5 * th) / th;
    cw = cos(0.5 * th);
  }
  double dq[4] = {k * om[0], k * om[1], k * om[2], cw};
  double Rd[9];
  quat_to_rot(dq, Rd);
  double W[9];
  sim3_W(om, zeta, W);
  const double ez = exp(zeta);
  double t[3] = {p[0], p[1], p[2]};
  for (int r = 0; r < 3; ++r)
    p[r] = ez * (Rd[3 * r] * t[0] + Rd[3 * r + 1] * t[1] + Rd[3 * r + 2] * t[2]) +
           (W[3 * r] * v[0] + W[3 * r + 1] * v[1] + W[3 * r + 2] * v[2]);
  // q' = dq (x) q
  const double ax = dq[0], ay = dq[1], az = dq[2], aw = dq[3];
  const double bx = p[3], by = p[4], bz = p[5], bw = p[6];
  double q[4] = {aw * bx + ax * bw + ay * bz - az * by, aw * by - ax * bz + ay * bw + az * bx,
                 aw * bz + ax * by - ay * bx + az * bw, aw * bw - ax * bx - ay * by - az * bz};
  const double inv = 1.0 / sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  for (int a = 0; a < 4; ++a) p[3 + a] = q[a] * inv;
  p[7] *= ez;
}

}  // namespace sim3ba
