"""CPU float64 oracle of the Sim(3) Gauss-Newton step of CoMo3R-SLAM, written from the paper.

TEST INFRASTRUCTURE ONLY.  Nothing in the product path (``paper_2605_30488_b200/``) may import,
call or execute this file; only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs do.  It shares no code with the CUDA path.

What it computes (section III-D), match by match, in float64, with none of
the GPU path's algebraic shortcuts: the ray-range residual of Eq. (1), the
confidence whitening and per-component Huber IRLS weights of PAPER.md:76, the chain-rule Jacobian
blocks of Eq. (6) and Dd/Dx, the endpoint adjoints -/+ Ad_{T_WCi^-1}
 applied to every match, the sums J^T W J / J^T W e scattered into the global 7N
system, removal of the gauge keyframes, the regularised Cholesky solve of Eq. (7)
with the epsilon escalation of PAPER.md:122, and the left retraction T <- Exp(tau) T
(PAPER.md:114).

Readings of silent / garbled passages are DESIGN.md "Readings" R1..R18 (quoted where used).

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): Exp vs scipy.linalg.expm of the 4x4 generator,
Exp/Log round trips, T Exp(tau) T^-1 = Exp(Ad_T tau), hand-computed residuals
(tests/golden/residual_hand_case.txt), central finite differences of the residual for both
endpoint Jacobians, the closed-form J_xi, kappa->inf reduction to numpy.linalg.lstsq on the
stacked finite-difference Jacobian, symmetric PSD H with zero block-row sums, zero gradient at
ground truth on clean data, numpy.linalg.solve on the reduced system, forced epsilon escalation,
monotone cost decrease and convergence to ground truth up to the fixed gauge.
Parity vs the authors' own code: **parity unpinned** (the paper prints no worked number for this
path and ships no code).

Pose layout: pose[8] = (t[3], q_xyzw[4], s) for T_WC: X -> s R(q) X + t.
Tangent ordering: tau = (v, omega, zeta).
"""
from __future__ import annotations

from dataclasses import dataclass
from math import comb, factorial
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np
import scipy.linalg


# ----------------------------------------------------------------------------------------------
@dataclass
class Params:
    """Robust-kernel and solver constants."""
    sigma_ray: float = 0.003      # sigma_r
    sigma_dist: float = 10.0      # sigma_d
    huber_k: float = 1.345        # kappa on the whitened residual
    conf_min: float = 0.0         # match valid iff both confidences > conf_min (reading R12)
    lm_lambda: float = 0.0        # lambda of Eq. (7); global backend: 0 (reading R7)
    eps0: float = 1e-6            # epsilon_0
    max_attempts: int = 6         # epsilon_r = eps0 * 100^r, r = 0..5

    @property
    def sigma(self) -> np.ndarray:
        return np.array([self.sigma_ray, self.sigma_ray, self.sigma_ray, self.sigma_dist])


# ----------------------------------------------------------------------------------------------
# SO(3) / Sim(3) tangent-space operations (PAPER.md:114 cites [27]; formulas: DESIGN.md card)
def hat(w: np.ndarray) -> np.ndarray:
    """[w]x, the 3x3 skew matrix with [w]x y = w x y."""
    return np.array([[0.0, -w[2], w[1]], [w[2], 0.0, -w[0]], [-w[1], w[0], 0.0]])


def quat_to_rot(q: np.ndarray) -> np.ndarray:
    x, y, z, w = q / np.linalg.norm(q)
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


def rot_to_quat(R: np.ndarray) -> np.ndarray:
    """xyzw unit quaternion of a rotation matrix (largest-component branch), w >= 0."""
    K = np.array([R[0, 0] + R[1, 1] + R[2, 2], R[0, 0] - R[1, 1] - R[2, 2],
                  -R[0, 0] + R[1, 1] - R[2, 2], -R[0, 0] - R[1, 1] + R[2, 2]])
    i = int(np.argmax(K))
    r = np.sqrt(max(0.0, 1.0 + K[i]))
    if i == 0:
        q = np.array([(R[2, 1] - R[1, 2]) / (2 * r), (R[0, 2] - R[2, 0]) / (2 * r),
                      (R[1, 0] - R[0, 1]) / (2 * r), r / 2])
    elif i == 1:
        q = np.array([r / 2, (R[0, 1] + R[1, 0]) / (2 * r), (R[0, 2] + R[2, 0]) / (2 * r),
                      (R[2, 1] - R[1, 2]) / (2 * r)])
    elif i == 2:
        q = np.array([(R[0, 1] + R[1, 0]) / (2 * r), r / 2, (R[1, 2] + R[2, 1]) / (2 * r),
                      (R[0, 2] - R[2, 0]) / (2 * r)])
    else:
        q = np.array([(R[0, 2] + R[2, 0]) / (2 * r), (R[1, 2] + R[2, 1]) / (2 * r), r / 2,
                      (R[1, 0] - R[0, 1]) / (2 * r)])
    q = q / np.linalg.norm(q)
    return -q if q[3] < 0 else q


def so3_exp(w: np.ndarray) -> np.ndarray:
    """Rodrigues: Exp(w) = I + sin(th)/th [w]x + (1-cos(th))/th^2 [w]x^2."""
    th = float(np.linalg.norm(w))
    W = hat(w)
    if th < 1e-5:
        a = 1.0 - th * th / 6.0 + th ** 4 / 120.0
        b = 0.5 - th * th / 24.0 + th ** 4 / 720.0
    else:
        a = np.sin(th) / th
        b = (1.0 - np.cos(th)) / (th * th)
    return np.eye(3) + a * W + b * (W @ W)


def so3_log(R: np.ndarray) -> np.ndarray:
    """Rotation vector of R, |w| <= pi, through the unit quaternion (stable near 0 and pi)."""
    q = rot_to_quat(R)
    nv = float(np.linalg.norm(q[:3]))
    if nv < 1e-12:
        return 2.0 * q[:3] / q[3]
    return 2.0 * np.arctan2(nv, q[3]) * q[:3] / nv


def _w_coeffs(theta: float, zeta: float) -> Tuple[float, float, float]:
    """A, B, C of W = C I + A [w]x + B [w]x^2 = int_0^1 e^{s zeta} Exp(s w) ds.

    With z = zeta + i theta and phi(z) = (e^z - 1)/z = sum_k z^k/(k+1)!:
    C = phi(zeta), A = Im phi(z)/theta, B = (C - Re phi(z))/theta^2.  For small theta the
    divisions are carried out term by term on the binomial expansion of (zeta + i theta)^k, so
    there is no cancellation; otherwise the closed forms of the DESIGN.md card are used.
    """
    C = 1.0 if zeta == 0.0 else float(np.expm1(zeta) / zeta)
    if theta < 0.5 and abs(zeta) < 3.0:
        A = 0.0
        B = 0.0
        for k in range(1, 48):
            inv = 1.0 / factorial(k + 1)
            # Im (zeta + i theta)^k / theta = sum_j C(k,2j+1) zeta^(k-2j-1) (-1)^j theta^(2j)
            for j in range(0, (k - 1) // 2 + 1):
                A += comb(k, 2 * j + 1) * zeta ** (k - 2 * j - 1) * (-1) ** j * theta ** (2 * j) * inv
            # (zeta^k - Re (zeta + i theta)^k)/theta^2 = sum_{j>=1} C(k,2j) zeta^(k-2j) (-1)^(j+1) theta^(2j-2)
            for j in range(1, k // 2 + 1):
                B += comb(k, 2 * j) * zeta ** (k - 2 * j) * (-1) ** (j + 1) * theta ** (2 * j - 2) * inv
        return A, B, C
    ez = np.exp(zeta)
    den = zeta * zeta + theta * theta
    A = (ez * (zeta * np.sin(theta) - theta * np.cos(theta)) + theta) / (theta * den)
    B = (C - (ez * (zeta * np.cos(theta) + theta * np.sin(theta)) - zeta) / den) / (theta * theta)
    return float(A), float(B), C


def sim3_w(omega: np.ndarray, zeta: float) -> np.ndarray:
    A, B, C = _w_coeffs(float(np.linalg.norm(omega)), float(zeta))
    Om = hat(omega)
    return C * np.eye(3) + A * Om + B * (Om @ Om)


def sim3_exp(tau: np.ndarray) -> Tuple[float, np.ndarray, np.ndarray]:
    """Exp(tau) = (e^zeta, Exp_SO3(omega), W v); tau = (v, omega, zeta)."""
    v, om, ze = np.asarray(tau[0:3], float), np.asarray(tau[3:6], float), float(tau[6])
    return float(np.exp(ze)), so3_exp(om), sim3_w(om, ze) @ v


def sim3_log(s: float, R: np.ndarray, t: np.ndarray) -> np.ndarray:
    om = so3_log(R)
    ze = float(np.log(s))
    v = np.linalg.solve(sim3_w(om, ze), t)
    return np.concatenate([v, om, [ze]])


def sim3_matrix(s: float, R: np.ndarray, t: np.ndarray) -> np.ndarray:
    T = np.eye(4)
    T[:3, :3] = s * R
    T[:3, 3] = t
    return T


def sim3_inv(s: float, R: np.ndarray, t: np.ndarray) -> Tuple[float, np.ndarray, np.ndarray]:
    return 1.0 / s, R.T, -(R.T @ t) / s


def sim3_mul(a, b) -> Tuple[float, np.ndarray, np.ndarray]:
    sa, Ra, ta = a
    sb, Rb, tb = b
    return sa * sb, Ra @ Rb, sa * (Ra @ tb) + ta


def sim3_adjoint(s: float, R: np.ndarray, t: np.ndarray) -> np.ndarray:
    """Ad_T with T Exp(tau) T^-1 = Exp(Ad_T tau), rows/cols ordered (v, omega, zeta)."""
    Ad = np.zeros((7, 7))
    Ad[0:3, 0:3] = s * R
    Ad[0:3, 3:6] = hat(t) @ R
    Ad[0:3, 6] = -t
    Ad[3:6, 3:6] = R
    Ad[6, 6] = 1.0
    return Ad


def pose_to_srt(p: np.ndarray) -> Tuple[float, np.ndarray, np.ndarray]:
    return float(p[7]), quat_to_rot(np.asarray(p[3:7], float)), np.asarray(p[0:3], float).copy()


def srt_to_pose(s: float, R: np.ndarray, t: np.ndarray) -> np.ndarray:
    return np.concatenate([t, rot_to_quat(R), [s]])


# ----------------------------------------------------------------------------------------------
# robust kernel
def huber_weight(r: np.ndarray, k: float) -> np.ndarray:
    """w(r) = min(1, kappa/|r|); w(0) = 1 (reading R11)."""
    a = np.abs(r)
    return np.where(a <= k, 1.0, k / np.maximum(a, 1e-300))


def huber_rho(r: np.ndarray, k: float) -> np.ndarray:
    a = np.abs(r)
    return np.where(a <= k, 0.5 * r * r, k * (a - 0.5 * k))


# ----------------------------------------------------------------------------------------------
# per-edge terms, vectorised over the matches of one edge (each match still gets the literal
# chain rule and its own Ad product; nothing is hoisted out of the per-match algebra)
@dataclass
class EdgeTerms:
    m: np.ndarray        # valid pixels of i
    n: np.ndarray        # matched pixels of j
    e: np.ndarray        # [M,4] residual Eq. (1)
    r: np.ndarray        # [M,4] whitened residual
    omega: np.ndarray    # [M,4] row weights q w_c / sigma_c^2
    J_xi: np.ndarray     # [M,4,7] d e / d xi (xi = perturbation of T_ij on the left)
    J_i: np.ndarray      # [M,4,7]
    J_j: np.ndarray      # [M,4,7]
    cost: float


def valid_matches(match_e: np.ndarray, conf_i: np.ndarray, conf_j: np.ndarray, conf_min: float):
    """Reading R12: valid <=> 0 <= n < HW and c_i[m] > c_min and c_j[n] > c_min."""
    HW = match_e.shape[0]
    m = np.flatnonzero((match_e >= 0) & (match_e < HW))
    n = match_e[m].astype(np.int64)
    keep = (conf_i[m] > conf_min) & (conf_j[n] > conf_min)
    return m[keep].astype(np.int64), n[keep]


def residual(Tij, Xi: np.ndarray, Xj: np.ndarray) -> np.ndarray:
    """Eq. (1): e = [psi(T Xj) - psi(Xi); |T Xj| - |Xi|], rows = matches."""
    s, R, t = Tij
    x = s * Xj @ R.T + t
    d = np.maximum(np.linalg.norm(x, axis=1), 1e-12)       # clamp, reading R11
    di = np.maximum(np.linalg.norm(Xi, axis=1), 1e-12)
    return np.concatenate([x / d[:, None] - Xi / di[:, None], (d - di)[:, None]], axis=1)


def edge_terms(pose_i: np.ndarray, pose_j: np.ndarray, Xi_all: np.ndarray, ci_all: np.ndarray,
               Xj_all: np.ndarray, cj_all: np.ndarray, match_e: np.ndarray, prm: Params) -> EdgeTerms:
    Ti = pose_to_srt(pose_i)
    Tj = pose_to_srt(pose_j)
    Ti_inv = sim3_inv(*Ti)
    Tij = sim3_mul(Ti_inv, Tj)                              # T_ij = T_WCi^-1 T_WCj
    Ad = sim3_adjoint(*Ti_inv)                              # Ad_{T_WCi^-1}

    m, n = valid_matches(match_e, ci_all, cj_all, prm.conf_min)
    Xi = Xi_all[m].astype(np.float64)
    Xj = Xj_all[n].astype(np.float64)
    ci = ci_all[m].astype(np.float64)
    cj = cj_all[n].astype(np.float64)
    M = m.shape[0]

    e = residual(Tij, Xi, Xj)
    q = np.sqrt(ci * cj)                                    # reading R5
    sig = prm.sigma
    r = np.sqrt(q)[:, None] * e / sig[None, :]              # Sigma_mn = Sigma / q
    w = huber_weight(r, prm.huber_k)
    omega = q[:, None] * w / (sig * sig)[None, :]
    cost = float(huber_rho(r, prm.huber_k).sum())

    s, R, t = Tij
    x = s * Xj @ R.T + t
    d = np.maximum(np.linalg.norm(x, axis=1), 1e-12)
    # Dx/Dxi = [I, -[x]x, x]  (Eq. (6))
    Dx = np.zeros((M, 3, 7))
    Dx[:, 0, 0] = Dx[:, 1, 1] = Dx[:, 2, 2] = 1.0
    Dx[:, 0, 4] = x[:, 2]
    Dx[:, 0, 5] = -x[:, 1]
    Dx[:, 1, 3] = -x[:, 2]
    Dx[:, 1, 5] = x[:, 0]
    Dx[:, 2, 3] = x[:, 1]
    Dx[:, 2, 4] = -x[:, 0]
    Dx[:, :, 6] = x
    # Dpsi/Dx = (I - x x^T / d^2) / d (Eq. (6)); Dd/Dx = x^T / d
    De = np.zeros((M, 4, 3))
    De[:, 0:3, :] = (np.eye(3)[None] - x[:, :, None] * x[:, None, :] / (d * d)[:, None, None]) / d[:, None, None]
    De[:, 3, :] = x / d[:, None]
    J_xi = De @ Dx                                          # 4 x 7 block per match
    J_j = J_xi @ Ad                                         # + Ad_{T_WCi^-1}
    J_i = -(J_xi @ Ad)                                      # - Ad_{T_WCi^-1}
    return EdgeTerms(m, n, e, r, omega, J_xi, J_i, J_j, cost)


# ----------------------------------------------------------------------------------------------
@dataclass
class System:
    H: np.ndarray            # [7N, 7N] before gauge removal and damping
    g: np.ndarray            # [7N]  g = sum J^T Omega e (reading R10)
    g_abs: np.ndarray        # [7N]  sum |J^T| Omega |e| (floor for converged iterations)
    cost: float
    n_valid: np.ndarray      # [E] int64
    checksum: np.ndarray     # [E] uint64: sum (m*HW + n) mod 2^64 over the valid matches
    edge_A: np.ndarray       # [E,7,7]  J_j^T Omega J_j summed (= H_jj contribution of the edge)
    edge_b: np.ndarray       # [E,7]    J_j^T Omega e summed (= g_j contribution of the edge)
    edge_cost: np.ndarray    # [E]
    edge_b_abs: np.ndarray   # [E,7]    sum |J_j^T| Omega |e| (floor for converged iterations)


def build_system(poses: np.ndarray, points: np.ndarray, conf: np.ndarray, edges: np.ndarray,
                 match: np.ndarray, prm: Params, edge_subset: Optional[Sequence[int]] = None) -> System:
    """Normal-equation assembly: H = sum J^T Omega J, g = sum J^T Omega e."""
    N, HW = points.shape[0], points.shape[1]
    E = edges.shape[0]
    H = np.zeros((7 * N, 7 * N))
    g = np.zeros(7 * N)
    g_abs = np.zeros(7 * N)
    n_valid = np.zeros(E, dtype=np.int64)
    checksum = np.zeros(E, dtype=np.uint64)
    edge_A = np.zeros((E, 7, 7))
    edge_b = np.zeros((E, 7))
    edge_cost = np.zeros(E)
    edge_b_abs = np.zeros((E, 7))
    cost = 0.0
    for e in (range(E) if edge_subset is None else edge_subset):
        i, j = int(edges[e, 0]), int(edges[e, 1])
        tm = edge_terms(poses[i], poses[j], points[i], conf[i], points[j], conf[j], match[e], prm)
        Ji = tm.J_i.reshape(-1, 7)
        Jj = tm.J_j.reshape(-1, 7)
        om = tm.omega.reshape(-1)
        ee = tm.e.reshape(-1)
        WJi = om[:, None] * Ji
        WJj = om[:, None] * Jj
        Hii, Hij, Hjj = Ji.T @ WJi, Ji.T @ WJj, Jj.T @ WJj
        gi, gj = WJi.T @ ee, WJj.T @ ee
        si, sj = slice(7 * i, 7 * i + 7), slice(7 * j, 7 * j + 7)
        H[si, si] += Hii
        H[si, sj] += Hij
        H[sj, si] += Hij.T
        H[sj, sj] += Hjj
        g[si] += gi
        g[sj] += gj
        g_abs[si] += np.abs(WJi).T @ np.abs(ee)
        edge_b_abs[e] = np.abs(WJj).T @ np.abs(ee)
        g_abs[sj] += edge_b_abs[e]
        n_valid[e] = tm.m.shape[0]
        with np.errstate(over="ignore"):
            checksum[e] = np.sum(tm.m.astype(np.uint64) * np.uint64(HW) + tm.n.astype(np.uint64),
                                 dtype=np.uint64)
        edge_A[e], edge_b[e], edge_cost[e] = Hjj, gj, tm.cost
        cost += tm.cost
    return System(H, g, g_abs, cost, n_valid, checksum, edge_A, edge_b, edge_cost, edge_b_abs)


def total_cost(poses, points, conf, edges, match, prm: Params) -> float:
    """E_global of Eq. (5)."""
    c = 0.0
    for e in range(edges.shape[0]):
        i, j = int(edges[e, 0]), int(edges[e, 1])
        Ti, Tj = pose_to_srt(poses[i]), pose_to_srt(poses[j])
        Tij = sim3_mul(sim3_inv(*Ti), Tj)
        m, n = valid_matches(match[e], conf[i], conf[j], prm.conf_min)
        ee = residual(Tij, points[i][m].astype(np.float64), points[j][n].astype(np.float64))
        q = np.sqrt(conf[i][m].astype(np.float64) * conf[j][n].astype(np.float64))
        c += float(huber_rho(np.sqrt(q)[:, None] * ee / prm.sigma[None, :], prm.huber_k).sum())
    return c


# ----------------------------------------------------------------------------------------------
@dataclass
class Solution:
    tau: np.ndarray          # [7N], zero on the fixed keyframes
    attempts: int            # factorisations tried (1 = first succeeded)
    eps_used: float          # epsilon of the successful attempt (nan if all failed)
    ok: bool


def free_index(n_kf: int, fixed_kf: Sequence[int]) -> np.ndarray:
    fixed = set(int(k) for k in fixed_kf)
    return np.concatenate([np.arange(7 * k, 7 * k + 7) for k in range(n_kf) if k not in fixed]
                          or [np.zeros(0, dtype=np.int64)]).astype(np.int64)


def solve(H: np.ndarray, g: np.ndarray, fixed_kf: Sequence[int], prm: Params) -> Solution:
    """Eq. (7) on the system with the gauge keyframes deleted:
    (H + lambda diag(H) + eps_r I) tau = -g by dense Cholesky; on factorisation failure
    eps_r = eps0 * 100^r for up to max_attempts attempts, else tau = 0."""
    N = g.shape[0] // 7
    fr = free_index(N, fixed_kf)
    Hr = H[np.ix_(fr, fr)]
    gr = g[fr]
    tau = np.zeros_like(g)
    for r in range(prm.max_attempts):
        eps = prm.eps0 * (100.0 ** r)
        A = Hr + prm.lm_lambda * np.diag(np.diag(Hr)) + eps * np.eye(Hr.shape[0])
        try:
            c, low = scipy.linalg.cho_factor(A, lower=True, check_finite=True)
            x = scipy.linalg.cho_solve((c, low), -gr)
            if not np.all(np.isfinite(x)):
                raise np.linalg.LinAlgError("non-finite")
        except (np.linalg.LinAlgError, ValueError):
            continue
        tau[fr] = x
        return Solution(tau, r + 1, eps, True)
    return Solution(tau, prm.max_attempts, float("nan"), False)


def retract(poses: np.ndarray, tau: np.ndarray) -> np.ndarray:
    """T_WCi <- Exp(tau_i) T_WCi; quaternion re-normalised (reading R15)."""
    out = np.empty_like(poses)
    for k in range(poses.shape[0]):
        out[k] = srt_to_pose(*sim3_mul(sim3_exp(tau[7 * k:7 * k + 7]), pose_to_srt(poses[k])))
    return out


def gn_step(poses, points, conf, edges, match, fixed_kf, prm: Params):
    """One Gauss-Newton iteration: assemble, solve, retract.  Returns (new poses, System, Solution)."""
    sysm = build_system(poses, points, conf, edges, match, prm)
    sol = solve(sysm.H, sysm.g, fixed_kf, prm)
    return retract(poses, sol.tau), sysm, sol


def pose_delta_log(pose_a: np.ndarray, pose_b: np.ndarray) -> np.ndarray:
    """Log(T_a T_b^-1) in R^7 (used by tests to compare accumulated updates)."""
    return sim3_log(*sim3_mul(pose_to_srt(pose_a), sim3_inv(*pose_to_srt(pose_b))))


# ----------------------------------------------------------------------------------------------
# integer bookkeeping (a0): CSR structures the assembly gathers from
def bookkeeping(n_kf: int, edges: np.ndarray) -> Dict[str, np.ndarray]:
    """Keyframe -> incident-edge CSR (edge order ascending) and the sorted list of unique unordered
    keyframe pairs with a pair -> edge CSR (edge order ascending).  Integer, unique result."""
    E = edges.shape[0]
    inc: List[List[int]] = [[] for _ in range(n_kf)]
    for e in range(E):
        inc[int(edges[e, 0])].append(e)
        inc[int(edges[e, 1])].append(e)
    kf_ptr = np.zeros(n_kf + 1, dtype=np.int32)
    for k in range(n_kf):
        kf_ptr[k + 1] = kf_ptr[k] + len(inc[k])
    kf_edge = np.array([e for l in inc for e in l], dtype=np.int32)
    pairs: Dict[Tuple[int, int], List[int]] = {}
    for e in range(E):
        a, b = int(edges[e, 0]), int(edges[e, 1])
        pairs.setdefault((max(a, b), min(a, b)), []).append(e)
    keys = sorted(pairs)
    pair_kf = np.array(keys, dtype=np.int32).reshape(-1, 2)      # (hi, lo)
    pair_ptr = np.zeros(len(keys) + 1, dtype=np.int32)
    for p, k in enumerate(keys):
        pair_ptr[p + 1] = pair_ptr[p] + len(pairs[k])
    pair_edge = np.array([e for k in keys for e in pairs[k]], dtype=np.int32)
    return dict(kf_ptr=kf_ptr, kf_edge=kf_edge, pair_kf=pair_kf, pair_ptr=pair_ptr, pair_edge=pair_edge)
