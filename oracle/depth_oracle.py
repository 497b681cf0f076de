"""CPU float64 oracle of the segment-level structure refinement with poses fixed (section III-E,
Eq. (8)-(10)), written from the paper.  SURVEY section 8(f) NEXT-1 (BASELINE config 5: "pose-depth alternation with 32
segments per KF each carrying one log-depth-scale unknown solved per segment with poses held fixed").

TEST INFRASTRUCTURE ONLY (same rule as sim3_gn_oracle.py): only ``tests/`` may import it; it shares no code with the
CUDA path.

What it computes, match by match, in the paper's order and notation:
  Eq. (8)  :130   X_{k,p}(eta_g) = |X_init| exp(eta_g) psi(X_init) = exp(eta_g) X_init, one eta_g per segment g
  Eq. (9)  :134   r_c = sqrt(q_mn) [T_ij X_j,n(eta) - X_i,m(eta)]_c / sigma_point, c = 1..3, per-component Huber rho
  :143            J_g = -d_i psi(X_i,m) = -X_i,m(eta),  J_h = d_j s_ij R_ij psi(X_j,n) = s_ij R_ij X_j,n(eta);
                  only the diagonal entries H_gg, H_hh of the data term are kept, the gradient is complete
  :138            E_bnd = sum_(g,h) ((eta_g - eta_h) + Delta_gh)^2, E_prior = sum_g eta_g^2, lambda_smooth = lambda_prior = 1;
                  the boundary term is Jacobi-decoupled likewise (diagonal kept, gradient complete), H_prior = lambda_prior I
  :143            independent 1x1 damped Newton steps, damping lambda_lm = 0.05, clip |Delta eta| <= 0.5, anchor-keyframe
                  segments fixed, up to ten iterations

Readings:
  D1  "H_prior = lambda_prior I" fixes the convention E = sum rho(r) + (lambda_smooth / 2) E_bnd + (lambda_prior / 2) E_prior
      with rho(r) = r^2 / 2 inside the Huber band: gradient lambda_prior eta_g and lambda_smooth (eta_g - eta_h + Delta_gh).
  D2  the form of the damping is not stated: multiplicative as in Eq. (7), Delta eta_g = -g_g / ((1 + lambda_lm) H_gg).
      PARITY UNPINNED against the authors' code for this choice.
  D3  Huber kappa is not restated for Eq. (9): 1.345 on the whitened residual.
  D4  segment labels, the 4-adjacent pair list and Delta_gh are INPUTS (label < 0 = excluded pixel: low SLIC confidence or a
      segment below 16 valid pixels); a match counts when both its pixels carry a label and it is valid for the
      GN step (R12).  q_mn = sqrt(c_i c_j) (R5).
  D5  a segment no term touches has H_gg = lambda_prior > 0, so the step is always defined.

Pins (tests/test_oracle_depth.py): gradient against central differences of the total objective; H_gg against the second
difference of the objective at a zero-residual point; eta = 0 is a fixed point on clean data at the true poses; a known
per-segment scale error is recovered; monotone decrease of the objective; anchors and clip honoured.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Sequence, Tuple

import numpy as np

from oracle.sim3_gn_oracle import huber_rho, huber_weight, pose_to_srt, sim3_inv, sim3_mul, valid_matches


@dataclass
class DepthParams:
    sigma_point: float = 0.05
    huber_k: float = 1.345        # reading D3
    lambda_smooth: float = 1.0
    lambda_prior: float = 1.0
    lambda_lm: float = 0.05
    eta_max: float = 0.5
    conf_min: float = 0.0


def depth_terms(poses, points, conf, edges, match, labels, n_seg: int, eta, pairs, delta, prm: DepthParams
                ) -> Tuple[np.ndarray, np.ndarray, float]:
    """Gradient g [M], Jacobi diagonal H [M] and objective value at eta (M = N * n_seg, segment id = k * n_seg + label)."""
    M = poses.shape[0] * n_seg
    g, H, cost = np.zeros(M), np.zeros(M), 0.0
    for e in range(edges.shape[0]):
        i, j = int(edges[e, 0]), int(edges[e, 1])
        m, n = valid_matches(match[e], conf[i], conf[j], prm.conf_min)
        keep = (labels[i, m] >= 0) & (labels[j, n] >= 0)
        m, n = m[keep], n[keep]
        if m.size == 0:
            continue
        gi = i * n_seg + labels[i, m].astype(np.int64)
        hj = j * n_seg + labels[j, n].astype(np.int64)
        s, R, t = sim3_mul(sim3_inv(*pose_to_srt(poses[i])), pose_to_srt(poses[j]))      # T_ij
        Xi = np.exp(eta[gi])[:, None] * points[i, m].astype(np.float64)                  # Eq. (8)
        Xj = np.exp(eta[hj])[:, None] * points[j, n].astype(np.float64)
        Jh = s * Xj @ R.T                                                                # s_ij R_ij X_j(eta)
        res = Jh + t - Xi                                                                # T_ij X_j - X_i
        Jg = -Xi
        q = np.sqrt(conf[i, m].astype(np.float64) * conf[j, n].astype(np.float64))
        r = np.sqrt(q)[:, None] * res / prm.sigma_point                                  # Eq. (9)
        om = q[:, None] * huber_weight(r, prm.huber_k) / prm.sigma_point ** 2
        cost += float(np.sum(huber_rho(r, prm.huber_k)))
        np.add.at(g, gi, np.sum(om * Jg * res, axis=1))
        np.add.at(H, gi, np.sum(om * Jg * Jg, axis=1))
        np.add.at(g, hj, np.sum(om * Jh * res, axis=1))
        np.add.at(H, hj, np.sum(om * Jh * Jh, axis=1))
    for (a, b), d0 in zip(np.asarray(pairs).reshape(-1, 2), np.asarray(delta).reshape(-1)):   # boundary term, reading D1
        d = eta[a] - eta[b] + d0
        g[a] += prm.lambda_smooth * d
        g[b] -= prm.lambda_smooth * d
        H[a] += prm.lambda_smooth
        H[b] += prm.lambda_smooth
        cost += 0.5 * prm.lambda_smooth * d * d
    g += prm.lambda_prior * eta                                                           # prior term
    H += prm.lambda_prior
    cost += 0.5 * prm.lambda_prior * float(np.sum(eta * eta))
    return g, H, cost


def depth_step(poses, points, conf, edges, match, labels, n_seg, eta, pairs, delta, anchor_kf: Sequence[int], prm: DepthParams):
    """One Jacobi-decoupled damped Newton iteration (reading D2); returns (new eta, objective at the input eta)."""
    g, H, cost = depth_terms(poses, points, conf, edges, match, labels, n_seg, eta, pairs, delta, prm)
    step = -g / ((1.0 + prm.lambda_lm) * H)
    step = np.clip(step, -prm.eta_max, prm.eta_max)
    for k in anchor_kf:
        step[k * n_seg:(k + 1) * n_seg] = 0.0
    return eta + step, cost


def depth_refine(poses, points, conf, edges, match, labels, n_seg, eta0, pairs, delta, anchor_kf, prm: DepthParams, n_iters: int = 10):
    eta, costs = np.array(eta0, dtype=np.float64), []
    for _ in range(n_iters):
        eta, c = depth_step(poses, points, conf, edges, match, labels, n_seg, eta, pairs, delta, anchor_kf, prm)
        costs.append(c)
    return eta, np.asarray(costs)
