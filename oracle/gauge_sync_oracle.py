"""CPU float64 oracle of the gauge synchronisation of two map components (section III-C, lines 92-104,
Eq. (3)-(4)), written from the paper.  SURVEY section 8(f) NEXT-2.

TEST INFRASTRUCTURE ONLY (same rule as sim3_gn_oracle.py): only ``tests/`` may import it; it shares no code with the
CUDA path.

What it computes, in the paper's order:
  1. lift the matched canonical points of the linking edge (i, j) into the two world frames,
     x_l = T_WCi X_i[m], y_l = T_WCj X_j[n]
  2. (s*, R*, t*) = argmin sum_l |x_l - (s R y_l + t)|^2                            (Eq. (3))
     by Umeyama's closed form: centroids, centred points, A = (1/N_c) sum x~ y~^T = U Lambda V^T,
     S = diag(1, 1, det(U V^T)), R* = U S V^T, s* = tr(S Lambda) / ((1/N_c) sum |y~|^2),
     t* = x_bar - s* R* y_bar                                                       (Eq. (4))
  3. fewer than N_c^min = 64 correspondences: T* = T_WCi T_WCj^-1
  4. T* is left-multiplied onto every pose of the moving component

Readings: the match set is the valid set of the GN step (reading R12); the sum of Eq. (3) is
unweighted as printed; the moving component is the one of keyframe j (y side); ``moving_is_i=True`` swaps the roles
(the similarity then maps x onto y and the fallback is T_WCj T_WCi^-1); the SVD is numpy.linalg.svd (a library step).

Pins (tests/test_oracle_gauge_sync.py): exact recovery of a known similarity on clean points; the reflection case
(det = +1 enforced, cost not above any nearby rotation); stationarity of the Eq. (3) objective under Sim(3)
perturbations on noisy data; rotation against scipy.spatial.transform.Rotation.align_vectors; relative poses inside
the moving component unchanged; endpoint fallback below 64 correspondences.
"""
from __future__ import annotations

from typing import Sequence, Tuple

import numpy as np

from oracle.sim3_gn_oracle import pose_to_srt, sim3_inv, sim3_mul, srt_to_pose, valid_matches

N_C_MIN = 64


def umeyama(x: np.ndarray, y: np.ndarray) -> Tuple[float, np.ndarray, np.ndarray]:
    """Eq. (3)-(4): the similarity (s, R, t) with x ~ s R y + t, rows = correspondences."""
    n_c = x.shape[0]
    x_bar, y_bar = x.sum(axis=0) / n_c, y.sum(axis=0) / n_c
    xt, yt = x - x_bar, y - y_bar
    A = np.zeros((3, 3))
    for l in range(n_c) if n_c <= 256 else ():       # the definition, term by term, on small inputs
        A += np.outer(xt[l], yt[l])
    if n_c > 256:
        A = xt.T @ yt
    A /= n_c
    U, lam, Vt = np.linalg.svd(A)
    S = np.diag([1.0, 1.0, np.linalg.det(U @ Vt)])
    R = U @ S @ Vt
    var_y = np.sum(yt * yt) / n_c
    s = np.trace(S @ np.diag(lam)) / var_y
    t = x_bar - s * R @ y_bar
    return float(s), R, t


def link_points(poses: np.ndarray, points: np.ndarray, conf: np.ndarray, edge: Sequence[int], match_e: np.ndarray,
                conf_min: float):
    """World-frame lifts (x_l, y_l) of the valid matches of edge (i, j)."""
    i, j = int(edge[0]), int(edge[1])
    m, n = valid_matches(match_e, conf[i], conf[j], conf_min)
    si, Ri, ti = pose_to_srt(poses[i])
    sj, Rj, tj = pose_to_srt(poses[j])
    x = si * points[i, m].astype(np.float64) @ Ri.T + ti
    y = sj * points[j, n].astype(np.float64) @ Rj.T + tj
    return x, y


def gauge_sync(poses: np.ndarray, points: np.ndarray, conf: np.ndarray, edge: Sequence[int], match_e: np.ndarray,
               moving_kf: Sequence[int], conf_min: float = 0.0, moving_is_i: bool = False, n_c_min: int = N_C_MIN):
    """Returns (new poses, (s*, R*, t*), N_c)."""
    i, j = int(edge[0]), int(edge[1])
    x, y = link_points(poses, points, conf, edge, match_e, conf_min)
    n_c = x.shape[0]
    Ti, Tj = pose_to_srt(poses[i]), pose_to_srt(poses[j])
    if n_c >= n_c_min:
        T = umeyama(y, x) if moving_is_i else umeyama(x, y)
    else:
        T = sim3_mul(Tj, sim3_inv(*Ti)) if moving_is_i else sim3_mul(Ti, sim3_inv(*Tj))
    out = poses.copy()
    for k in moving_kf:
        out[k] = srt_to_pose(*sim3_mul(T, pose_to_srt(poses[k])))
    return out, T, n_c
