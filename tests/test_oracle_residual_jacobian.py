"""Pins of the oracle's residual (Eq. (1)), robust weights and analytic
Jacobians (Eq. (6)): hand-computed values, central finite differences through
scipy.linalg.expm, and the closed-form J_xi."""
import os

import numpy as np
import pytest
import scipy.linalg

from oracle import sim3_gn_oracle as orc
from tests.test_oracle_lie import gen4

GOLD = os.path.join(os.path.dirname(__file__), "golden", "residual_hand_case.txt")


def load_gold():
    out = {}
    with open(GOLD) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            out[k] = np.array([float(x) for x in v])
    return out


def pose(t, q, s):
    return np.array([*t, *q, s], dtype=float)


def test_hand_case_A():
    g = load_gold()
    Ti = pose([0, 0, 0], [0, 0, 0, 1], 1.0)
    Tj = pose([0, 0, 1], [0, 0, 0, 1], 2.0)
    Tij = orc.sim3_mul(orc.sim3_inv(*orc.pose_to_srt(Ti)), orc.pose_to_srt(Tj))
    e = orc.residual(Tij, np.array([[3.0, 0, 4.0]]), np.array([[0, 0, 2.0]]))
    assert np.allclose(e[0], g["A_e"], atol=1e-15)


def test_hand_case_B_full_chain():
    g = load_gold()
    c45 = np.sqrt(0.5)
    Ti = pose([1, 0, 0], [0, 0, c45, c45], 2.0)
    Tj = pose([1, 2, 0], [0, 0, 0, 1], 1.0)
    prm = orc.Params(sigma_ray=0.5, sigma_dist=2.0, huber_k=0.5)
    Xi = np.array([[0, -2.0, 0]], dtype=np.float32)
    Xj = np.array([[2.0, 0, 0]], dtype=np.float32)
    ci = np.array([0.64])
    cj = np.array([0.25])
    tm = orc.edge_terms(Ti, Tj, Xi, ci, Xj, cj, np.array([0], dtype=np.int32), prm)
    assert np.allclose(tm.e[0], g["B_e"], atol=1e-14)
    assert np.allclose(tm.r[0], g["B_r"], atol=1e-14)
    assert np.allclose(tm.omega[0], g["B_omega"], atol=1e-14)
    assert np.isclose(tm.cost, g["B_cost"][0], atol=1e-14)
    assert np.allclose(orc.huber_weight(tm.r[0], 0.5), g["B_w"], atol=1e-14)


def test_huber_kernel_values():
    k = 1.345
    r = np.array([0.0, 0.5, k, -k, 2 * k, -4 * k])
    assert np.allclose(orc.huber_weight(r, k), [1, 1, 1, 1, 0.5, 0.25])
    assert np.allclose(orc.huber_rho(r, k), [0, 0.125, 0.5 * k * k, 0.5 * k * k, 1.5 * k * k, 3.5 * k * k])
    # rho'(r) = w(r) r  (IRLS weight definition), checked by finite differences
    for x in (0.3, 1.0, 2.0, 5.0):
        d = (orc.huber_rho(np.array([x + 1e-6]), k) - orc.huber_rho(np.array([x - 1e-6]), k)) / 2e-6
        assert np.isclose(d[0], orc.huber_weight(np.array([x]), k)[0] * x, rtol=1e-6)


def _srt_from_4x4(T):
    M = T[:3, :3]
    s = np.cbrt(np.linalg.det(M))
    return float(s), M / s, T[:3, 3].copy()


def _res_under_perturbation(Ti4, Tj4, di, dj, Xi, Xj):
    Ti = scipy.linalg.expm(gen4(di)) @ Ti4
    Tj = scipy.linalg.expm(gen4(dj)) @ Tj4
    return orc.residual(_srt_from_4x4(np.linalg.inv(Ti) @ Tj), Xi, Xj)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_jacobians_vs_central_differences(seed):
    rng = np.random.default_rng(seed)
    M = 6
    qi, qj = rng.normal(size=4), rng.normal(size=4)
    Pi = pose(rng.normal(0, 1, 3), qi / np.linalg.norm(qi), np.exp(rng.normal(0, 0.3)))
    Pj = pose(rng.normal(0, 1, 3), qj / np.linalg.norm(qj), np.exp(rng.normal(0, 0.3)))
    Xi = rng.normal(0, 2, (M, 3)).astype(np.float32)
    Xj = rng.normal(0, 2, (M, 3)).astype(np.float32)
    c = np.ones(M)
    prm = orc.Params()
    tm = orc.edge_terms(Pi, Pj, Xi, c, Xj, c, np.arange(M, dtype=np.int32), prm)
    Ti4 = orc.sim3_matrix(*orc.pose_to_srt(Pi))
    Tj4 = orc.sim3_matrix(*orc.pose_to_srt(Pj))
    h = 1e-6
    Xi64, Xj64 = Xi.astype(float), Xj.astype(float)
    for k in range(7):
        d = np.zeros(7)
        d[k] = h
        z = np.zeros(7)
        fd_i = (_res_under_perturbation(Ti4, Tj4, d, z, Xi64, Xj64) -
                _res_under_perturbation(Ti4, Tj4, -d, z, Xi64, Xj64)) / (2 * h)
        fd_j = (_res_under_perturbation(Ti4, Tj4, z, d, Xi64, Xj64) -
                _res_under_perturbation(Ti4, Tj4, z, -d, Xi64, Xj64)) / (2 * h)
        scale = max(1.0, np.abs(tm.J_i).max())
        assert np.allclose(tm.J_i[:, :, k], fd_i, atol=2e-8 * scale), k
        assert np.allclose(tm.J_j[:, :, k], fd_j, atol=2e-8 * scale), k
    assert np.array_equal(tm.J_i, -tm.J_j)


def test_closed_form_J_xi():
    """J_xi = [[P, -[u]x, 0], [u^T, 0, d]], P = (I - u u^T)/d  (DESIGN.md formula card)."""
    rng = np.random.default_rng(5)
    M = 8
    qi, qj = rng.normal(size=4), rng.normal(size=4)
    Pi = pose(rng.normal(0, 1, 3), qi / np.linalg.norm(qi), 0.7)
    Pj = pose(rng.normal(0, 1, 3), qj / np.linalg.norm(qj), 1.9)
    Xi = rng.normal(0, 2, (M, 3)).astype(np.float32)
    Xj = rng.normal(0, 2, (M, 3)).astype(np.float32)
    c = np.ones(M)
    tm = orc.edge_terms(Pi, Pj, Xi, c, Xj, c, np.arange(M, dtype=np.int32), orc.Params())
    s, R, t = orc.sim3_mul(orc.sim3_inv(*orc.pose_to_srt(Pi)), orc.pose_to_srt(Pj))
    for m in range(M):
        x = s * R @ Xj[m].astype(float) + t
        d = np.linalg.norm(x)
        u = x / d
        ref = np.zeros((4, 7))
        ref[0:3, 0:3] = (np.eye(3) - np.outer(u, u)) / d
        ref[0:3, 3:6] = -np.array([[0, -u[2], u[1]], [u[2], 0, -u[0]], [-u[1], u[0], 0]])
        ref[3, 0:3] = u
        ref[3, 6] = d
        assert np.allclose(tm.J_xi[m], ref, atol=1e-13)


def test_validity_rule_and_checksum():
    HW = 10
    match = np.array([3, -1, 10, 0, 9, 2, 2, -5, 11, 4], dtype=np.int32)
    ci = np.array([1, 1, 1, 0, 1, 1, 0.2, 1, 1, 1.0])
    cj = np.array([1, 1, 0.1, 1, 1, 1, 1, 1, 1, 1.0])
    m, n = orc.valid_matches(match, ci, cj, 0.15)
    # m=0->3 ok; 1 invalid; 2->10 out of range; 3: c_i=0; 4->9 ok; 5->2: c_j[2]=0.1 no; 6->2 no; 7 neg; 8 oor; 9->4 ok
    assert m.tolist() == [0, 4, 9] and n.tolist() == [3, 9, 4]
