"""Pins of the oracle's Sim(3) tangent-space operations against things other than
itself: scipy.linalg.expm of the 4x4 generator, group identities, and limits."""
import numpy as np
import pytest
import scipy.linalg

from oracle import sim3_gn_oracle as orc


def gen4(tau):
    """4x4 generator tau^ = [[ [w]x + zeta I, v ], [0, 0]] typed out independently."""
    v, w, z = tau[0:3], tau[3:6], tau[6]
    G = np.zeros((4, 4))
    G[0, 1], G[0, 2] = -w[2], w[1]
    G[1, 0], G[1, 2] = w[2], -w[0]
    G[2, 0], G[2, 1] = -w[1], w[0]
    G[0, 0] = G[1, 1] = G[2, 2] = z
    G[:3, 3] = v
    return G


def rand_tau(rng, scale_w=1.0, scale_z=1.0):
    return np.concatenate([rng.normal(0, 1, 3), rng.normal(0, scale_w, 3), [rng.normal(0, scale_z)]])


@pytest.mark.parametrize("sw,sz", [(1.0, 0.5), (1e-3, 1e-3), (1e-7, 0.3), (0.7, 1e-8), (1e-9, 1e-9),
                                   (0.0, 0.0), (2.0, 2.0), (0.3, 2.5), (1e-2, 1e-2)])
def test_exp_matches_expm(sw, sz):
    rng = np.random.default_rng(11)
    for _ in range(40):
        tau = rand_tau(rng, sw, sz)
        th = np.linalg.norm(tau[3:6])
        if th > 3.0:
            tau[3:6] *= 3.0 / th
        T = orc.sim3_matrix(*orc.sim3_exp(tau))
        ref = scipy.linalg.expm(gen4(tau))
        assert np.allclose(T, ref, rtol=0, atol=5e-14 * max(1.0, np.abs(ref).max()))


def test_exp_zero_is_identity():
    s, R, t = orc.sim3_exp(np.zeros(7))
    assert s == 1.0 and np.array_equal(R, np.eye(3)) and np.array_equal(t, np.zeros(3))


def test_exp_inverse():
    rng = np.random.default_rng(1)
    for _ in range(50):
        tau = rand_tau(rng, 0.8, 0.4)
        P = orc.sim3_matrix(*orc.sim3_exp(tau)) @ orc.sim3_matrix(*orc.sim3_exp(-tau))
        assert np.allclose(P, np.eye(4), atol=1e-13)


def test_log_exp_roundtrip():
    rng = np.random.default_rng(2)
    for sc in (1.0, 1e-3, 1e-8):
        for _ in range(50):
            tau = rand_tau(rng, sc, sc)
            th = np.linalg.norm(tau[3:6])
            if th > 3.0:
                tau[3:6] *= 3.0 / th
            back = orc.sim3_log(*orc.sim3_exp(tau))
            assert np.allclose(back, tau, rtol=1e-9, atol=1e-13)


def test_exp_log_roundtrip_on_group():
    rng = np.random.default_rng(3)
    for _ in range(50):
        q = rng.normal(size=4)
        pose = np.concatenate([rng.normal(0, 2, 3), q / np.linalg.norm(q), [np.exp(rng.normal(0, 0.5))]])
        s, R, t = orc.pose_to_srt(pose)
        s2, R2, t2 = orc.sim3_exp(orc.sim3_log(s, R, t))
        assert np.isclose(s, s2, rtol=1e-12) and np.allclose(R, R2, atol=1e-12) and np.allclose(t, t2, atol=1e-11)


def test_adjoint_identity():
    """T Exp(tau) T^-1 = Exp(Ad_T tau), checked through expm."""
    rng = np.random.default_rng(4)
    for _ in range(40):
        q = rng.normal(size=4)
        pose = np.concatenate([rng.normal(0, 2, 3), q / np.linalg.norm(q), [np.exp(rng.normal(0, 0.5))]])
        T = orc.pose_to_srt(pose)
        T4 = orc.sim3_matrix(*T)
        tau = rand_tau(rng, 0.5, 0.3)
        lhs = T4 @ scipy.linalg.expm(gen4(tau)) @ np.linalg.inv(T4)
        rhs = scipy.linalg.expm(gen4(orc.sim3_adjoint(*T) @ tau))
        assert np.allclose(lhs, rhs, atol=1e-11 * max(1.0, np.abs(lhs).max()))


def test_adjoint_of_inverse_is_inverse_adjoint():
    rng = np.random.default_rng(5)
    q = rng.normal(size=4)
    pose = np.concatenate([rng.normal(0, 2, 3), q / np.linalg.norm(q), [1.7]])
    T = orc.pose_to_srt(pose)
    A = orc.sim3_adjoint(*T)
    Ai = orc.sim3_adjoint(*orc.sim3_inv(*T))
    assert np.allclose(A @ Ai, np.eye(7), atol=1e-12)
    # the printed block form of Ad_{T^-1}: [[R^T/s, -R^T [t]x / s, R^T t / s], [0, R^T, 0], [0, 0, 1]]
    s, R, t = T
    ref = np.zeros((7, 7))
    ref[0:3, 0:3] = R.T / s
    ref[0:3, 3:6] = -R.T @ _skew(t) / s
    ref[0:3, 6] = R.T @ t / s
    ref[3:6, 3:6] = R.T
    ref[6, 6] = 1.0
    assert np.allclose(Ai, ref, atol=1e-12)


def _skew(t):
    return np.array([[0, -t[2], t[1]], [t[2], 0, -t[0]], [-t[1], t[0], 0]])


def test_quaternion_rotation_roundtrip_and_inverse_composition():
    rng = np.random.default_rng(6)
    for _ in range(100):
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        R = orc.quat_to_rot(q)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-14) and np.isclose(np.linalg.det(R), 1.0)
        q2 = orc.rot_to_quat(R)
        assert np.allclose(q2, q if q[3] >= 0 else -q, atol=1e-12)
    # Rz(90 deg): x -> y
    R = orc.quat_to_rot(np.array([0, 0, np.sin(np.pi / 4), np.cos(np.pi / 4)]))
    assert np.allclose(R @ [1, 0, 0], [0, 1, 0], atol=1e-15)


def test_sim3_mul_inv_match_4x4():
    rng = np.random.default_rng(7)
    ps = []
    for _ in range(2):
        q = rng.normal(size=4)
        ps.append(orc.pose_to_srt(np.concatenate([rng.normal(0, 2, 3), q / np.linalg.norm(q), [np.exp(rng.normal())]])))
    A, B = (orc.sim3_matrix(*p) for p in ps)
    assert np.allclose(orc.sim3_matrix(*orc.sim3_mul(ps[0], ps[1])), A @ B, atol=1e-12)
    assert np.allclose(orc.sim3_matrix(*orc.sim3_inv(*ps[0])), np.linalg.inv(A), atol=1e-12)


def test_retract_matches_expm():
    rng = np.random.default_rng(8)
    q = rng.normal(size=(3, 4))
    poses = np.concatenate([rng.normal(0, 2, (3, 3)), q / np.linalg.norm(q, axis=1, keepdims=True),
                            np.exp(rng.normal(0, 0.3, (3, 1)))], axis=1)
    tau = rng.normal(0, 0.2, 21)
    out = orc.retract(poses, tau)
    for k in range(3):
        ref = scipy.linalg.expm(gen4(tau[7 * k:7 * k + 7])) @ orc.sim3_matrix(*orc.pose_to_srt(poses[k]))
        assert np.allclose(orc.sim3_matrix(*orc.pose_to_srt(out[k])), ref, atol=1e-12)
        assert np.isclose(np.linalg.norm(out[k, 3:7]), 1.0, atol=1e-15)
