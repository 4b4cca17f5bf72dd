"""Pins of the oracle's roll-pitch-yaw residual variant (PAPER.md:L47, L115-117 read literally; NEXT-4 ii) -- CPU only."""
import numpy as np
from scipy.spatial.transform import Rotation

from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl


def test_rpy_matches_scipy_and_reconstructs_the_rotation():
    rng = np.random.default_rng(0)
    for R in Rotation.random(200, random_state=1).as_matrix():
        a = orc.rpy(R)
        assert np.allclose(a, Rotation.from_matrix(R).as_euler("xyz"), atol=1e-12)       # fixed-axis x-y-z = roll, pitch, yaw
        assert np.allclose(Rotation.from_euler("ZYX", a[::-1]).as_matrix(), R, atol=1e-12)  # R = Rz(yaw) Ry(pitch) Rx(roll)
    assert np.allclose(orc.rpy(np.eye(3)), 0)


def test_residual_is_the_wrapped_elementwise_difference():
    ch = wl.panda_chain()
    rng = np.random.default_rng(2)
    for _ in range(50):
        q = 0.5 * (ch.q_lo + ch.q_hi) + 0.4 * (ch.q_hi - ch.q_lo) * rng.uniform(-1, 1, 7)
        p, R = orc.fk(ch, q)
        Rt = Rotation.random(random_state=int(rng.integers(1 << 30)))
        xyzw = Rt.as_quat()
        tq = np.r_[xyzw[3], xyzw[:3]]
        tp = rng.normal(size=3)
        r = orc.residual_rpy(p, R, tp, tq, 2.0, 0.5)
        d = Rotation.from_matrix(R).as_euler("xyz") - Rt.as_euler("xyz")
        d = (d + np.pi) % (2 * np.pi) - np.pi
        assert np.allclose(r[:3], 2.0 * (p - tp), atol=1e-14)
        assert np.allclose(np.abs(r[3:]), 0.5 * np.abs(d), atol=1e-12)
        assert np.all(np.abs(r[3:]) <= 0.5 * np.pi + 1e-12)
    # same pose -> zero; a pure yaw offset shows up in the yaw row only
    p, R = orc.fk(ch, 0.5 * (ch.q_lo + ch.q_hi))
    xyzw = Rotation.from_matrix(R).as_quat()
    assert np.abs(orc.residual_rpy(p, R, p, np.r_[xyzw[3], xyzw[:3]])).max() < 1e-12
    xyzw = (Rotation.from_euler("z", -0.3) * Rotation.from_matrix(R)).as_quat()
    r = orc.residual_rpy(p, R, p, np.r_[xyzw[3], xyzw[:3]])
    assert np.allclose(r, [0, 0, 0, 0, 0, 0.3], atol=1e-12)


def test_jacobian_is_the_exact_derivative_of_the_rpy_residual():
    for ch in (wl.panda_chain(), wl.random_chain_8dof(3)):
        rng = np.random.default_rng(3)
        for _ in range(20):
            q = 0.5 * (ch.q_lo + ch.q_hi) + 0.3 * (ch.q_hi - ch.q_lo) * rng.uniform(-1, 1, ch.dof)
            p, R = orc.fk(ch, q)
            if abs(orc.rpy(R)[1]) > 1.4:
                continue                                       # near the pitch singularity E is ill-conditioned
            tq = np.array([0.9, 0.1, -0.3, 0.2])
            tp = np.zeros(3)
            J = orc.jacobian_rpy(ch, q)
            h = 1e-6
            F = np.zeros_like(J)
            for j in range(ch.dof):
                e = np.zeros(ch.dof)
                e[j] = h
                pp, Rp = orc.fk(ch, q + e)
                pm, Rm = orc.fk(ch, q - e)
                F[:, j] = (orc.residual_rpy(pp, Rp, tp, tq) - orc.residual_rpy(pm, Rm, tp, tq)) / (2 * h)
            assert np.abs(J - F).max() < 1e-7                 # exact, also away from r = 0 (unlike the rotation-vector reading)


def test_lm_with_the_rpy_residual_converges_to_the_same_pose():
    ch = wl.panda_chain()
    rng = np.random.default_rng(4)
    truth = wl.smooth_joint_paths(ch, 1, 120, 3, 0.3, rng)[0]
    p, R = orc.fk(ch, truth)
    tq = wl._R_to_quat_wxyz(R)
    seeds = np.clip(truth + 0.05 * rng.normal(size=truth.shape), ch.q_lo, ch.q_hi)
    st = orc.lm_run(ch, orc.Params(tol=0.0, rot_mode=1), p, tq, seeds, 10)
    free = (st.status & 16) == 0
    assert free.mean() > 0.9 and st.res_norm[free].max() < 1e-11
    # the pose it reaches is the target pose whatever the residual parametrisation
    pr, Rr = orc.fk(ch, st.q)
    assert np.abs(pr - p)[free].max() < 1e-11 and np.abs(Rr - R)[free].max() < 1e-10
    # and rot_mode = 0 is untouched by the new field
    a = orc.lm_run(ch, orc.Params(tol=0.0), p, tq, seeds, 5)
    b = orc.lm_run(ch, orc.Params(tol=0.0, rot_mode=0), p, tq, seeds, 5)
    assert np.array_equal(a.q, b.q)
