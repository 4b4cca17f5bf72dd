"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

Each pin checks the oracle against something OTHER than itself: a closed form, a library
routine, finite differences, a textbook identity, or a limit.  P-numbers follow DESIGN.md.
"""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl

PI = np.pi


def make_chain(a, alpha, d, theta=None, jt=None, lo=-10.0, hi=10.0, tool=(0, 0, 0, 1, 0, 0, 0)):
    n = len(a)
    return wl.Chain(name="t", dof=n, joint_type=np.zeros(n, np.int32) if jt is None else np.array(jt, np.int32),
                    a=np.array(a, float), alpha=np.array(alpha, float), d=np.array(d, float),
                    theta=np.zeros(n) if theta is None else np.array(theta, float),
                    q_lo=np.full(n, lo), q_hi=np.full(n, hi), tool=np.array(tool, float))


def rand_q(ch, rng, frac=1.0):
    mid, half = 0.5 * (ch.q_lo + ch.q_hi), 0.5 * (ch.q_hi - ch.q_lo)
    return mid + frac * half * rng.uniform(-1, 1, ch.dof)


# ------------------------------------------------------------------ P1: FK closed forms

def test_p1_panda_zero_pose_golden():
    """Panda DH at q = 0: flange at (0.088, 0, 0.926) m, R = diag(1, -1, -1) -- closed form of the
    table (tests/golden/panda_zero_pose.txt)."""
    import os
    g = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "panda_zero_pose.txt"), comments="#")
    p, R = orc.fk(wl.panda_chain(), np.zeros(7))
    assert np.allclose(p, g[0], atol=1e-12)
    assert np.allclose(R, g[1:4], atol=1e-12)


def test_p1_identity_chain_is_rot_z_of_sum():
    rng = np.random.default_rng(0)
    ch = make_chain([0] * 5, [0] * 5, [0] * 5)
    q = rng.uniform(-3, 3, 5)
    p, R = orc.fk(ch, q)
    assert np.allclose(p, 0, atol=1e-12)
    assert np.allclose(R, Rotation.from_euler("z", q.sum()).as_matrix(), atol=1e-12)


def test_p1_planar_chain_closed_form():
    """k-R planar arm: frame j sits at the END of link j-1 (a_{j-1} = L_{j-1}); the tool carries
    the last link.  x = sum L_i cos(sum_{k<=i} q_k), y likewise with sin."""
    rng = np.random.default_rng(1)
    L = rng.uniform(0.1, 0.5, 4)
    ch = make_chain([0, L[0], L[1], L[2]], [0] * 4, [0] * 4, tool=(L[3], 0, 0, 1, 0, 0, 0))
    for _ in range(20):
        q = rng.uniform(-3, 3, 4)
        cs = np.cumsum(q)
        p, R = orc.fk(ch, q)
        assert np.allclose(p, [np.sum(L * np.cos(cs)), np.sum(L * np.sin(cs)), 0], atol=1e-12)
        assert np.allclose(R, Rotation.from_euler("z", cs[-1]).as_matrix(), atol=1e-12)


def test_p1_single_prismatic_and_alpha():
    ch = make_chain([0], [0], [0], jt=[1])
    p, R = orc.fk(ch, np.array([0.37]))
    assert np.allclose(p, [0, 0, 0.37], atol=1e-15) and np.allclose(R, np.eye(3), atol=1e-15)
    # alpha = +pi/2 about x turns the joint's z axis onto world -y (Craig: Rot_x(alpha) z = (0,-s,c))
    ch = make_chain([0.2], [PI / 2], [0], jt=[1])
    p, _ = orc.fk(ch, np.array([0.5]))
    assert np.allclose(p, [0.2, -0.5, 0], atol=1e-12)
    # theta offset on a revolute joint and d along the rotated z
    ch = make_chain([0], [0], [0.3], theta=[PI / 2], tool=(1, 0, 0, 1, 0, 0, 0))
    p, _ = orc.fk(ch, np.array([0.0]))
    assert np.allclose(p, [0, 1, 0.3], atol=1e-12)


def test_p1_rotation_orthonormal_periodic_and_tool():
    rng = np.random.default_rng(2)
    for ch in (wl.panda_chain(), wl.random_chain_8dof(3)):
        for _ in range(20):
            q = rand_q(ch, rng)
            p, R = orc.fk(ch, q)
            assert np.allclose(R.T @ R, np.eye(3), atol=1e-12)
            assert abs(np.linalg.det(R) - 1) < 1e-12
            for j in np.nonzero(ch.joint_type == 0)[0]:
                q2 = q.copy()
                q2[j] += 2 * PI
                p2, R2 = orc.fk(ch, q2)
                assert np.allclose(p2, p, atol=1e-12) and np.allclose(R2, R, atol=1e-12)
    # a rotated tool: FK with tool == FK without tool composed with the tool by hand
    ch = wl.panda_chain()
    q = rand_q(ch, rng)
    ch0 = wl.panda_chain()
    ch0.tool = np.array([0, 0, 0, 1, 0, 0, 0.0])
    tq = Rotation.from_rotvec([0.3, -0.2, 0.9])
    ch.tool = np.concatenate([[0.01, 0.02, 0.107], tq.as_quat()[[3, 0, 1, 2]]])
    p0, R0 = orc.fk(ch0, q)
    p1, R1 = orc.fk(ch, q)
    assert np.allclose(p1, p0 + R0 @ ch.tool[:3], atol=1e-12)
    assert np.allclose(R1, R0 @ tq.as_matrix(), atol=1e-12)


def test_p1_axes_are_frame_columns():
    """z_j, o_j: joint j's axis passes through o_j; moving only joint j rotates the flange about it."""
    rng = np.random.default_rng(3)
    ch = wl.panda_chain()
    q = rand_q(ch, rng)
    p, R, z, o = orc.fk_axes(ch, q)
    assert np.allclose(np.linalg.norm(z, axis=1), 1, atol=1e-12)
    for j in range(7):
        dq = 0.37
        q2 = q.copy()
        q2[j] += dq
        p2, R2 = orc.fk(ch, q2)
        Rj = Rotation.from_rotvec(dq * z[j]).as_matrix()
        assert np.allclose(p2, o[j] + Rj @ (p - o[j]), atol=1e-12)
        assert np.allclose(R2, Rj @ R, atol=1e-12)


# ------------------------------------------------------------------ P2: Log map / residual

def test_p2_log_matches_scipy_and_geodesic():
    rng = np.random.default_rng(4)
    for _ in range(300):
        w = rng.normal(size=3)
        w *= rng.uniform(0, PI - 0.01) / np.linalg.norm(w)
        E = Rotation.from_rotvec(w).as_matrix()
        got = orc.log_so3(E)
        assert np.allclose(got, w, atol=1e-12)                                  # round trip
        assert np.allclose(got, Rotation.from_matrix(E).as_rotvec(), atol=1e-12)  # library routine
        assert abs(np.linalg.norm(got) - np.arccos(np.clip((np.trace(E) - 1) / 2, -1, 1))) < 1e-7


def test_p2_log_small_angle_branch_is_continuous():
    axis = np.array([0.6, -0.48, 0.64])
    for ang in (0.0, 1e-9, 1e-6, 0.99e-4, 1.01e-4, 1e-3):
        E = Rotation.from_rotvec(ang * axis).as_matrix()
        assert np.allclose(orc.log_so3(E), ang * axis, atol=1e-15 + 1e-12 * ang)


def test_p2_log_near_pi_reproduces_the_rotation():
    rng = np.random.default_rng(5)
    for eps in (0.0, 1e-9, 1e-6, 5e-5, 2e-4, 1e-3):
        for _ in range(10):
            a = rng.normal(size=3)
            a /= np.linalg.norm(a)
            E = Rotation.from_rotvec((PI - eps) * a).as_matrix()
            w = orc.log_so3(E)
            assert abs(np.linalg.norm(w) - (PI - eps)) < 1e-6
            assert np.allclose(Rotation.from_rotvec(w).as_matrix(), E, atol=2e-8)


def test_p2_residual_definition():
    """r = [p - p_t ; Log(R R_t^T)]: zero at the target, position part linear, rotation part equal
    to the world-frame rotation vector taking the target orientation to the current one, and
    independent of the quaternion's sign and scale (DESIGN R11)."""
    rng = np.random.default_rng(6)
    for _ in range(50):
        Rt = Rotation.random(random_state=rng.integers(1 << 30))
        w = rng.normal(size=3) * 0.5
        R = (Rotation.from_rotvec(w) * Rt).as_matrix()
        tq = Rt.as_quat()[[3, 0, 1, 2]]
        tp = rng.normal(size=3)
        p = tp + rng.normal(size=3) * 0.1
        r = orc.residual(p, R, tp, tq)
        assert np.allclose(r[:3], p - tp, atol=1e-15)
        assert np.allclose(r[3:], w, atol=1e-12)
        assert np.allclose(orc.residual(p, R, tp, -2.5 * tq), r, atol=1e-12)
        assert np.allclose(orc.residual(tp, Rt.as_matrix(), tp, tq), 0, atol=1e-15)
        r2 = orc.residual(p, R, tp, tq, w_pos=2.0, w_rot=0.5)
        assert np.allclose(r2, np.concatenate([2 * r[:3], 0.5 * r[3:]]), atol=1e-15)


def test_quat_to_R_matches_scipy():
    rng = np.random.default_rng(7)
    for _ in range(50):
        q = rng.normal(size=4)
        assert np.allclose(orc.quat_to_R(q), Rotation.from_quat(q[[1, 2, 3, 0]]).as_matrix(), atol=1e-13)


# ------------------------------------------------------------------ P3: Jacobian

def fd_jacobian(ch, q, h=1e-5):
    J = np.zeros((6, ch.dof))
    _, R = orc.fk(ch, q)
    for j in range(ch.dof):
        e = np.zeros(ch.dof)
        e[j] = h
        pp, Rp = orc.fk(ch, q + e)
        pm, Rm = orc.fk(ch, q - e)
        J[:3, j] = (pp - pm) / (2 * h)
        S = ((Rp - Rm) / (2 * h)) @ R.T  # [omega]_x
        J[3:, j] = [S[2, 1] - S[1, 2], S[0, 2] - S[2, 0], S[1, 0] - S[0, 1]]
        J[3:, j] *= 0.5
    return J


@pytest.mark.parametrize("which", ["panda", "rand8"])
def test_p3_jacobian_vs_finite_differences(which):
    rng = np.random.default_rng(8)
    ch = wl.panda_chain() if which == "panda" else wl.random_chain_8dof(3)
    worst = 0.0
    for _ in range(200):
        q = rand_q(ch, rng)
        J = orc.jacobian(ch, q)
        worst = max(worst, np.abs(J - fd_jacobian(ch, q)).max())
        for j in range(ch.dof):
            assert abs(np.linalg.norm(J[3:, j]) - (0.0 if ch.joint_type[j] else 1.0)) < 1e-12
    assert worst < 1e-7  # BASELINE.json north_star: "finite-difference Jacobian to 1e-7"


def test_p3_planar_jacobian_closed_form():
    rng = np.random.default_rng(9)
    L = np.array([0.3, 0.25, 0.2])
    ch = make_chain([0, L[0], L[1]], [0] * 3, [0] * 3, tool=(L[2], 0, 0, 1, 0, 0, 0))
    q = rng.uniform(-2, 2, 3)
    cs = np.cumsum(q)
    J = orc.jacobian(ch, q)
    for j in range(3):
        assert np.isclose(J[0, j], -np.sum(L[j:] * np.sin(cs[j:])), atol=1e-12)
        assert np.isclose(J[1, j], np.sum(L[j:] * np.cos(cs[j:])), atol=1e-12)
    assert np.allclose(J[2], 0) and np.allclose(J[3:5], 0) and np.allclose(J[5], 1)


def test_p4_residual_linearisation_order():
    """r(q+e) - r(q) - J e = O(|e|^2) when r_rot = 0 (DESIGN R2/R3): slope >= 1.9 on log-log."""
    rng = np.random.default_rng(10)
    ch = wl.panda_chain()
    q = rand_q(ch, rng, 0.6)
    p, R = orc.fk(ch, q)
    tq = Rotation.from_matrix(R).as_quat()[[3, 0, 1, 2]]
    J = orc.jacobian(ch, q)
    u = rng.normal(size=7)
    u /= np.linalg.norm(u)
    hs = np.array([1e-1, 1e-2, 1e-3])
    errs = []
    for h in hs:
        p2, R2 = orc.fk(ch, q + h * u)
        errs.append(np.linalg.norm(orc.residual(p2, R2, p, tq) - J @ (h * u)))
    slopes = np.diff(np.log(errs)) / np.diff(np.log(hs))
    assert np.all(slopes > 1.9), slopes


# ------------------------------------------------------------------ P5-P7: normal equations

def test_p5_solve_is_ridge_regression_and_dual_form():
    rng = np.random.default_rng(11)
    for ch in (wl.panda_chain(), wl.random_chain_8dof(3)):
        n = ch.dof
        for lam in (1e-4, 1e-3, 1e-1, 10.0):
            q = rand_q(ch, rng, 0.7)
            J = orc.jacobian(ch, q)
            r = rng.normal(size=6) * 0.1
            delta = orc.lm_delta(J, r, lam)
            A = J.T @ J + lam * np.eye(n)
            assert np.linalg.norm(A @ delta + J.T @ r) <= 1e-12 * np.linalg.norm(J.T @ r)
            # augmented least squares [J; sqrt(lam) I] delta = -[r; 0] via QR/SVD: never forms J^T J
            aug = np.vstack([J, np.sqrt(lam) * np.eye(n)])
            ref = np.linalg.lstsq(aug, -np.concatenate([r, np.zeros(n)]), rcond=None)[0]
            assert np.allclose(delta, ref, atol=1e-10 * max(1.0, np.abs(ref).max()))
            dual = -J.T @ np.linalg.solve(J @ J.T + lam * np.eye(6), r)
            assert np.allclose(delta, dual, atol=1e-10 * max(1.0, np.abs(dual).max()))


def test_lu_solve_pivots():
    A = np.array([[0.0, 2.0, 1.0], [1.0, 0.0, 3.0], [4.0, 1.0, 0.0]])  # zero leading pivot
    b = np.array([1.0, 2.0, 3.0])
    assert np.allclose(orc.lu_solve(A, b), np.linalg.solve(A, b), atol=1e-14)
    with pytest.raises(np.linalg.LinAlgError):
        orc.lu_solve(np.zeros((3, 3)), b)


def test_p6_lambda_to_infinity_is_scaled_gradient_descent():
    rng = np.random.default_rng(12)
    ch = wl.panda_chain()
    J = orc.jacobian(ch, rand_q(ch, rng, 0.7))
    r = rng.normal(size=6) * 0.1
    g = J.T @ r
    for lam in (1e6, 1e8, 1e10):
        delta = orc.lm_delta(J, r, lam)
        rel = np.linalg.norm(lam * delta + g) / np.linalg.norm(g)
        assert rel <= 10 * np.linalg.norm(J, 2) ** 2 / lam


def test_p7_lambda_to_zero_is_newton_on_square_system():
    rng = np.random.default_rng(13)
    ch = wl.panda_chain()
    J = orc.jacobian(ch, rand_q(ch, rng, 0.5))[:, [0, 1, 2, 3, 4, 5]]  # joint 7 locked
    r = rng.normal(size=6) * 0.01
    delta = orc.lm_delta(J, r, 1e-12)
    assert np.allclose(delta, -np.linalg.solve(J, r), atol=1e-8)
