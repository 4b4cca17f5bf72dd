"""Pins of the trajectory-level oracle (oracle/lm_traj_oracle.c) -- CPU only.

The stacked residual r = [w_pose r_pose ; w_diff (q_{k+1} - q_k)] (Fig. 6), its
Jacobian and the LM update are checked against things other
than the oracle itself: hand-made closed forms, finite differences, numpy's least-squares solution
of the augmented system (never forms J^T J), scipy's banded solver on the second-difference
matrix, the per-waypoint oracle (already pinned by test_oracle_pins.py) and limits in lambda.
"""
import numpy as np
import pytest
from scipy.linalg import solveh_banded

from oracle import lm_oracle as orc
from oracle import lm_traj_oracle as torc
from paper_2309_09102_b200 import workloads as wl


def problem(ch, n, sigma, seed, B=1, amp=0.3):
    """B trajectories of n waypoints: targets = FK(smooth truth), q0 = truth + noise (fp64)."""
    rng = np.random.default_rng(seed)
    truth = wl.smooth_joint_paths(ch, B, n, 3, amp, rng)
    p, R = orc.fk(ch, truth.reshape(-1, ch.dof))
    tq = wl._R_to_quat_wxyz(R)
    q0 = np.clip(truth + sigma * rng.normal(size=truth.shape) * np.where(ch.joint_type == 1, 0.1, 1.0),
                 ch.q_lo, ch.q_hi)
    return truth, p.reshape(B, n, 3), tq.reshape(B, n, 4), q0


CHAINS = [wl.panda_chain(), wl.random_chain_8dof(3)]


def test_residual_layout_and_closed_forms():
    ch = wl.panda_chain()
    d, n = ch.dof, 9
    _, tp, tq, q0 = problem(ch, n, 0.05, 1)
    pp = orc.Params(w_pos=2.0, w_rot=0.5)
    tprm = torc.TrajParams(w_pose=3.0, w_diff=0.25)
    r = torc.residual(ch, pp, tprm, tp[0], tq[0], q0[0])
    assert r.shape == (6 * n + d * (n - 1),) and torc.rows(d, n) == r.size
    # pose rows: the per-waypoint residual (pinned by test_oracle_pins) times w_pose
    p, R = orc.fk(ch, q0[0])
    for i in range(n):
        ri = orc.residual(p[i], R[i], tp[0, i], tq[0, i], 2.0, 0.5)
        assert np.allclose(r[6 * i:6 * i + 6], 3.0 * ri, rtol=0, atol=1e-15)
    # differencing rows: w_diff (q_{k+1} - q_k), PAPER.md:L123 -- on a linear ramp every row equals the slope
    mid = 0.5 * (ch.q_lo + ch.q_hi)
    slope = np.linspace(-0.01, 0.02, d)
    ramp = mid[None, :] + np.arange(n)[:, None] * slope[None, :]
    r = torc.residual(ch, pp, tprm, tp[0], tq[0], ramp)
    assert np.allclose(r[6 * n:].reshape(n - 1, d), 0.25 * slope[None, :], atol=1e-15)
    # n = 1: no differencing rows
    assert torc.residual(ch, pp, tprm, tp[0, :1], tq[0, :1], q0[0, :1]).shape == (6,)


@pytest.mark.parametrize("ch", CHAINS, ids=lambda c: c.name)
def test_jacobian_against_finite_differences(ch):
    d, n = ch.dof, 6
    truth, tp, tq, q0 = problem(ch, n, 0.05, 2)
    pp = orc.Params(w_pos=1.5, w_rot=0.7)
    tprm = torc.TrajParams(w_pose=2.0, w_diff=0.3)

    def fd(q, h=1e-6):
        cols = []
        for u in range(n * d):
            e = np.zeros(n * d)
            e[u] = h
            rp = torc.residual(ch, pp, tprm, tp[0], tq[0], (q.ravel() + e).reshape(n, d))
            rm = torc.residual(ch, pp, tprm, tp[0], tq[0], (q.ravel() - e).reshape(n, d))
            cols.append((rp - rm) / (2 * h))
        return np.stack(cols, axis=1)

    # at zero rotational residual the geometric Jacobian IS the derivative of the residual (DESIGN R2/R3)
    J = torc.jacobian(ch, pp, tprm, truth[0])
    assert J.shape == (6 * n + d * (n - 1), n * d)
    assert np.abs(J - fd(truth[0])).max() < 1e-7
    # away from it: position rows and differencing rows are exact derivatives, rotation rows agree
    # to O(|r_rot|) (the J_l^-1 factor the method drops on purpose)
    J = torc.jacobian(ch, pp, tprm, q0[0])
    F = fd(q0[0])
    rot = np.zeros(J.shape[0], bool)
    for i in range(n):
        rot[6 * i + 3:6 * i + 6] = True
    assert np.abs(J[~rot] - F[~rot]).max() < 1e-7
    assert np.abs(J[rot] - F[rot]).max() < 0.2
    # structure: "identity for q_{i+1}, negated identity for q_i"; nothing else off the blocks
    D = J[6 * n:]
    for k in range(n - 1):
        blk = D[d * k:d * k + d]
        assert np.array_equal(blk[:, d * k:d * k + d], -0.3 * np.eye(d))
        assert np.array_equal(blk[:, d * (k + 1):d * (k + 2)], 0.3 * np.eye(d))
        assert np.count_nonzero(blk) == 2 * d
    for i in range(n):
        blk = J[6 * i:6 * i + 6].copy()
        blk[:, d * i:d * i + d] = 0
        assert not blk.any()


@pytest.mark.parametrize("ch", CHAINS, ids=lambda c: c.name)
@pytest.mark.parametrize("weights", [(1.0, 1.0), (1.0, 0.1), (0.0, 1.0), (2.0, 0.0)])
def test_delta_is_the_damped_least_squares_solution(ch, weights):
    """delta = argmin |J x + r|^2 + lam |x|^2, via numpy lstsq on [J; sqrt(lam) I] (never forms J^T J);
    the dense-LU and the banded-Cholesky oracle paths agree with it and with each other."""
    d, n = ch.dof, 7
    _, tp, tq, q0 = problem(ch, n, 0.1, 3)
    pp = orc.Params()
    tprm = torc.TrajParams(w_pose=weights[0], w_diff=weights[1])
    for lam in (1e-4, 1e-2, 1.0):
        J = torc.jacobian(ch, pp, tprm, q0[0])
        r = torc.residual(ch, pp, tprm, tp[0], tq[0], q0[0])
        aug = np.vstack([J, np.sqrt(lam) * np.eye(n * d)])
        rhs = -np.concatenate([r, np.zeros(n * d)])
        x = np.linalg.lstsq(aug, rhs, rcond=None)[0].reshape(n, d)
        dd = torc.delta(ch, pp, tprm, tp[0], tq[0], q0[0], lam, dense=True)
        db = torc.delta(ch, pp, tprm, tp[0], tq[0], q0[0], lam, dense=False)
        assert np.abs(dd - x).max() < 1e-9 * max(1.0, np.abs(x).max() / lam * 1e-3 + 1)
        assert np.abs(db - dd).max() < 1e-10 * max(1.0, np.abs(dd).max())
        # normal-equation residual
        A = J.T @ J + lam * np.eye(n * d)
        assert np.linalg.norm(A @ db.ravel() + J.T @ r) <= 1e-10 * max(np.linalg.norm(J.T @ r), 1e-12)


def test_banded_equals_dense_over_sizes():
    pp = orc.Params(w_pos=1.0, w_rot=0.8)
    for ch in CHAINS:
        for n in (1, 2, 3, 12, 25):
            _, tp, tq, q0 = problem(ch, n, 0.1, 10 + n)
            for wts, lam in (((1.0, 1.0), 1e-3), ((1.0, 0.05), 1e-4), ((0.5, 3.0), 10.0)):
                tprm = torc.TrajParams(w_pose=wts[0], w_diff=wts[1])
                a = torc.delta(ch, pp, tprm, tp[0], tq[0], q0[0], lam, dense=True)
                b = torc.delta(ch, pp, tprm, tp[0], tq[0], q0[0], lam, dense=False)
                assert np.abs(a - b).max() <= 1e-10 * max(1.0, np.abs(a).max())


def test_diff_only_step_is_the_second_difference_system():
    """w_pose = 0 (the paper's trajectory-length term on its own, L123): the normal equations
    decouple per joint into (D^T D + lam I) x = -D^T D q with D the (n-1) x n differencing matrix,
    a scalar tridiagonal system -- solved here with scipy's banded solver."""
    ch = wl.panda_chain()
    d, n = ch.dof, 40
    _, tp, tq, q0 = problem(ch, n, 0.1, 5)
    pp = orc.Params()
    w = 0.7
    tprm = torc.TrajParams(w_pose=0.0, w_diff=w)
    for lam in (1e-3, 0.5):
        got = torc.delta(ch, pp, tprm, tp[0], tq[0], q0[0], lam)
        diag = np.full(n, 2.0)
        diag[0] = diag[-1] = 1.0
        ab = np.vstack([w * w * diag + lam, np.r_[np.full(n - 1, -w * w), 0.0]])  # lower form
        for a in range(d):
            qa = q0[0, :, a]
            DtDq = diag * qa - np.r_[0.0, qa[:-1]] - np.r_[qa[1:], 0.0]
            x = solveh_banded(ab, -w * w * DtDq, lower=True)
            assert np.abs(got[:, a] - x).max() < 1e-11
    # lam -> 0: the minimiser of |D(q + x)|^2 closest to q is the constant trajectory at the mean
    got = torc.delta(ch, pp, tprm, tp[0], tq[0], q0[0], 1e-10)
    assert np.abs((q0[0] + got) - q0[0].mean(axis=0, keepdims=True)).max() < 1e-6


def test_w_diff_zero_decouples_into_the_per_waypoint_step():
    """Without the differencing rows J^T J is block diagonal: every waypoint's block
    of delta is the per-waypoint LM step of oracle/lm_oracle.c (pinned in test_oracle_pins.py)."""
    for ch in CHAINS:
        d, n = ch.dof, 11
        _, tp, tq, q0 = problem(ch, n, 0.1, 6)
        pp = orc.Params(w_pos=1.0, w_rot=1.0)
        lam = 3e-3
        got = torc.delta(ch, pp, torc.TrajParams(w_pose=1.0, w_diff=0.0), tp[0], tq[0], q0[0], lam)
        p, R = orc.fk(ch, q0[0])
        for i in range(n):
            r = orc.residual(p[i], R[i], tp[0, i], tq[0, i])
            ref = orc.lm_delta(orc.jacobian(ch, q0[0, i]), r, lam)
            assert np.abs(got[i] - ref).max() < 1e-11


def test_lambda_to_infinity_is_scaled_gradient_descent():
    ch = wl.panda_chain()
    n = 8
    _, tp, tq, q0 = problem(ch, n, 0.1, 7)
    pp, tprm = orc.Params(), torc.TrajParams(w_pose=1.0, w_diff=0.5)
    J = torc.jacobian(ch, pp, tprm, q0[0])
    r = torc.residual(ch, pp, tprm, tp[0], tq[0], q0[0])
    lam = 1e9
    got = torc.delta(ch, pp, tprm, tp[0], tq[0], q0[0], lam)
    g = (J.T @ r).reshape(n, -1)
    assert np.abs(lam * got + g).max() <= 10 * np.linalg.norm(J, 2) ** 2 / lam * np.abs(g).max() + 1e-12


def trace(ch, pp, tprm, tp, tq, q0, iters, dense=False):
    st = torc.init_state(q0, tprm)
    out = []
    for _ in range(iters):
        before = st.copy()
        torc.advance(ch, pp, tprm, tp, tq, st, iters, at_most=1, dense=dense)
        out.append((before, st.copy()))
    return out


def test_lm_iteration_rules():
    ch = wl.panda_chain()
    B, n = 6, 16
    _, tp, tq, q0 = problem(ch, n, 0.15, 8, B=B, amp=0.5)
    pp = orc.Params()
    tprm = torc.TrajParams(w_pose=1.0, w_diff=0.3, lambda0=1e-3)
    steps = trace(ch, pp, tprm, tp, tq, q0, 10)
    lam = np.full(B, tprm.lambda0)
    some_reject = False
    for k, (b, a) in enumerate(steps):
        acc = a.accepted == 1
        some_reject |= bool((~acc).any())
        assert np.all(a.iters == k + 1)
        assert np.array_equal(acc, a.F_trial < a.F_before)          # strict decrease accepts
        assert np.all(a.F_total <= a.F_before)                      # cost never increases
        assert np.array_equal(a.q[~acc], b.q[~acc])                 # rejected: q bit-identical
        assert np.array_equal(a.q[acc], a.trial_q[acc])
        assert np.array_equal((a.mask >> np.uint64(k)) & np.uint64(1), acc.astype(np.uint64))
        lam = np.where(acc, np.maximum(lam / 10, tprm.lambda_min), np.minimum(lam * 10, tprm.lambda_max))
        assert np.allclose(a.lam, lam, rtol=1e-14)
        for t in range(B):
            # cost bookkeeping: F = w_pose^2 F_pose + w_diff^2 F_diff = |stacked residual|^2
            r = torc.residual(ch, pp, tprm, tp[t], tq[t], a.q[t])
            assert np.isclose(a.F_total[t], r @ r, rtol=1e-13)
            assert np.isclose(a.F_total[t], a.F_pose[t] + 0.09 * a.F_diff[t], rtol=1e-13)
            assert np.isclose(a.F_diff[t], (np.diff(a.q[t], axis=0) ** 2).sum(), rtol=1e-13)
            # trial point = clamp(q + delta(q, lambda))
            dlt = torc.delta(ch, pp, tprm, tp[t], tq[t], b.q[t], b.lam[t])
            assert np.allclose(a.trial_q[t], np.clip(b.q[t] + dlt, ch.q_lo, ch.q_hi), atol=1e-14)
    # one call of 10 iterations = 10 calls of one, bit for bit; the dense driver follows the same path
    full = torc.lm_run(ch, pp, tprm, tp, tq, q0, 10)
    assert np.array_equal(full.q, steps[-1][1].q) and np.array_equal(full.mask, steps[-1][1].mask)
    small = torc.lm_run(ch, pp, tprm, tp[:2, :], tq[:2, :], q0[:2, :], 4, dense=True)
    ref = torc.lm_run(ch, pp, tprm, tp[:2, :], tq[:2, :], q0[:2, :], 4, dense=False)
    assert np.array_equal(small.mask, ref.mask) and np.abs(small.q - ref.q).max() < 1e-9
    # a far start with lambda0 tiny produces at least one rejected step somewhere (exercises the up-branch)
    tprm2 = torc.TrajParams(w_pose=1.0, w_diff=0.3, lambda0=1e-4, lambda_min=1e-8)
    rng = np.random.default_rng(0)
    far = np.clip(q0 + 0.8 * rng.normal(size=q0.shape), ch.q_lo, ch.q_hi)
    st = torc.lm_run(ch, pp, tprm2, tp, tq, far, 12)
    bits = (st.mask[:, None] >> np.arange(12, dtype=np.uint64)[None, :]) & np.uint64(1)
    assert (bits == 0).any() or some_reject


def test_stacked_objective_shortens_the_path_and_keeps_the_pose():
    """Behaviour the paper describes (L113, L123): from a pose-valid trajectory with jitter along the
    arm's self-motion, the trajectory-level step lowers the differencing cost while the pose error
    stays near zero."""
    ch = wl.panda_chain()
    B, n = 3, 60
    truth, tp, tq, _ = problem(ch, n, 0.0, 9, B=B)
    rng = np.random.default_rng(1)
    # pose-only refinement from jittered seeds -> pose-valid but jittery in the null space
    seeds = np.clip(truth + 0.05 * rng.normal(size=truth.shape), ch.q_lo, ch.q_hi)
    st = orc.lm_run(ch, orc.Params(tol=0.0), tp.reshape(-1, 3), tq.reshape(-1, 4), seeds.reshape(-1, 7), 10)
    assert st.res_norm.max() < 1e-10
    q_pose = st.q.reshape(B, n, 7)
    tprm = torc.TrajParams(w_pose=1.0, w_diff=0.05)
    out = torc.lm_run(ch, orc.Params(), tprm, tp, tq, q_pose, 8)
    len0 = (np.diff(q_pose, axis=1) ** 2).sum(axis=(1, 2))
    assert np.all(out.F_diff < 0.8 * len0)
    assert np.all(np.sqrt(out.F_pose / n) < 2e-4)       # rms pose residual per waypoint stays small
    assert np.all(out.F_total < len0 * 0.05 ** 2)
