"""P8: pins of the oracle's LM iteration (accept/reject, lambda rule, convergence) -- CPU only."""
import numpy as np
from scipy.spatial.transform import Rotation

from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl

PI = np.pi


def oracle_fk(ch):
    return lambda q: orc.fk(ch, q)


def near_truth_problem(ch, W, sigma, seed):
    rng = np.random.default_rng(seed)
    truth = wl.smooth_joint_paths(ch, 1, W, 3, 0.3, rng)
    w = wl._from_truth("t", ch, truth, sigma, rng, oracle_fk(ch), 0.0, 20)
    return w


def trace(ch, prm, w, n_iters):
    """Step the oracle one iteration at a time and keep every intermediate state."""
    st = orc.init_state(w.seeds.astype(np.float64), prm)
    tp, tq = w.target_pos.astype(np.float64), w.target_quat.astype(np.float64)
    out = []
    for _ in range(n_iters):
        before = st.copy()
        orc.advance(ch, prm, tp, tq, st, n_iters, at_most=1)
        out.append((before, st.copy()))
    return out


def test_p8_monotone_reject_keeps_q_lambda_rule():
    ch = wl.panda_chain()
    prm = orc.Params(tol=0.0)
    w = near_truth_problem(ch, 64, 0.1, 20)
    steps = trace(ch, prm, w, 12)
    lam_expect = np.full(w.W, prm.lambda0)
    for k, (b, a) in enumerate(steps):
        acc = a.accepted == 1
        assert np.all(a.accepted >= 0)
        assert np.all(a.iters == k + 1)
        # accept <=> strict decrease of F (DESIGN R5); F never increases
        assert np.array_equal(acc, a.F_trial < a.F_before)
        assert np.all(a.res_norm ** 2 <= a.F_before * (1 + 1e-15))
        # rejected iterations leave q bit-identical; accepted ones take the trial point
        assert np.array_equal(a.q[~acc], b.q[~acc])
        assert np.array_equal(a.q[acc], a.trial_q[acc])
        assert np.array_equal((a.mask >> np.uint64(k)) & np.uint64(1), acc.astype(np.uint64))
        lam_expect = np.where(acc, np.maximum(lam_expect / 10, prm.lambda_min),
                              np.minimum(lam_expect * 10, prm.lambda_max))
        assert np.allclose(a.lam, lam_expect, rtol=1e-14)
        # trial point = clamp(q + delta) with delta from the Jacobian at the current q
        for i in (0, 17, 63):
            J = orc.jacobian(ch, b.q[i])
            p, R = orc.fk(ch, b.q[i])
            r = orc.residual(p, R, w.target_pos[i].astype(float), w.target_quat[i].astype(float))
            d = orc.lm_delta(J, r, b.lam[i])
            assert np.allclose(a.trial_q[i], np.clip(b.q[i] + d, ch.q_lo, ch.q_hi), atol=1e-15)
            assert np.isclose(a.F_before[i], r @ r, rtol=1e-14)


def test_p8_converges_to_rounding_within_8_iterations():
    for ch, sigma in ((wl.panda_chain(), 0.1), (wl.random_chain_8dof(3), 0.1)):
        prm = orc.Params(tol=0.0)
        w = near_truth_problem(ch, 200, sigma, 21)
        # exact (fp64) targets so that F can reach the fp64 floor
        p, R = orc.fk(ch, w.truth)
        tq = wl._R_to_quat_wxyz(R)
        st = orc.lm_run(ch, prm, p, tq, w.seeds.astype(np.float64), 8)
        # a waypoint whose accepted steps hit a joint limit follows the projected (clamped) step
        # and may converge slowly; every other one is at rounding level
        free = (st.status & 16) == 0
        assert free.mean() > 0.9 and st.res_norm[free].max() <= 1e-12
        assert np.all(st.q >= ch.q_lo) and np.all(st.q <= ch.q_hi)
        if ch.dof == 7:
            # redundant arm: the pose is pinned, the joints are NOT (1-D self-motion manifold)
            assert np.abs(st.q - w.truth).max() > 1e-4


def test_p8_one_to_three_steps_when_seeds_are_close():
    """'when initial seeds are in close vicinity to a valid solution, only 1 to 3
    steps are required' -- validity = 0.1 mm / 0.1 deg (L45)."""
    ch = wl.panda_chain()
    prm = orc.Params(tol=0.0)
    for sigma in (0.02, 0.05):
        w = near_truth_problem(ch, 300, sigma, 22)
        need = np.full(w.W, 99)
        for k, (_, a) in enumerate(trace(ch, prm, w, 4)):
            valid = (a.pos_err < 1e-4) & (a.rot_err < np.deg2rad(0.1))
            need = np.where(valid & (need == 99), k + 1, need)
        assert need.min() >= 1 and need.max() <= 3, np.bincount(need)


def test_p8_locked_six_dof_chain_recovers_the_true_joints():
    """Square (6-DoF) system: joint 7 frozen into the tool transform => the IK branch is isolated
    and LM must return the ground-truth joints, not just the pose."""
    full = wl.panda_chain()
    q7 = 0.4
    A7 = Rotation.from_euler("x", full.alpha[6]) * Rotation.from_euler("z", q7)
    tool_p = np.array([full.a[6], 0, 0]) + A7.apply([0, 0, 0.107])
    ch = wl.Chain(name="panda6", dof=6, joint_type=np.zeros(6, np.int32), a=full.a[:6], alpha=full.alpha[:6],
                  d=full.d[:6], theta=full.theta[:6], q_lo=full.q_lo[:6], q_hi=full.q_hi[:6],
                  tool=np.concatenate([tool_p, A7.as_quat()[[3, 0, 1, 2]]]))
    rng = np.random.default_rng(23)
    truth7 = wl.smooth_joint_paths(full, 1, 100, 3, 0.3, rng)[0]
    truth7[:, 6] = q7
    # the 6-DoF chain + tool is the 7-DoF chain at q7 (checks the tool handling as well)
    p7, R7 = orc.fk(full, truth7)
    p6, R6 = orc.fk(ch, truth7[:, :6])
    assert np.allclose(p6, p7, atol=1e-12) and np.allclose(R6, R7, atol=1e-12)
    seeds = np.clip(truth7[:, :6] + rng.normal(size=(100, 6)) * 0.05, ch.q_lo, ch.q_hi)
    st = orc.lm_run(ch, orc.Params(tol=0.0, lambda_min=1e-12), p6, wl._R_to_quat_wxyz(R6), seeds, 16)
    assert st.res_norm.max() < 1e-12
    assert np.abs(st.q - truth7[:, :6]).max() < 1e-10


def test_freeze_rule_and_resumability():
    """DESIGN R7: a waypoint freezes the first time sqrt(F) < tol is seen at the top of the loop;
    stepping one iteration at a time gives the same bits as one uninterrupted run."""
    ch = wl.panda_chain()
    w = wl.config2(oracle_fk(ch), B=2, n=40)
    prm = orc.Params(tol=w.tol)
    tp, tq, s = w.target_pos.astype(float), w.target_quat.astype(float), w.seeds.astype(float)
    one = orc.lm_run(ch, prm, tp, tq, s, w.max_iters)
    assert np.all(one.status & 1) and one.res_norm.max() < w.tol
    assert 2 <= one.iters.max() <= 8 and one.iters.min() >= 1
    st = orc.init_state(s, prm)
    total = 0
    for _ in range(int(one.iters.max()) + 2):
        orc.advance(ch, prm, tp, tq, st, w.max_iters, at_most=1)
        total += st.executed
    assert total == one.iters.sum() == one.executed
    for k in ("q", "lam", "iters", "mask", "status", "res_norm"):
        assert np.array_equal(getattr(st, k), getattr(one, k)), k
    # frozen waypoints had sqrt(F) >= tol before their last iteration
    t1 = orc.lm_run(ch, prm, tp, tq, s, 1)
    assert np.all(t1.iters == 1)
    # single- and multi-threaded runs are bit-identical (waypoints are independent)
    one1 = orc.lm_run(ch, prm, tp, tq, s, w.max_iters, nthreads=1)
    assert np.array_equal(one1.q, one.q) and np.array_equal(one1.mask, one.mask)


def test_max_iter_status_and_clamp():
    ch = wl.panda_chain()
    w = wl.config4(oracle_fk(ch), B=4, n=25)
    prm = orc.Params(tol=1e-5)
    st = orc.lm_run(ch, prm, w.target_pos.astype(float), w.target_quat.astype(float),
                    w.seeds.astype(float), 10)
    frozen = (st.status & 1) == 1
    assert np.all(((st.status & 2) == 2) == (~frozen & (st.iters == 10)))
    assert np.all(st.res_norm[frozen] < 1e-5) and np.all(st.res_norm[~frozen] >= 1e-5)
    assert np.all(st.q >= ch.q_lo) and np.all(st.q <= ch.q_hi)
    assert np.all(np.isfinite(st.q)) and np.all(np.isfinite(st.res_norm))


def test_workload_generators_are_seeded_and_in_limits():
    ch = wl.panda_chain()
    a = wl.config2(oracle_fk(ch), B=3, n=20)
    b = wl.config2(oracle_fk(ch), B=3, n=20)
    assert np.array_equal(a.seeds, b.seeds) and np.array_equal(a.target_quat, b.target_quat)
    for w in (a, wl.config1(oracle_fk(ch)), wl.config4(oracle_fk(ch), B=3, n=20),
              wl.config3(oracle_fk(wl.random_chain_8dof(3)), B=3, n=20)):
        c = w.chain
        assert w.seeds.dtype == np.float32 and w.target_pos.shape == (w.W, 3)
        assert np.all(w.seeds >= c.q_lo.astype(np.float32)) and np.all(w.seeds <= c.q_hi.astype(np.float32))
        assert np.all(w.seeds.astype(np.float64) >= c.q_lo) and np.all(w.seeds.astype(np.float64) <= c.q_hi)
        assert np.allclose(np.linalg.norm(w.target_quat, axis=1), 1, atol=1e-6)
        if w.truth is not None:
            assert np.all(w.truth >= c.q_lo) and np.all(w.truth <= c.q_hi)
