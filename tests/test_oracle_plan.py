"""Pins of the schedule oracle (oracle/lm_plan_oracle.py) -- CPU only."""
import numpy as np

from oracle import lm_oracle as orc
from oracle import lm_plan_oracle as porc
from oracle import lm_traj_oracle as torc
from paper_2309_09102_b200 import workloads as wl

DEG = np.pi / 180.0


def problem(ch, B, n, sigma, seed, amp=0.3):
    rng = np.random.default_rng(seed)
    truth = wl.smooth_joint_paths(ch, B, n, 3, amp, rng)
    p, R = orc.fk(ch, truth.reshape(-1, ch.dof))
    tq = wl._R_to_quat_wxyz(R)
    q0 = np.clip(truth + sigma * rng.normal(size=truth.shape) * np.where(ch.joint_type == 1, 0.1, 1.0), ch.q_lo, ch.q_hi)
    return truth, p.reshape(B, n, 3), tq.reshape(B, n, 4), q0


def test_length_and_mjac_closed_forms():
    # PAPER.md:L55 / L95 on hand-made trajectories
    n, d = 11, 8
    slope = np.array([0.002, -0.01, 0.02, 0.0, -0.03, 0.005, 0.0, 0.01])
    q = (np.arange(n)[:, None] * slope[None, :])[None]
    assert np.isclose(porc.trajectory_length(q)[0], (n - 1) * np.abs(slope).sum())
    jt = np.array([1, 0, 0, 0, 0, 0, 0, 0])
    mr, mp = porc.mjac(q, jt)
    assert np.isclose(mr[0], 0.03) and np.isclose(mp[0], 0.002)
    q2 = q.copy()
    q2[0, 5:, 2] += 0.5                       # one jump of joint 3 between timesteps 4 and 5
    mr, mp = porc.mjac(q2, jt)
    assert np.isclose(mr[0], 0.52) and np.isclose(mp[0], 0.002)
    assert np.isclose(porc.trajectory_length(q2)[0], (n - 1) * np.abs(slope).sum() + 0.5)
    assert porc.mjac(q[:, :1], jt)[0][0] == 0.0 and porc.trajectory_length(q[:, :1])[0] == 0.0


def test_zero_cycles_is_the_pose_only_oracle_and_validity_is_what_the_paper_states():
    ch = wl.panda_chain()
    B, n = 6, 150
    _, tp, tq, q0 = problem(ch, B, n, 0.01, 31)
    pp = orc.Params(tol=1e-6)
    res = porc.plan(ch, pp, torc.TrajParams(), porc.PlanParams(pose_iters=10), tp, tq, q0, 0)
    ref = orc.lm_run(ch, pp, tp.reshape(-1, 3), tq.reshape(-1, 4), q0.reshape(-1, 7), 10)
    assert np.array_equal(res.q.reshape(-1, 7), ref.q)
    assert res.valid.all() and np.all(res.first_valid_cycle == 0) and np.all(res.records == 1)
    assert np.array_equal(res.q_valid, res.q)
    # independent re-evaluation of the validity constraints of PAPER.md:L45 / L53
    p, R = orc.fk(ch, res.q_valid.reshape(-1, 7))
    for w in range(B * n):
        r = orc.residual(p[w], R[w], tp.reshape(-1, 3)[w], tq.reshape(-1, 4)[w])
        assert np.linalg.norm(r[:3]) < 1e-4 and np.linalg.norm(r[3:]) < 0.1 * DEG
    assert np.abs(np.diff(res.q_valid, axis=1)).max() <= 7 * DEG
    assert np.allclose(res.length, np.abs(np.diff(res.q_valid, axis=1)).sum(axis=(1, 2)))
    assert np.all(res.traj_iters == 0)


def test_cycles_shorten_the_path_and_keep_a_valid_solution():
    ch = wl.panda_chain()
    B, n = 4, 150
    _, tp, tq, q0 = problem(ch, B, n, 0.01, 32)
    pp = orc.Params(tol=1e-6)
    t = torc.TrajParams(w_pose=1.0, w_diff=1.0)
    r0 = porc.plan(ch, pp, t, porc.PlanParams(pose_iters=10), tp, tq, q0, 0)
    r3 = porc.plan(ch, pp, t, porc.PlanParams(pose_iters=10), tp, tq, q0, 3)
    assert r3.valid.all() and np.all(r3.first_valid_cycle == 0)
    assert np.all(r3.traj_iters == 3)
    assert np.all(r3.length < r0.length)        # the differencing term shortens the trajectory
    assert np.all(r3.records >= 2)
    # the recorded trajectory is valid by the independent test
    p, R = orc.fk(ch, r3.q_valid.reshape(-1, 7))
    err = np.array([np.linalg.norm(orc.residual(p[w], R[w], tp.reshape(-1, 3)[w], tq.reshape(-1, 4)[w])[:3]) for w in range(B * n)])
    assert err.max() < 1e-4


def test_discontinuity_and_unreachable_targets_are_not_valid_and_gate_the_trajectory_step():
    ch = wl.panda_chain()
    B, n = 3, 150
    truth, tp, tq, q0 = problem(ch, B, n, 0.005, 33)
    # trajectory 1: a self-motion jump in the seeds (another IK branch for the second half): pose-valid, mjac-invalid
    alt = truth[1].copy()
    alt[n // 2:, 0] += 0.6
    alt[n // 2:, 6] -= 0.6
    pa, Ra = orc.fk(ch, alt)
    tp[1], tq[1] = pa, wl._R_to_quat_wxyz(Ra)
    q0[1] = alt
    # trajectory 2: targets 5 m away: never pose-valid
    tp[2] = tp[2] + np.array([5.0, 0, 0])
    pp = orc.Params(tol=1e-6)
    res = porc.plan(ch, pp, torc.TrajParams(w_pose=1.0, w_diff=0.1), porc.PlanParams(pose_iters=8), tp, tq, q0, 2)
    assert res.valid[0] and not res.valid[1] and not res.valid[2]
    assert res.mjac_rev[1] > 7 * DEG and res.max_pos_err[1] < 1e-4
    assert res.max_pos_err[2] > 1.0
    assert np.isnan(res.q_valid[1]).all() and np.isnan(res.length[2])
    assert res.traj_iters[0] == 2 and res.traj_iters[1] == 2 and res.traj_iters[2] == 0   # only pose-valid ones step (P2)


def test_collision_free_is_part_of_validity():
    """"At no timestep in the trajectory can the robot collide with itself or the environment"."""
    from oracle import lm_coll_oracle as corc
    ch, model = wl.panda_chain(), wl.panda_capsules()
    B, n = 2, 60
    rng = np.random.default_rng(35)
    base = np.array([[0.0, 0.2, 0.0, -1.8, 0.0, 2.0, 0.8], [0.0, 1.2, 0.0, -2.9, 0.0, 2.2, 0.8]])   # open arm / folded through the base
    truth = np.clip(base[:, None, :] + np.cumsum(0.004 * rng.normal(size=(B, n, 7)), axis=1), ch.q_lo, ch.q_hi)
    p, R = orc.fk(ch, truth.reshape(-1, 7))
    tp, tq = p.reshape(B, n, 3), wl._R_to_quat_wxyz(R).reshape(B, n, 4)
    caps = corc.Capsules(model, w_coll=1.0, d_safe=0.02)
    clr = porc.min_clearance(ch, caps, truth)
    assert clr[0] > 0.02 and clr[1] < 0                                   # the second one penetrates
    # brute check of min_clearance against the per-waypoint distances
    assert np.isclose(clr[1], min(corc.residual(ch, caps, truth[1, i])[0].min() for i in range(n)))
    res = porc.plan(ch, orc.Params(tol=1e-6), torc.TrajParams(w_pose=1.0, w_diff=0.1, caps=caps),
                    porc.PlanParams(pose_iters=8), tp, tq, truth, 0)
    assert res.valid[0] and not res.valid[1]
    assert res.max_pos_err[1] < 1e-4 and res.mjac_rev[1] < 7 * DEG       # pose-valid and smooth: only the collision fails it
    # without a capsule model both are valid
    res0 = porc.plan(ch, orc.Params(tol=1e-6), torc.TrajParams(w_pose=1.0, w_diff=0.1), porc.PlanParams(pose_iters=8), tp, tq, truth, 0)
    assert res0.valid.all()
