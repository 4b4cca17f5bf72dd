"""The rotation residual r_rot = Log(R_ee R_t^T) over its WHOLE range on the GPU (S2; "geodesic distance",
L115-117), against oracle/lm_oracle.c (orc_log_so3; its own small-angle and near-pi branches are pinned in
tests/test_oracle_pins.py).  The documented workloads keep the rotation error below 90 degrees; an IK seed on the wrong
wrist flip is 180 degrees away, and the kernel has branches of its own there (the small-angle series below
sin(theta) = 1e-4, the cos(theta) < 0 reflection of atan2_pos, log_far for cos(theta) < -1/2).

Construction: seeds q (fp32), (p, R) = oracle FK(q) in fp64, target rotation R_t = Exp(-theta a) R so that
R R_t^T = Exp(theta a) for theta over 15 values from 0 to pi and 20 random axes a each; the target quaternion is
rounded to fp32 ONCE and both sides read that value.  Trajectory b holds theta[b], so the trajectory-level step
(which shares eval_pose) is exercised on the same poses.

Within 1e-6 of pi the SIGN of the axis is not determined by fp32 data (+pi a and -pi a are the same rotation): there
the norms are compared, and each side's trial cost is checked against the oracle's residual at that side's own trial
point; everywhere else the trial point itself is held to the 1e-4 bar."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import lm_oracle as orc
from oracle import lm_traj_oracle as torc
from paper_2309_09102_b200 import workloads as wl

import helpers as H

pytestmark = pytest.mark.gpu

THETAS = np.array([0.0, 1e-9, 1e-5, 0.99e-4, 1.01e-4, 1.0, np.pi / 2, 2.0, 2.2, 3.0, np.pi - 1e-3, np.pi - 2e-4, np.pi - 5e-5,
                   np.pi - 1e-6, np.pi])
N_AXES = 20
SIGN_FREE = THETAS >= np.pi - 2e-6


def rotation_problem(ch, seed):
    rng = np.random.default_rng(seed)
    B, n, d = len(THETAS), N_AXES, ch.dof
    mid, half = 0.5 * (ch.q_lo + ch.q_hi), 0.5 * (ch.q_hi - ch.q_lo)
    base = mid + 0.5 * half * rng.uniform(-1, 1, size=(B, 1, d))
    q = np.clip(base + np.cumsum(0.02 * rng.normal(size=(B, n, d)), axis=1), ch.q_lo + 0.1 * half, ch.q_hi - 0.1 * half).astype(np.float32)
    p, R = orc.fk(ch, q.reshape(B * n, d).astype(np.float64))
    axes = rng.normal(size=(B, n, 3))
    axes[:, 0] = [1.0, 0.0, 0.0]                                   # axis-aligned: two components of a are exactly 0
    axes[:, 1] = [0.0, 0.7071067811865476, -0.7071067811865476]
    axes[:, 2] = [1e-4, 1.0, 1e-3]                                 # one tiny component (the ill-conditioned one for a square root)
    axes /= np.linalg.norm(axes, axis=2, keepdims=True)
    rot = Rotation.from_rotvec((-THETAS[:, None, None] * axes).reshape(B * n, 3)).as_matrix()
    Rt = rot @ R
    tq = wl._R_to_quat_wxyz(Rt).astype(np.float32)
    tp = (p + 1e-3 * rng.normal(size=p.shape)).astype(np.float32)
    return B, n, q, tp, tq


def oracle_residuals(ch, q, tp, tq):
    p, R = orc.fk(ch, q.astype(np.float64))
    r = np.stack([orc.residual(p[i], R[i], tp[i].astype(np.float64), tq[i].astype(np.float64)) for i in range(len(q))])
    return np.linalg.norm(r, axis=1), np.linalg.norm(r[:, :3], axis=1), np.linalg.norm(r[:, 3:], axis=1)


@pytest.mark.parametrize("chain_name", ["panda", "rand8", "rot_tool"])
def test_residual_and_one_step_over_the_whole_rotation_range(chain_name):
    from paper_2309_09102_b200 import lm
    if chain_name == "rand8":
        ch = wl.random_chain_8dof(3)
    else:
        ch = wl.panda_chain()
        if chain_name == "rot_tool":                               # not a benchmark structure: the generic kernel
            ch.tool = np.array([0.01, -0.02, 0.107, 0.9238795325112867, 0.2, -0.1, 0.3104])
            ch.tool[3:] /= np.linalg.norm(ch.tool[3:])
    B, n, q, tp, tq = rotation_problem(ch, 7)
    W, d = B * n, ch.dof
    q = q.reshape(W, d)
    theta = np.repeat(THETAS, n)
    free = np.repeat(SIGN_FREE, n)
    s = lm.Solver(ch, B, n, tp, tq, q, params=lm.lm_default_params(tol=0.0))
    g0 = s.fetch()                                                 # state = seeds: |r|, pos_err, rot_err at the seeds
    rn, pe, re = oracle_residuals(ch, q, tp, tq)
    assert np.abs(re - theta).max() <= 2e-6                        # the construction: the oracle sees the angles it was given
    print("rotation range:", chain_name, "max |res_norm - oracle|", np.abs(g0["res_norm"] - rn).max(),
          "max |rot_err - oracle|", np.abs(g0["rot_err"] - re).max())
    assert np.abs(g0["res_norm"] - rn).max() <= 2e-6
    assert np.abs(g0["pos_err"] - pe).max() <= 2e-6
    assert np.abs(g0["rot_err"] - re).max() <= 2e-6
    # one teacher-forced LM step from the seeds, lambda = 1 (a step of ~1 rad: not clamped away, well conditioned)
    lam = np.ones(W, np.float32)
    s.enable_trace()
    s.set_state(q, lam)
    s.step()
    g = s.fetch()
    s.close()
    prm = orc.Params(lambda0=1.0, tol=0.0)
    st = orc.State(q=q.astype(np.float64), lam=lam.astype(np.float64), iters=np.zeros(W, np.int32), mask=np.zeros(W, np.uint64),
                   status=np.zeros(W, np.uint32))
    orc.advance(ch, prm, tp.astype(np.float64), tq.astype(np.float64), st, 1)
    dq = np.abs(g["trial_q"] - st.trial_q).max(axis=1)
    per_theta = dq.reshape(B, n).max(axis=1)
    print("max |trial_q - oracle| per theta:", dict(zip(np.round(THETAS, 6).tolist(), per_theta.tolist())))
    assert dq[~free].max() <= H.TOL_Q, per_theta
    assert np.abs(np.sqrt(g["F_before"]) - np.sqrt(st.F_before)).max() <= 2e-6          # |r| to the fp32 floor of a pose
    assert np.abs(np.sqrt(g["F_trial"]) - np.sqrt(st.F_trial))[~free].max() <= 2e-6 + 8 * dq[~free].max()
    dec = ~free & H.decisive(st.F_before, st.F_trial)
    assert dec.sum() > W // 2
    assert np.array_equal(((g["mask"] & np.uint64(1)) == 1)[dec], (st.accepted == 1)[dec])
    # where the sign of the axis is free: the GPU's step is a valid one -- its reported trial cost is the oracle's cost
    # at the GPU's own trial point, and it goes downhill as the oracle's does
    rn_t, _, _ = oracle_residuals(ch, g["trial_q"][free], tp[free], tq[free])
    assert np.abs(np.sqrt(g["F_trial"][free]) - rn_t).max() <= 2e-6
    assert np.all(np.isfinite(g["trial_q"])) and np.all(g["F_trial"][free] < g["F_before"][free])


def test_trajectory_level_step_over_the_whole_rotation_range():
    """lm_traj_run(1) on the same poses (the stacked step calls the same eval_pose): trial point of every trajectory
    whose angles leave the sign of the axis determined, costs of all of them."""
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    B, n, q, tp, tq = rotation_problem(ch, 8)
    d = ch.dof
    lam = np.ones(B, np.float32)
    s = lm.Solver(ch, B, n, tp, tq, q.reshape(B * n, d), params=lm.lm_default_params(tol=0.0))
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=0.3))
    s.traj_reset(lam)
    s.traj_enable_trace()
    s.traj_run(1)
    g = s.traj_fetch()
    s.close()
    tprm = torc.TrajParams(w_pose=1.0, w_diff=0.3)
    st = torc.init_state(q.astype(np.float64), tprm)
    st.lam[:] = 1.0
    torc.advance(ch, orc.Params(), tprm, tp.astype(np.float64).reshape(B, n, 3), tq.astype(np.float64).reshape(B, n, 4), st, 1)
    err = np.abs(g["trial_q"].reshape(B, n, d) - st.trial_q).max(axis=(1, 2))
    print("trajectory-level step, max |trial_q - oracle| per theta:", dict(zip(np.round(THETAS, 6).tolist(), err.tolist())))
    assert np.allclose(g["F_before"], st.F_before, rtol=1e-5)      # sums over 20 waypoints, dominated by theta^2
    assert err[~SIGN_FREE].max() <= H.TOL_Q
    assert np.allclose(g["F_trial"][~SIGN_FREE], st.F_trial[~SIGN_FREE], rtol=1e-4, atol=1e-9)
    dec = ~SIGN_FREE & (np.abs(st.F_before - st.F_trial) > 1e-3 * st.F_before)
    assert np.array_equal((g["mask"] & np.uint64(1)).astype(bool)[dec], (st.accepted == 1)[dec])
    assert np.all(np.isfinite(g["trial_q"]))
