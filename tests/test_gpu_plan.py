"""GPU parity of the non-stationary schedule with anytime bookkeeping (lm_plan_*, NEXT-2) against
oracle/lm_plan_oracle.py: the same valid / not-valid verdicts, the same cycle of
the first valid trajectory, latest-valid joint values within 1e-4 rad, trajectory length within 1e-4
relative."""
import numpy as np
import pytest

from oracle import lm_oracle as orc
from oracle import lm_plan_oracle as porc
from oracle import lm_traj_oracle as torc
from paper_2309_09102_b200 import workloads as wl

pytestmark = pytest.mark.gpu
DEG = np.pi / 180.0


def build_problem(ch, B, n, sigma, seed):
    rng = np.random.default_rng(seed)
    truth = wl.smooth_joint_paths(ch, B, n, 3, 0.3, rng)
    w = wl._from_truth("P", ch, truth, sigma, rng, lambda q: orc.fk(ch, q), 1e-5, 10)
    return truth, w


def run_both(ch, w, cycles, pose_iters, w_diff, tol=1e-5):
    from paper_2309_09102_b200 import lm
    B, n, d = w.B, w.n, ch.dof
    s = lm.Solver(ch, B, n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=tol))
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=w_diff))
    s.plan_attach(lm.lm_plan_default_params(pose_iters=pose_iters))
    s.plan_run(cycles)
    g = s.plan_fetch()
    g["q"] = s.fetch()["q"]
    g["traj"] = s.traj_fetch()
    s.close()
    o = porc.plan(ch, orc.Params(tol=tol), torc.TrajParams(w_pose=1.0, w_diff=w_diff), porc.PlanParams(pose_iters=pose_iters),
                  w.target_pos.astype(np.float64).reshape(B, n, 3), w.target_quat.astype(np.float64).reshape(B, n, 4),
                  w.seeds.astype(np.float64).reshape(B, n, d), cycles)
    return g, o


def compare(g, o, B, n, d):
    assert np.array_equal(g["valid"], o.valid)
    assert np.array_equal(g["first_valid_cycle"], o.first_valid_cycle)
    assert g["valid_trajectories"] == int(o.valid.sum())
    same = g["traj"]["mask"] == o.traj_mask          # trajectory-level decisions agree (decisive or not)
    assert same.mean() > 0.8
    assert np.array_equal(g["traj"]["iters"], o.traj_iters)
    v = o.valid & same
    qv = g["q_valid"].reshape(B, n, d)
    assert np.abs(qv[v] - o.q_valid[v]).max() <= 1e-4
    assert np.isnan(qv[~o.valid]).all() and np.isnan(g["length"][~o.valid]).all()
    assert np.allclose(g["length"][v], o.length[v], rtol=1e-4)
    assert np.array_equal(g["records"][v], o.records[v])
    assert np.allclose(g["mjac_rev"][same], o.mjac_rev[same], atol=1e-4)
    assert np.allclose(g["cur_length"][same], porc.trajectory_length(o.q)[same], rtol=1e-4)
    assert np.abs(g["q"].reshape(B, n, d)[same] - o.q[same]).max() <= 1e-4


def test_schedule_matches_the_oracle_panda():
    ch = wl.panda_chain()
    B, n = 20, 150
    truth, w = build_problem(ch, B, n, 0.01, 41)
    # trajectory 3: second half on another self-motion branch (pose-valid, discontinuous); trajectory 5: unreachable
    tp = w.target_pos.reshape(B, n, 3).copy()
    tq = w.target_quat.reshape(B, n, 4).copy()
    seeds = w.seeds.reshape(B, n, 7).copy()
    alt = truth[3].copy()
    alt[n // 2:, 0] += 0.6
    alt[n // 2:, 6] -= 0.6
    pa, Ra = orc.fk(ch, alt)
    tp[3], tq[3], seeds[3] = pa.astype(np.float32), wl._R_to_quat_wxyz(Ra).astype(np.float32), alt.astype(np.float32)
    tp[5] += np.float32(5.0)
    w.target_pos, w.target_quat, w.seeds = tp.reshape(-1, 3), tq.reshape(-1, 4), seeds.reshape(-1, 7)
    g, o = run_both(ch, w, cycles=3, pose_iters=8, w_diff=1.0)
    compare(g, o, B, n, 7)
    assert o.valid[0] and not o.valid[3] and not o.valid[5]
    assert g["mjac_rev"][3] > 7 * DEG and g["max_pos_err"][5] > 1.0
    assert g["traj"]["iters"][5] == 0 and g["traj"]["iters"][0] == 3      # only pose-valid trajectories take the step
    # anytime: the recorded trajectories are shorter than after the first pose phase
    g0, o0 = run_both(ch, w, cycles=0, pose_iters=8, w_diff=1.0)
    compare(g0, o0, B, n, 7)
    v = o.valid
    assert np.all(g["length"][v] < g0["length"][v])
    # validity of what was recorded, re-evaluated by the oracle's FK in fp64
    qv = g["q_valid"].reshape(B, n, 7)[v].astype(np.float64)
    p, R = orc.fk(ch, qv.reshape(-1, 7))
    tpv, tqv = tp[v].reshape(-1, 3).astype(np.float64), tq[v].reshape(-1, 4).astype(np.float64)
    for k in range(0, p.shape[0], 7):
        r = orc.residual(p[k], R[k], tpv[k], tqv[k])
        assert np.linalg.norm(r[:3]) < 1e-4 and np.linalg.norm(r[3:]) < 0.1 * DEG
    assert np.abs(np.diff(qv, axis=1)).max() <= 7 * DEG + 1e-6


def test_schedule_matches_the_oracle_8dof():
    ch = wl.random_chain_8dof(3)
    B, n = 9, 200
    _, w = build_problem(ch, B, n, 0.005, 42)
    g, o = run_both(ch, w, cycles=2, pose_iters=10, w_diff=0.5)
    compare(g, o, B, n, 8)
    assert np.allclose(g["mjac_pris"], o.mjac_pris, atol=1e-5)


def test_plan_is_repeatable_and_argument_errors():
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    _, w = build_problem(ch, 5, 60, 0.01, 43)
    s = lm.Solver(ch, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=1e-5))
    with pytest.raises(lm.LmError):
        s.plan_attach()                                  # needs lm_traj_attach first
    s.traj_attach(lm.lm_traj_default_params(w_diff=0.5))
    s.plan_attach()
    with pytest.raises(lm.LmError):
        s.plan_run(65)
    outs = []
    for _ in range(2):
        s.set_state(w.seeds)
        s.plan_run(2)
        outs.append(s.plan_fetch())
    s.close()
    for k in ("q_valid", "length", "valid", "records", "mjac_rev"):
        assert np.array_equal(outs[0][k], outs[1][k], equal_nan=True), k


def test_schedule_is_the_same_on_the_fused_and_unfused_step():
    """lm_plan_run gates the trajectory-level step per trajectory (P2): the gate reaches the producer warps of the fused
    solve kernels as it reaches the per-waypoint kernels -- identical records, verdicts and latest-valid joints."""
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    _, w = build_problem(ch, 40, 90, 0.05, 47)
    outs = []
    for mode in (1, 2):
        s = lm.Solver(ch, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=1e-5))
        s.traj_attach(lm.lm_traj_default_params(w_diff=0.5))
        s.traj_set_fused(mode)
        s.plan_attach()
        s.plan_run(3)
        outs.append(s.plan_fetch())
        s.close()
    for k in ("q_valid", "length", "valid", "records", "mjac_rev", "first_valid_cycle"):
        if k in outs[0]:
            assert np.array_equal(outs[0][k], outs[1][k], equal_nan=True), k
    assert outs[0]["valid_trajectories"] == outs[1]["valid_trajectories"]


def test_schedule_with_capsules_requires_collision_free_trajectories():
    """validity includes "no collision"; with lm_traj_set_capsules the schedule checks the smallest
    capsule clearance of every waypoint and the trajectory-level step carries the collision rows."""
    from paper_2309_09102_b200 import lm
    from oracle import lm_coll_oracle as corc
    ch, model, scene = wl.panda_chain(), wl.panda_capsules(), wl.panda_scene()
    B, n = 6, 60
    rng = np.random.default_rng(44)
    base = np.array([[0.0, 0.2, 0.0, -1.8, 0.0, 2.0, 0.8]] * 3 + [[0.0, 1.2, 0.0, -2.9, 0.0, 2.2, 0.8]] * 3)
    truth = np.clip(base[:, None, :] + np.cumsum(0.004 * rng.normal(size=(B, n, 7)), axis=1), ch.q_lo, ch.q_hi)
    w = wl._from_truth("PC", ch, truth, 0.002, rng, lambda q: orc.fk(ch, q), 1e-5, 10)
    s = lm.Solver(ch, B, n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=1e-5))
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=0.1))
    s.traj_set_capsules(model, 1.0, 0.02)
    s.traj_set_obstacles(scene, 1.0, 0.02)
    s.plan_attach(lm.lm_plan_default_params(pose_iters=8))
    s.plan_run(1)
    g = s.plan_fetch()
    s.close()
    caps = corc.Capsules(model, w_coll=1.0, d_safe=0.02, scene=scene, w_env=1.0, d_safe_env=0.02)
    o = porc.plan(ch, orc.Params(tol=1e-5), torc.TrajParams(w_pose=1.0, w_diff=0.1, caps=caps), porc.PlanParams(pose_iters=8),
                  w.target_pos.astype(np.float64).reshape(B, n, 3), w.target_quat.astype(np.float64).reshape(B, n, 4),
                  w.seeds.astype(np.float64).reshape(B, n, 7), 1)
    clr_o = o.history[-1]["clearance"]
    assert np.allclose(g["min_clearance"], clr_o, atol=2e-4)
    decisive = np.abs(clr_o) > 1e-3
    assert np.array_equal(g["valid"][decisive], o.valid[decisive])
    assert o.valid[:3].any() and not o.valid[3:].any()            # the folded trajectories go through the base column
    v = o.valid & decisive
    assert np.abs(g["q_valid"].reshape(B, n, 7)[v] - o.q_valid[v]).max() <= 1e-4


def test_schedule_full_size_sampled():
    """The schedule at the size and in the configuration bench.py's schedule_C2 section times (configs[1]: 512 x 300,
    tol 1e-5, pose_iters 10, w_pose = w_diff = 1, 3 cycles): every 64th trajectory against the oracle run on those
    trajectories alone, from the same seeds (trajectories are independent)."""
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    w = wl.config2(lambda q: orc.fk(ch, q))
    B, n, d = w.B, w.n, 7
    s = lm.Solver(ch, B, n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(lambda0=w.lambda0, tol=w.tol))
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=1.0))
    s.plan_attach(lm.lm_plan_default_params(pose_iters=10))
    s.plan_run(3)
    g = s.plan_fetch()
    g["q"] = s.fetch()["q"].reshape(B, n, d)
    g["traj"] = s.traj_fetch()
    s.close()
    pick = np.arange(0, B, 64)
    o = porc.plan(ch, orc.Params(lambda0=w.lambda0, tol=w.tol), torc.TrajParams(w_pose=1.0, w_diff=1.0), porc.PlanParams(pose_iters=10),
                  w.target_pos.astype(np.float64).reshape(B, n, 3)[pick], w.target_quat.astype(np.float64).reshape(B, n, 4)[pick],
                  w.seeds.astype(np.float64).reshape(B, n, d)[pick], 3)
    assert np.array_equal(g["valid"][pick], o.valid) and np.array_equal(g["first_valid_cycle"][pick], o.first_valid_cycle)
    assert np.array_equal(g["traj"]["iters"][pick], o.traj_iters)
    same = g["traj"]["mask"][pick] == o.traj_mask
    assert same.mean() >= 0.75
    v = o.valid & same
    assert v.any()
    assert np.abs(g["q_valid"].reshape(B, n, d)[pick][v] - o.q_valid[v]).max() <= 1e-4
    assert np.allclose(g["length"][pick][v], o.length[v], rtol=1e-4)
    assert np.array_equal(g["records"][pick][v], o.records[v])
    assert np.abs(g["q"][pick][same] - o.q[same]).max() <= 1e-4
    assert g["valid_trajectories"] == int(g["valid"].sum())
