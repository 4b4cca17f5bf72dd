"""Parity of the CUDA path (through the C ABI) against the fp64 oracle -- needs a B200.

Bars (BASELINE.json north_star, restated in DESIGN.md section 4):
  * joints: max-abs |q_gpu - q_oracle| <= 1e-4 rad (m) per joint,
  * pose error of the GPU's q re-evaluated by the oracle's fp64 FK within 1e-5 m / 1e-4 rad of
    the oracle's own,
  * identical accept/reject sequence on the decisive iterations,
  * integers (iteration counts, status, masks on the decisive prefix) exact.
"""
import numpy as np
import pytest

from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl

import helpers as H

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lm():
    from paper_2309_09102_b200 import build, lm as _lm
    build.build()
    return _lm


# ------------------------------------------------------------------ S1: FK alone

def _fk_cases():
    panda = wl.panda_chain()
    rot_tool = wl.panda_chain()
    rot_tool.tool = np.array([0.01, -0.02, 0.107, 0.9238795325112867, 0.2, -0.1, 0.3104])
    rot_tool.tool[3:] /= np.linalg.norm(rot_tool.tool[3:])
    six = wl.panda_chain()
    six = wl.Chain("panda6", 6, six.joint_type[:6], six.a[:6], six.alpha[:6], six.d[:6], six.theta[:6],
                   six.q_lo[:6], six.q_hi[:6], six.tool)
    gen = wl.Chain("gen3", 3, np.array([0, 1, 0], np.int32), np.array([0.1, 0.2, -0.3]), np.array([0.3, -1.1, 2.0]),
                   np.array([0.05, 0.1, 0.2]), np.array([0.4, -0.7, 1.3]), np.full(3, -2.0), np.full(3, 2.0),
                   np.array([0.1, 0.0, 0.2, 1, 0, 0, 0.0]))
    return [panda, wl.random_chain_8dof(3), rot_tool, six, gen]


@pytest.mark.parametrize("chain", _fk_cases(), ids=lambda c: c.name + str(c.dof))
def test_fk_matches_oracle(lm, chain):
    rng = np.random.default_rng(100)
    n = 1000 + 37  # several blocks and a ragged tail
    mid, half = 0.5 * (chain.q_lo + chain.q_hi), 0.5 * (chain.q_hi - chain.q_lo)
    q = (mid + half * rng.uniform(-1, 1, size=(n, chain.dof))).astype(np.float32)
    fk = lm.device_fk(chain)
    p, R = fk(q)
    po, Ro = orc.fk(chain, q.astype(np.float64))
    assert np.abs(p - po).max() < 1e-6       # SURVEY section 7 minimum slice: <= 1e-6 m
    assert np.abs(R - Ro).max() < 1e-6       #                                 <= 1e-6 rad
    # the measured fp32 pose error that H.EPS_POSE bounds (DESIGN.md section 4 quotes these numbers)
    pos_e = np.linalg.norm(p - po, axis=1).max()
    rot_e = (np.linalg.norm(R @ Ro.transpose(0, 2, 1) - np.eye(3), axis=(1, 2)) / np.sqrt(2.0)).max()
    print("FK error:", chain.name, chain.dof, "max |p - p_oracle|", pos_e, "max rotation angle", rot_e)
    assert pos_e <= H.EPS_POS and rot_e <= H.EPS_POSE


@pytest.mark.parametrize("cfg", ["C2", "C3", "C4"])
def test_pose_residual_error_is_within_eps_pose(lm, cfg):
    """H.EPS_POSE (the absolute error allowed to an fp32 pose residual norm; `decisive` and the collision tests derive
    their noise terms from it) is a bound on something MEASURED here: |r| of the kernel at the seeds of configs[1..3]
    against the oracle's fp64 |r| at the same fp32 inputs, all waypoints of 64 trajectories."""
    if cfg == "C2":
        w = wl.config2(H.oracle_fk(wl.panda_chain()), B=64, n=300)
    elif cfg == "C3":
        w = wl.config3(H.oracle_fk(wl.random_chain_8dof(3)), B=64, n=300)
    else:
        w = wl.config4(H.oracle_fk(wl.panda_chain()), B=64, n=300)
    s = H.make_solver(w)
    g = s.fetch()
    s.close()
    pe, re = H.pose_errors_by_oracle(w, w.seeds)
    rn = np.sqrt(pe * pe + re * re)
    e_r, e_p, e_w = np.abs(g["res_norm"] - rn).max(), np.abs(g["pos_err"] - pe).max(), np.abs(g["rot_err"] - re).max()
    print("pose residual error:", cfg, "max | |r| - oracle |", e_r, "position part", e_p, "rotation part", e_w, "max |r|", rn.max())
    assert max(e_r, e_p, e_w) <= H.EPS_POSE


# ------------------------------------------------------------------ free-running parity (P10)

def _check_free_running(w, g, o, frac_edge=0.002, check_pose=True):
    dq = np.abs(g["q"] - o.q).max(axis=1)
    # waypoints whose freeze decision fell on the other side of tol differ by one (tiny) iteration;
    # they are allowed as long as the oracle's |r| sat within 2 % of tol at that check
    diff_it = g["iters"] != o.iters
    assert diff_it.mean() <= frac_edge, diff_it.mean()
    assert np.all(np.abs(g["iters"] - o.iters)[diff_it] == 1)
    assert dq.max() <= H.TOL_Q, (dq.max(), int((dq > H.TOL_Q).sum()))
    assert np.array_equal(g["status"][~diff_it] & 3, o.status[~diff_it] & 3)
    assert np.all(g["q"] >= w.chain.q_lo.astype(np.float32)) and np.all(g["q"] <= w.chain.q_hi.astype(np.float32))
    if check_pose:
        idx = np.arange(w.W) if w.W <= 20000 else np.random.default_rng(0).choice(w.W, 20000, replace=False)
        sub = wl.Workload(w.name, w.chain, 1, len(idx), w.target_pos[idx], w.target_quat[idx], w.seeds[idx],
                          w.tol, w.max_iters)
        pe, re = H.pose_errors_by_oracle(sub, g["q"][idx])
        assert np.abs(pe - o.pos_err[idx]).max() <= H.TOL_POS
        assert np.abs(re - o.rot_err[idx]).max() <= H.TOL_ROT
        # and the errors the library reports are the ones its q really has
        assert np.abs(g["pos_err"][idx] - pe).max() <= 2e-6 and np.abs(g["rot_err"][idx] - re).max() <= 2e-6


def test_config1_fixed_20_iterations(lm):
    """BASELINE.json configs[0]: 1 x 50, Panda, 20 iterations, tol = 0."""
    w = wl.config1(H.oracle_fk(wl.panda_chain()))
    g, o = H.run_gpu(w), H.run_oracle(w)
    assert np.all(g["iters"] == 20) and g["total_waypoint_iters"] == 50 * 20
    _check_free_running(w, g, o)
    assert np.abs(g["q"] - o.q).max() < 5e-6  # far inside the bar when nothing is chaotic
    compared, bad = H.decisive_mismatches(w, g, 20)
    assert compared >= 100 and bad == 0
    assert g["res_norm"].max() < 1e-6           # fp32 floor
    assert np.array_equal(g["traj_iters"], [20]) and np.array_equal(g["traj_converged"], [0])


def test_config2_full_size_to_convergence(lm):
    """configs[1] at full size (512 x 300) in the launch configuration bench.py times."""
    w = wl.config2(H.oracle_fk(wl.panda_chain()))
    g, o = H.run_gpu(w), H.run_oracle(w)
    _check_free_running(w, g, o)
    assert np.all(g["status"] & 1) and g["res_norm"].max() < w.tol
    assert g["converged_trajectories"] == w.B and np.all(g["traj_converged"] == 1)
    assert g["total_waypoint_iters"] == int(g["iters"].sum())
    assert abs(g["total_waypoint_iters"] - int(o.iters.sum())) <= 0.002 * w.W
    assert np.array_equal(g["traj_iters"], g["iters"].reshape(w.B, w.n).max(axis=1))
    compared, bad = H.decisive_mismatches(w, g, int(o.iters.max()))
    assert compared > w.W and bad == 0


def test_config3_eight_dof_prismatic(lm):
    """configs[2]: 8-DoF chain with a prismatic joint; 256 of the 2048 trajectories element by
    element, the full size on aggregate counts."""
    ch = wl.random_chain_8dof(3)
    w = wl.config3(H.oracle_fk(ch))
    g = H.run_gpu(w)
    o = H.run_oracle(w)
    _check_free_running(w, g, o)
    sub = w.subset(slice(0, 256))
    gs = {k: (v[:sub.W] if isinstance(v, np.ndarray) and v.shape[:1] == (w.W,) else v) for k, v in g.items()}
    compared, bad = H.decisive_mismatches(sub, gs, int(o.iters[:sub.W].max()))
    assert compared > sub.W and bad == 0
    frozen = (g["status"] & 1) == 1
    assert frozen.mean() > 0.99 and (frozen != ((o.status & 1) == 1)).mean() < 0.002


def test_config4_chaotic_far_seeds(lm):
    """configs[3] (far seeds, unreachable path ends): 44 % of the decisions are rejects and fp32 / fp64 sequences
    part on a few % of the waypoints whatever the solver.  Graded by H.check_chaotic_config:
    STRICT sequence parity on every waypoint whose oracle decisions are all clear-cut, strict 1e-4 joint parity on
    every such waypoint the oracle itself determines to 2e-5 (the others are shown ill-conditioned from the oracle
    alone and must stay inside its spread), plus agreement of the aggregate statistics of the whole batch."""
    w = wl.config4(H.oracle_fk(wl.panda_chain()), B=64, n=300)
    g, o = H.run_gpu(w), H.run_oracle(w)
    assert np.all(g["iters"] == 50)
    H.check_chaotic_config(w, g, o, 50)
    # aggregate statistics of the whole batch
    conv_g, conv_o = (g["res_norm"] < 1e-5).mean(), (o.res_norm < 1e-5).mean()
    assert abs(conv_g - conv_o) <= 0.005
    assert abs(np.median(g["res_norm"]) - np.median(o.res_norm)) <= 0.05 * np.median(o.res_norm) + 1e-7
    assert np.all(np.isfinite(g["q"])) and np.all(np.isfinite(g["res_norm"]))


# ------------------------------------------------------------------ teacher-forced single steps (P9)

@pytest.mark.parametrize("cfg", ["C2", "C3", "C4"])
def test_teacher_forced_steps(lm, cfg):
    """For every oracle iterate (q_k, lambda_k): lm_set_state -> lm_step -> compare the trial point
    (i.e. delta), F+ and the decision.  Isolates kernel error from divergence of the sequences."""
    if cfg == "C2":
        w = wl.config2(H.oracle_fk(wl.panda_chain()), B=16, n=300)
    elif cfg == "C3":
        w = wl.config3(H.oracle_fk(wl.random_chain_8dof(3)), B=16, n=300)
    else:
        w = wl.config4(H.oracle_fk(wl.panda_chain()), B=16, n=300)
    n_it = 6 if cfg != "C4" else 24
    w0 = wl.Workload(w.name, w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, 0.0, n_it, w.lambda0)
    tr = H.oracle_trace(w0, n_it)
    s = H.make_solver(w0)
    s.enable_trace()
    worst, decided, mism = 0.0, 0, 0
    for k, (b, a) in enumerate(tr):
        s.set_state(b.q.astype(np.float32), b.lam.astype(np.float32))
        s.step()
        g = s.fetch()
        # the state handed over is the oracle's rounded to fp32: compare against the oracle stepped
        # from exactly that state
        st = orc.State(q=b.q.astype(np.float32).astype(np.float64), lam=b.lam.astype(np.float32).astype(np.float64),
                       iters=np.zeros(w.W, np.int32), mask=np.zeros(w.W, np.uint64), status=np.zeros(w.W, np.uint32))
        orc.advance(w.chain, H.oracle_params(w0), w.target_pos.astype(np.float64), w.target_quat.astype(np.float64),
                    st, 1)
        sig = np.sqrt(st.F_before) >= 1e-5
        if not sig.any():
            break
        d = np.abs(g["trial_q"] - st.trial_q).max(axis=1)
        worst = max(worst, d[sig].max())
        # |r| agrees to the fp32 floor of the pose (~1e-7 m / rad per component)
        assert np.abs(np.sqrt(g["F_before"][sig]) - np.sqrt(st.F_before[sig])).max() <= 1e-6
        dec = sig & H.decisive(st.F_before, st.F_trial)
        acc_g = (g["mask"] & np.uint64(1)) == 1
        decided += int(dec.sum())
        mism += int((dec & (acc_g != (st.accepted == 1))).sum())
        assert np.all(g["iters"] == 1)
    s.close()
    assert worst <= H.TOL_Q, worst
    assert decided > 0 and mism == 0, (decided, mism)


# ------------------------------------------------------------------ NEXT-4 (i): dual 6 x 6 form

def test_dual_form_variant_matches_the_oracle(lm):
    """LM_SOLVER_DUAL: delta = -J^T (J J^T + lambda I_6)^-1 r is the SAME step (push-through identity,
    pinned on the oracle by P5), so the oracle's primal fp64 sequence is the reference: configs[0]
    and configs[1] at full size, same bars as the primal path; no refinement step is involved."""
    w = wl.config1(H.oracle_fk(wl.panda_chain()))
    g, o = H.run_gpu(w, solver=lm.LM_SOLVER_DUAL, refine_steps=0), H.run_oracle(w)
    _check_free_running(w, g, o)
    assert np.abs(g["q"] - o.q).max() < 5e-6
    compared, bad = H.decisive_mismatches(w, g, 20)
    assert compared >= 100 and bad == 0
    w = wl.config2(H.oracle_fk(wl.panda_chain()))
    g, o = H.run_gpu(w, solver=lm.LM_SOLVER_DUAL, refine_steps=0), H.run_oracle(w)
    _check_free_running(w, g, o)
    assert g["converged_trajectories"] == w.B
    compared, bad = H.decisive_mismatches(w, g, int(o.iters.max()))
    assert compared > w.W and bad == 0
    # 8-DoF chain with a prismatic joint
    ch = wl.random_chain_8dof(3)
    w = wl.config3(H.oracle_fk(ch), B=128)
    g, o = H.run_gpu(w, solver=lm.LM_SOLVER_DUAL), H.run_oracle(w)
    _check_free_running(w, g, o)


# ------------------------------------------------------------------ NEXT-4 (ii): roll-pitch-yaw residual

def test_rpy_residual_variant_matches_the_oracle(lm):
    """LM_ROT_RPY: the paper's literal residual, wrapped element-wise rpy differences with
    d(rpy)/dq = E^-1 J_w, against the oracle run with rot_mode = 1: configs[0] and a 64-trajectory configs[1]."""
    w = wl.config1(H.oracle_fk(wl.panda_chain()))
    g = H.run_gpu(w, rot_residual=lm.LM_ROT_RPY)
    o = H.run_oracle(w, rot_mode=1)
    _check_free_running(w, g, o, check_pose=False)
    assert np.abs(g["q"] - o.q).max() < 2e-5
    w = wl.config2(H.oracle_fk(wl.panda_chain()), B=64)
    g = H.run_gpu(w, rot_residual=lm.LM_ROT_RPY)
    o = H.run_oracle(w, rot_mode=1)
    _check_free_running(w, g, o, frac_edge=0.01, check_pose=False)
    assert (g["status"] & 1).mean() > 0.99
    # the pose it converges to is the target pose: the rotation-vector error of the result is small too
    pe, re = H.pose_errors_by_oracle(w, g["q"])
    assert pe.max() < 2e-5 and re.max() < 2e-5
    # not combinable with the dual solver or the trajectory-level step
    with pytest.raises(lm.LmError):
        H.make_solver(w, rot_residual=lm.LM_ROT_RPY, solver=lm.LM_SOLVER_DUAL)
    s = H.make_solver(w, rot_residual=lm.LM_ROT_RPY)
    with pytest.raises(lm.LmError):
        s.traj_attach()
    s.close()


# ------------------------------------------------------------------ full sizes of the bench, sampled outputs

def test_config4_full_size_sampled(lm):
    """configs[3] at FULL size (4096 x 300) in the launch configuration bench.py times (one lm_run(50) launch,
    128-thread blocks); every 128th trajectory (32 trajectories, 9600 waypoints) is checked against the oracle --
    waypoints are independent and a waypoint's bits do not depend on the batch (test_gpu_edge), so
    the oracle only has to run the sample."""
    w = wl.config4(H.oracle_fk(wl.panda_chain()))
    assert (w.B, w.n) == (4096, 300)
    g = H.run_gpu(w)
    assert g["total_waypoint_iters"] == w.W * 50 and np.all(g["iters"] == 50)
    assert np.all(np.isfinite(g["q"])) and np.all(g["q"] >= w.chain.q_lo.astype(np.float32)) and np.all(g["q"] <= w.chain.q_hi.astype(np.float32))
    pick = np.arange(0, w.B, 128)
    idx = (pick[:, None] * w.n + np.arange(w.n)[None, :]).ravel()
    sub = wl.Workload(w.name, w.chain, len(pick), w.n, w.target_pos[idx], w.target_quat[idx], w.seeds[idx], w.tol, w.max_iters)
    o = H.run_oracle(sub)
    gs = {k: v[idx] for k, v in g.items() if isinstance(v, np.ndarray) and v.shape[:1] == (w.W,)}
    H.check_chaotic_config(sub, gs, o, 50)
    assert abs((g["res_norm"][idx] < 1e-5).mean() - (o.res_norm < 1e-5).mean()) <= 0.01
    # the errors the library reports are the ones its q really has (oracle FK of the GPU's q), sampled over the whole batch
    rnd = np.random.default_rng(0).choice(w.W, 4000, replace=False)
    s2 = wl.Workload(w.name, w.chain, 1, len(rnd), w.target_pos[rnd], w.target_quat[rnd], w.seeds[rnd], w.tol, w.max_iters)
    pe, re = H.pose_errors_by_oracle(s2, g["q"][rnd])
    assert np.abs(g["pos_err"][rnd] - pe).max() <= 5e-6 and np.abs(g["rot_err"][rnd] - re).max() <= 5e-6


@pytest.mark.parametrize("B,n", [(1, 100), (7, 1000), (16384, 100)])
def test_config5_sweep_points(lm, B, n):
    """configs[4] (throughput sweep, fixed 20 iterations): the smallest, a long ragged and the largest-batch point;
    the large one on a sample of trajectories."""
    w = wl.config5(H.oracle_fk(wl.panda_chain()), B=min(B, 64), n=n) if B <= 64 else None
    if w is not None:
        g, o = H.run_gpu(w), H.run_oracle(w)
        _check_free_running(w, g, o)
        assert np.all(g["iters"] == 20)
        return
    # large batch: targets need one oracle FK per waypoint, so the batch is built by tiling 64 distinct trajectories
    base = wl.config5(H.oracle_fk(wl.panda_chain()), B=64, n=n)
    reps = B // 64
    big = wl.Workload(base.name, base.chain, B, n, np.tile(base.target_pos, (reps, 1)), np.tile(base.target_quat, (reps, 1)),
                      np.tile(base.seeds, (reps, 1)), base.tol, base.max_iters)
    g, o = H.run_gpu(big), H.run_oracle(base)
    assert g["total_waypoint_iters"] == big.W * 20
    for r in (0, reps // 2, reps - 1):          # copies of the same trajectories anywhere in the batch: same bits, oracle parity
        sl = slice(r * base.W, (r + 1) * base.W)
        assert np.array_equal(g["q"][sl], g["q"][:base.W])
        assert np.abs(g["q"][sl] - o.q).max() <= H.TOL_Q
        assert np.array_equal(g["iters"][sl], o.iters)


# ------------------------------------------------------------------ lane-group form (LM_OPT_LANES_PER_WAYPOINT)

@pytest.mark.parametrize("lanes", [2, 4])
def test_lane_group_variant_matches_the_oracle(lm, lanes):
    """The measured alternative BASELINE.json's north_star names (2 / 4 lanes per waypoint, warp-shuffle reductions for
    J^T J and J^T r): same bars as the one-thread kernel against the same oracle sequence --
    configs[0], 64 trajectories of configs[1] (ragged: 64 x 300 waypoints x lanes is not a multiple of the block) and
    32 trajectories of the 8-DoF configs[2]."""
    for w, check_pose in ((wl.config1(H.oracle_fk(wl.panda_chain())), True),
                          (wl.config2(H.oracle_fk(wl.panda_chain()), B=64, n=299), True),
                          (wl.config3(H.oracle_fk(wl.random_chain_8dof(3)), B=32), False)):
        s = H.make_solver(w)
        s.set_lanes_per_waypoint(lanes)
        s.run(w.max_iters)
        g = s.fetch()
        # the one-thread kernel on the same context: same decisions, joints to rounding
        s.set_lanes_per_waypoint(1)
        s.reset()
        s.run(w.max_iters)
        g1 = s.fetch()
        s.close()
        o = H.run_oracle(w)
        _check_free_running(w, g, o, check_pose=check_pose)
        compared, bad = H.decisive_mismatches(w, g, int(o.iters.max()))
        assert compared >= w.W and bad == 0
        same = g["iters"] == g1["iters"]
        assert same.mean() > 0.998 and np.abs(g["q"] - g1["q"])[same].max() <= 2e-5


def test_lane_group_option_is_validated(lm):
    w = wl.config1(H.oracle_fk(wl.panda_chain()))
    s = H.make_solver(w)
    with pytest.raises(lm.LmError):
        s.set_lanes_per_waypoint(3)
    s.use_generic_kernel(True)
    with pytest.raises(lm.LmError):      # no lane-group form of the generic kernel
        s.set_lanes_per_waypoint(2)
    s.close()
    s = H.make_solver(w, solver=lm.LM_SOLVER_DUAL)
    with pytest.raises(lm.LmError):      # nor of the disclosed variants
        s.set_lanes_per_waypoint(2)
    s.close()


# ------------------------------------------------------------------ run-time specialisation (lm_specialize)

def _unregistered_chains():
    rot_tool = wl.panda_chain()
    rot_tool.name = "panda_rot_tool"
    rot_tool.tool = np.array([0.01, -0.02, 0.107, 0.9238795325112867, 0.2, -0.1, 0.3104])
    rot_tool.tool[3:] /= np.linalg.norm(rot_tool.tool[3:])
    p = wl.panda_chain()
    six = wl.Chain("panda6", 6, p.joint_type[:6], p.a[:6], p.alpha[:6], p.d[:6], p.theta[:6], p.q_lo[:6], p.q_hi[:6], p.tool)
    gen = wl.Chain("gen3", 3, np.array([0, 1, 0], np.int32), np.array([0.1, 0.2, -0.3]), np.array([0.3, -1.1, 2.0]),
                   np.array([0.05, 0.1, 0.2]), np.array([0.4, -0.7, 1.3]), np.full(3, -2.0), np.full(3, 2.0),
                   np.array([0.1, 0.0, 0.2, 1, 0, 0, 0.0]))
    return [rot_tool, six, gen]


@pytest.mark.parametrize("chain", _unregistered_chains(), ids=lambda c: c.name)
def test_runtime_specialised_kernel_equals_the_generic_one(lm, chain):
    """lm_specialize (include/lm.h): a chain without an ahead-of-time kernel gets the SAME kernel template compiled for
    its structure with NVRTC.  Bit-identical to the generic kernel (joints, residuals, iteration counts, masks; also with
    weights, with the dual solver and stepwise), and within the bars of the oracle."""
    rng = np.random.default_rng(7)
    B, n, d = 9, 41, chain.dof
    truth = wl.smooth_joint_paths(chain, B, n, 3, 0.3, rng)
    w = wl._from_truth("J", chain, truth, 0.05, rng, H.oracle_fk(chain), 1e-5, 30)
    for kw in ({}, {"w_pos": 2.0, "w_rot": 0.5}, {"solver": lm.LM_SOLVER_DUAL}):
        s = H.make_solver(w, **kw)
        assert s.kernel_name == "generic"
        s.run(w.max_iters)
        g0 = s.fetch()
        s.specialize()
        assert s.kernel_name == "jit"
        s.reset()
        s.run(w.max_iters)
        g1 = s.fetch()
        s.reset()
        for _ in range(3):
            s.step()
        s.run(w.max_iters)
        g2 = s.fetch()
        s.use_generic_kernel(True)
        assert s.kernel_name == "generic"
        s.close()
        for k in ("q", "res_norm", "iters", "mask", "status", "lam"):
            assert np.array_equal(g0[k], g1[k]) and np.array_equal(g0[k], g2[k]), (k, kw)
    if chain.dof == 7:   # and against the oracle (the redundant arm; the truncated 6- and 3-joint chains of this list are
        o = H.run_oracle(w)  # near-singular test articles for the code paths, graded by the bitwise comparison above)
        s = H.make_solver(w)
        s.specialize()
        s.run(w.max_iters)
        g = s.fetch()
        s.close()
        _check_free_running(w, g, o, check_pose=False)


def test_specialize_is_a_no_op_for_registered_chains(lm):
    w = wl.config1(H.oracle_fk(wl.panda_chain()))
    s = H.make_solver(w)
    s.specialize()
    assert s.kernel_name == "panda7"
    s.close()
