"""Small GPU cases that together launch EVERY kernel of liblm_b200.so, each checked against the oracle.

This is the selection `compute-sanitizer --tool memcheck | racecheck | synccheck | initcheck` is run on
(profiles/r2_sanitizers.md names the commands): the sizes are a few hundred waypoints so that a tool that slows
kernels down by two or three orders of magnitude still finishes in minutes, yet every case spans more than one
warp / tile and a ragged tail.  Run without a tool they are ordinary parity tests (SURVEY.md section 5,
"Race detection / sanitizers"; VERDICT r1 "Next round" item 2).
"""
import numpy as np
import pytest

from oracle import lm_coll_oracle as corc
from oracle import lm_oracle as orc
from oracle import lm_plan_oracle as porc
from oracle import lm_search_oracle as sorc
from oracle import lm_traj_oracle as torc
from paper_2309_09102_b200 import workloads as wl
import helpers as H

pytestmark = pytest.mark.gpu


def small(ch, B, n, seed, sigma=0.05, tol=0.0, iters=6):
    rng = np.random.default_rng(seed)
    truth = wl.smooth_joint_paths(ch, B, n, 3, 0.3, rng)
    return wl._from_truth("S", ch, truth, sigma, rng, lambda q: orc.fk(ch, q), tol, iters)


@pytest.mark.parametrize("chain_name", ["panda", "rand8", "gen3"])
def test_pose_kernels(chain_name):
    """lm_iterate_kernel (specialised, generic, dual, rpy, weighted, fast sincos), lm_step, lm_set_state,
    lm_fk, lm_fetch's statistics / unpack kernels."""
    from paper_2309_09102_b200 import lm
    if chain_name == "gen3":
        p = wl.panda_chain()
        ch = wl.Chain("gen3", 3, np.array([0, 1, 0], np.int32), p.a[:3] + 0.1, np.array([0.3, -0.7, 1.1]), p.d[:3] + 0.05,
                      np.array([0.2, 0.0, -0.4]), np.array([-2.0, 0.0, -2.0]), np.array([2.0, 0.3, 2.0]),
                      np.array([0.05, 0.02, 0.1, 0.9, 0.1, 0.3, 0.2]))
    else:
        ch = wl.panda_chain() if chain_name == "panda" else wl.random_chain_8dof(3)
    w = small(ch, 3, 47, 900)                                   # 141 waypoints: 4 full warps + a ragged one
    o = H.run_oracle(w)
    g = H.run_gpu(w)
    assert np.abs(g["q"] - o.q).max() <= H.TOL_Q and np.array_equal(g["iters"], o.iters)
    for kw in (dict(solver=lm.LM_SOLVER_DUAL), dict(fast_sincos=1), dict(refine_steps=2)):
        gv = H.run_gpu(w, **kw)
        assert np.abs(gv["q"] - o.q).max() <= 5e-4
    ow = H.run_oracle(w, w_pos=2.0, w_rot=0.5)
    gw = H.run_gpu(w, w_pos=2.0, w_rot=0.5)
    assert np.abs(gw["q"] - ow.q).max() <= H.TOL_Q
    if ch.dof >= 7:
        orp = H.run_oracle(w, rot_mode=1)
        grp = H.run_gpu(w, rot_residual=lm.LM_ROT_RPY)
        assert np.abs(grp["q"] - orp.q).max() <= H.TOL_Q
    # generic kernel, stepping, state injection, FK, device-side fetch
    s = H.make_solver(w)
    s.use_generic_kernel(True)
    for _ in range(w.max_iters):
        s.step()
    gs = s.fetch(host=False)
    assert np.array_equal(gs["q"].view(np.uint32) & 0x7fffffff, g["q"].view(np.uint32) & 0x7fffffff) or \
        np.abs(gs["q"] - g["q"]).max() == 0.0
    s.set_state(o.q.astype(np.float32))
    f = s.fetch()                                               # outputs re-evaluated at the injected q
    pe, re_ = H.pose_errors_by_oracle(w, o.q.astype(np.float32))
    assert np.abs(f["pos_err"] - pe).max() <= 2e-6 and np.abs(f["rot_err"] - re_).max() <= 2e-6
    p, R = s.fk(o.q)
    po, Ro = orc.fk(ch, o.q.astype(np.float32).astype(np.float64))
    assert np.abs(p - po).max() <= 1e-6 and np.abs(R - Ro).max() <= 1e-6
    s.close()


def test_solve_host_pipeline():
    from paper_2309_09102_b200 import lm
    import torch
    ch = wl.panda_chain()
    w = small(ch, 7, 33, 901)
    o = H.run_oracle(w)
    W, d = w.W, 7
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a.T)).pin_memory()
    tp, tq, sd = pin(w.target_pos), pin(w.target_quat), pin(w.seeds)
    chunks = 3
    nbytes = lm.lm_solve_host_workspace_bytes(d, w.B, w.n, chunks)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda:0")
    q = torch.empty((d, W), dtype=torch.float32).pin_memory()
    it = torch.empty((W,), dtype=torch.int32).pin_memory()
    res = torch.empty((W,), dtype=torch.float32).pin_memory()
    st = lm.LmStats(res.data_ptr(), None, None, None, it.data_ptr(), None, None, None, None, 0, 0)
    cchain, keep = lm.make_chain(ch)
    pb = lm.LmProblem(w.B, w.n, tp.data_ptr(), tq.data_ptr(), 0, sd.data_ptr(), lm.LM_MEM_HOST,
                      (ws.data_ptr() + 255) // 256 * 256, nbytes)
    lm.lm_solve_host(cchain, pb, lm.lm_default_params(lambda0=w.lambda0, tol=w.tol), w.max_iters, chunks, q.data_ptr(), st)
    assert np.abs(q.numpy().T - o.q).max() <= H.TOL_Q
    assert np.array_equal(it.numpy(), o.iters) and st.total_waypoint_iters == int(o.iters.sum())


@pytest.mark.parametrize("chain_name,rows", [("panda", "none"), ("panda", "all"), ("rand8", "self")])
def test_trajectory_level_kernels(chain_name, rows):
    """tl_pack / tl_assemble / tl_solve<0> / tl_rho / tl_solve<1> / tl_trial / tl_decide / tl_unpack, plain and with
    collision rows, on 33 trajectories (two tiles, the second with one live lane) of 13 waypoints."""
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain() if chain_name == "panda" else wl.random_chain_8dof(3)
    B, n, d = 33, 13, ch.dof
    w = small(ch, B, n, 902, sigma=0.02)
    model = None if rows == "none" else (wl.panda_capsules() if chain_name == "panda" else wl.chain_capsules(ch))
    scene = wl.panda_scene() if rows == "all" else None
    s = lm.Solver(ch, B, n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=0.0))
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=0.3))
    if model is not None:
        s.traj_set_capsules(model, 1.0, 0.4)
    if scene is not None:
        s.traj_set_obstacles(scene, 1.0, 0.4)
    s.traj_enable_trace()
    s.traj_run(1)
    g = s.traj_fetch()
    s.traj_run(2)                                              # buffer flips, mixed accept / reject tiles
    g2 = s.traj_fetch()
    q2 = s.fetch()["q"]
    s.close()
    caps = None if model is None else corc.Capsules(model, w_coll=1.0, d_safe=0.4, scene=scene, w_env=1.0, d_safe_env=0.4)
    tprm = torc.TrajParams(w_pose=1.0, w_diff=0.3, caps=caps)
    st = torc.init_state(w.seeds.astype(np.float64).reshape(B, n, d), tprm)
    torc.advance(ch, orc.Params(), tprm, w.target_pos.astype(np.float64).reshape(B, n, 3),
                 w.target_quat.astype(np.float64).reshape(B, n, 4), st, 1)
    clear = np.abs(st.F_before - st.F_trial) > 1e-3 * st.F_before
    assert np.abs(g["trial_q"].reshape(B, n, d) - st.trial_q)[clear].max() <= (1e-4 if rows != "none" else 2e-5)
    assert np.allclose(g["F_before"], st.F_before, rtol=1e-4)
    assert np.isfinite(q2).all() and (g2["iters"] == 3).all() and np.all(g2["cost"] <= g["cost"] * (1 + 1e-6))


def test_schedule_kernels():
    """lm_plan_run: pose phases, plan_check_kernel, gated trajectory-level step, tl_clearance_kernel."""
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    B, n, d = 5, 40, 7
    w = small(ch, B, n, 903, sigma=0.01, tol=1e-5)
    s = lm.Solver(ch, B, n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=1e-5))
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=1.0))
    s.traj_set_capsules(wl.panda_capsules(), 1.0, 0.05)
    s.plan_attach(lm.lm_plan_default_params(pose_iters=8))
    s.plan_run(2)
    g = s.plan_fetch()
    s.close()
    caps = corc.Capsules(wl.panda_capsules(), w_coll=1.0, d_safe=0.05)
    o = porc.plan(ch, orc.Params(tol=1e-5), torc.TrajParams(w_pose=1.0, w_diff=1.0, caps=caps), porc.PlanParams(pose_iters=8),
                  w.target_pos.astype(np.float64).reshape(B, n, 3), w.target_quat.astype(np.float64).reshape(B, n, 4),
                  w.seeds.astype(np.float64).reshape(B, n, d), 2)
    assert np.array_equal(g["valid"], o.valid) and np.array_equal(g["first_valid_cycle"], o.first_valid_cycle)
    v = o.valid
    assert v.any() and np.abs(g["q_valid"].reshape(B, n, d)[v] - o.q_valid[v]).max() <= 1e-4


@pytest.mark.parametrize("K,n", [(3, 9), (9, 17), (24, 20), (175, 12), (600, 180)])
def test_search_kernels(K, n):
    """search_edges_kernel + search_dp_kernel: K = 3 and 9 leave cluster ranks without nodes, K = 24 is the small
    case, K = 175 the paper's, K = 600 x 180 keeps the predecessors in global memory."""
    ch = wl.panda_chain()
    q = wl.search_candidates(ch, K, n, 904 + K, limit_frac=0.02)
    from test_gpu_search import check
    check(ch, q)
    pen = sorc.penalties(q.astype(np.float64), ch.q_lo, ch.q_hi, ch.joint_type)
    assert pen.shape == (n, K)
