"""Bit-stability (P11), edge cases and API behaviour of the CUDA path -- needs a B200."""
import numpy as np
import pytest

from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl

import helpers as H

pytestmark = pytest.mark.gpu

KEYS = ("q", "res_norm", "pos_err", "rot_err", "lam", "iters", "mask", "status")


@pytest.fixture(scope="module")
def lm():
    from paper_2309_09102_b200 import build, lm as _lm
    build.build()
    return _lm


def same_bits(a, b, keys=KEYS, sl=None):
    for k in keys:
        x, y = a[k], b[k]
        if sl is not None:
            y = y[sl]
        assert np.array_equal(x.view(np.uint32) if x.dtype == np.float32 else x,
                              y.view(np.uint32) if y.dtype == np.float32 else y), k


@pytest.fixture(scope="module")
def w_small():
    return wl.config2(H.oracle_fk(wl.panda_chain()), B=7, n=101)  # W = 707: ragged tail


def test_bitwise_repeatable_and_launch_geometry_independent(lm, w_small):
    ref = H.run_gpu(w_small)
    same_bits(H.run_gpu(w_small), ref)
    for block in (32, 64, 96, 256):
        s = H.make_solver(w_small)
        s.set_launch(block)
        s.run(w_small.max_iters)
        same_bits(s.fetch(), ref)
        s.close()


def test_bits_independent_of_batch_composition(lm, w_small):
    ref = H.run_gpu(w_small)
    sub = w_small.subset(slice(2, 5))
    same_bits(H.run_gpu(sub), ref, sl=slice(2 * w_small.n, 5 * w_small.n))
    # a single waypoint on its own
    i = 3 * w_small.n + 17
    one = wl.Workload("one", w_small.chain, 1, 1, w_small.target_pos[i:i + 1], w_small.target_quat[i:i + 1],
                      w_small.seeds[i:i + 1], w_small.tol, w_small.max_iters)
    same_bits(H.run_gpu(one), ref, sl=slice(i, i + 1))


@pytest.mark.parametrize("cfg", ["tol", "fixed"])
def test_run_equals_repeated_steps(lm, w_small, cfg):
    w = w_small if cfg == "tol" else wl.Workload("f", w_small.chain, w_small.B, w_small.n, w_small.target_pos,
                                                 w_small.target_quat, w_small.seeds, 0.0, 9)
    N = 9
    ref = H.run_gpu(w, max_iters=N)
    s = H.make_solver(w)
    for _ in range(N):
        s.step()
    got = s.fetch()
    s.close()
    same_bits(got, ref, keys=("q", "res_norm", "lam", "iters", "mask"))
    assert np.array_equal(got["status"] & 1, ref["status"] & 1)
    # resumed run: run(4) then run(9) == run(9); reset restarts from the seeds
    s = H.make_solver(w)
    s.run(4)
    mid = s.fetch()
    assert mid["iters"].max() <= 4
    s.run(N)
    same_bits(s.fetch(), ref)
    s.reset()
    s.run(N)
    same_bits(s.fetch(), ref)
    s.close()


def test_shared_targets_host_inputs_and_device_fetch(lm):
    ch = wl.panda_chain()
    w1 = wl.config2(H.oracle_fk(ch), B=1, n=77)
    B = 5
    rng = np.random.default_rng(7)
    seeds = np.clip(np.tile(w1.seeds, (B, 1)) + rng.normal(size=(B * 77, 7)).astype(np.float32) * 0.02,
                    ch.q_lo.astype(np.float32) + 1e-6, ch.q_hi.astype(np.float32) - 1e-6).astype(np.float32)
    tiled = wl.Workload("tiled", ch, B, 77, np.tile(w1.target_pos, (B, 1)), np.tile(w1.target_quat, (B, 1)), seeds,
                        w1.tol, w1.max_iters)
    ref = H.run_gpu(tiled)
    prm = lm.lm_default_params(lambda0=tiled.lambda0, tol=tiled.tol)
    s = lm.Solver(ch, B, 77, w1.target_pos, w1.target_quat, seeds, params=prm, shared_targets=True)
    s.run(tiled.max_iters)
    same_bits(s.fetch(), ref)
    same_bits(s.fetch(host=False), ref)   # lm_fetch into device buffers
    s.close()
    same_bits(H.run_gpu(tiled, host_inputs=True), ref)  # LM_MEM_HOST: pinned host inputs
    s = lm.Solver(ch, B, 77, w1.target_pos, w1.target_quat, seeds, params=prm, shared_targets=True, host_inputs=True)
    s.run(tiled.max_iters)
    same_bits(s.fetch(), ref)
    s.close()


@pytest.mark.parametrize("W", [1, 31, 33, 129])
def test_ragged_sizes(lm, W):
    w = wl.config2(H.oracle_fk(wl.panda_chain()), B=1, n=W)
    g, o = H.run_gpu(w), H.run_oracle(w)
    assert np.abs(g["q"] - o.q).max() <= H.TOL_Q and np.all((g["status"] & 1) == 1)
    assert g["total_waypoint_iters"] == g["iters"].sum()


def test_zero_iterations_and_already_converged(lm, w_small):
    g = H.run_gpu(w_small, max_iters=0)
    assert np.array_equal(g["q"], w_small.seeds) and np.all(g["iters"] == 0) and np.all(g["mask"] == 0)
    assert np.all(g["lam"] == np.float32(w_small.lambda0))
    o = H.run_oracle(w_small, max_iters=0)
    assert np.abs(g["res_norm"] - o.res_norm).max() < 1e-6
    # fetch before any run is the same thing
    s = H.make_solver(w_small)
    g2 = s.fetch()
    s.close()
    same_bits(g2, g)
    # seeds that already meet tol: frozen at once, zero iterations
    ch = w_small.chain
    q = np.clip(w_small.truth, ch.q_lo, ch.q_hi).astype(np.float32)
    p, R = orc.fk(ch, q.astype(np.float64))
    at = wl.Workload("at", ch, w_small.B, w_small.n, p.astype(np.float32), wl._R_to_quat_wxyz(R).astype(np.float32),
                     q, 1e-5, 50)
    g = H.run_gpu(at)
    assert np.all(g["iters"] == 0) and np.all(g["status"] == 1) and np.array_equal(g["q"], q)
    assert g["converged_trajectories"] == at.B


def test_weights_match_oracle(lm):
    w = wl.config2(H.oracle_fk(wl.panda_chain()), B=4, n=64)
    w = wl.Workload(w.name, w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, 0.0, 8)
    g = H.run_gpu(w, w_pos=2.0, w_rot=0.5)
    o = H.run_oracle(w, w_pos=2.0, w_rot=0.5)
    assert np.abs(g["q"] - o.q).max() <= H.TOL_Q
    assert np.abs(g["pos_err"] - o.pos_err).max() < 1e-6 and np.abs(g["rot_err"] - o.rot_err).max() < 1e-6
    g1 = H.run_gpu(w)
    assert np.abs(g1["q"] - g["q"]).max() > 1e-6  # the weights do change the iteration


def test_bad_inputs_do_not_poison_neighbours(lm, w_small):
    ref = H.run_gpu(w_small)
    seeds = w_small.seeds.copy()
    bad = [5, 64, 300]
    seeds[5, 2] = np.nan
    seeds[64, :] = np.inf
    tq = w_small.target_quat.copy()
    tp = w_small.target_pos.copy()
    tp[300] = [5.0, 5.0, 5.0]  # far outside the workspace: unreachable
    w = wl.Workload("bad", w_small.chain, w_small.B, w_small.n, tp, tq, seeds, w_small.tol, 20)
    g = H.run_gpu(w)
    ok = np.ones(w.W, bool)
    ok[bad] = False
    refc = H.run_gpu(wl.Workload("r", w.chain, w.B, w.n, w_small.target_pos, w_small.target_quat, w_small.seeds, w.tol, 20))
    for k in ("q", "iters", "mask"):
        assert np.array_equal(g[k][ok], refc[k][ok]), k
    assert np.all(g["status"][[5, 64]] & (lm.LM_ST_BREAKDOWN | lm.LM_ST_NONFINITE))
    assert not np.any(g["status"][[5, 64]] & lm.LM_ST_FROZEN) and np.all(g["mask"][[5, 64]] == 0)
    assert np.all(g["iters"][[5, 64]] == 20)
    # unreachable target: finite, inside the limits, not converged, hits the iteration limit
    assert np.all(np.isfinite(g["q"][300])) and g["status"][300] & lm.LM_ST_MAXITER
    assert np.all(g["q"][300] >= w.chain.q_lo.astype(np.float32)) and np.all(g["q"][300] <= w.chain.q_hi.astype(np.float32))
    assert g["res_norm"][300] > 1.0
    assert ref["q"].shape == g["q"].shape


def test_joint_limit_clamp(lm):
    """targets reachable only outside a narrowed limit => q stays on the limit."""
    ch = wl.panda_chain()
    w = wl.config2(H.oracle_fk(ch), B=2, n=50)
    narrow = wl.panda_chain()
    narrow.q_hi = np.minimum(narrow.q_hi, w.truth.max(axis=0) - 0.05)
    narrow.q_lo = np.maximum(narrow.q_lo, w.truth.min(axis=0) + 0.05)
    seeds = np.clip(w.seeds, narrow.q_lo.astype(np.float32) + 1e-6, narrow.q_hi.astype(np.float32) - 1e-6)
    wn = wl.Workload("narrow", narrow, w.B, w.n, w.target_pos, w.target_quat, seeds, 0.0, 12)
    g, o = H.run_gpu(wn), H.run_oracle(wn)
    assert np.all(g["q"] >= narrow.q_lo.astype(np.float32)) and np.all(g["q"] <= narrow.q_hi.astype(np.float32))
    assert np.any(g["status"] & lm.LM_ST_CLAMPED)
    # Free-running on a non-smooth problem.  A waypoint held on a limit ends at a CONSTRAINED minimum with F > 0: there
    # the fp64 oracle goes on "accepting" steps that lower F by 1e-10 relative, fp32 cannot see such a decrease and
    # rejects, lambda parts and q slides along the flat valley floor (measured: 4 of 100 waypoints, 3-5e-4 rad, same F).
    # Those decisions are not decisive (margin < 1e-3), so the protocol is the one of configs[3]: strict sequence and
    # joint parity on every waypoint whose ORACLE decisions are all clear-cut, identical decisive prefixes and the same
    # cost on all.  Single clamped steps are strict: the next test.
    rep = H.check_chaotic_config(wn, g, o, 12, min_clear=0.5)
    compared, bad = H.decisive_mismatches(wn, g, 12)
    assert compared > 3 * wn.W and bad == 0
    rel = np.abs(g["res_norm"] - o.res_norm) / np.maximum(o.res_norm, 1e-5)
    print("clamp free-running: max relative |r| difference over all waypoints", rel.max())
    assert rel.max() <= 0.05            # both sides sit in the same valley (not asserted to 1e-5: the sequences parted)


def test_clamped_trial_points_teacher_forced(lm):
    """PAPER.md:L170 / DESIGN R6 where strict parity IS attainable: single steps from the oracle's own iterates on the
    narrowed-limit problem, restricted to the waypoints whose ORACLE trial point was clamped (at least one joint on a
    limit).  Every joint of the GPU's trial point within 1e-4 of the oracle's, the clamped joints exactly on the fp32
    limit, the decision identical wherever the oracle's margin is clear, the CLAMPED status bit on every accepted
    clamped step -- no fraction, no percentile."""
    ch = wl.panda_chain()
    w = wl.config2(H.oracle_fk(ch), B=2, n=50)
    narrow = wl.panda_chain()
    narrow.q_hi = np.minimum(narrow.q_hi, w.truth.max(axis=0) - 0.05)
    narrow.q_lo = np.maximum(narrow.q_lo, w.truth.min(axis=0) + 0.05)
    seeds = np.clip(w.seeds, narrow.q_lo.astype(np.float32) + 1e-6, narrow.q_hi.astype(np.float32) - 1e-6)
    n_it = 12
    wn = wl.Workload("narrow", narrow, w.B, w.n, w.target_pos, w.target_quat, seeds, 0.0, n_it)
    lo32, hi32 = narrow.q_lo.astype(np.float32), narrow.q_hi.astype(np.float32)
    lo32 = np.where(lo32.astype(np.float64) < narrow.q_lo, np.nextafter(lo32, np.float32(np.inf)), lo32)   # rounded inward,
    hi32 = np.where(hi32.astype(np.float64) > narrow.q_hi, np.nextafter(hi32, np.float32(-np.inf)), hi32)  # as lm.h states
    tr = H.oracle_trace(wn, n_it)
    s = H.make_solver(wn)
    s.enable_trace()
    tp, tq = wn.target_pos.astype(np.float64), wn.target_quat.astype(np.float64)
    n_clamped, n_decided, n_acc_clamped = 0, 0, 0
    for k, (b, a) in enumerate(tr):
        q32, lam32 = b.q.astype(np.float32), b.lam.astype(np.float32)
        s.set_state(q32, lam32)
        s.step()
        g = s.fetch()
        st = orc.State(q=q32.astype(np.float64), lam=lam32.astype(np.float64), iters=np.zeros(wn.W, np.int32),
                       mask=np.zeros(wn.W, np.uint64), status=np.zeros(wn.W, np.uint32))
        orc.advance(narrow, H.oracle_params(wn), tp, tq, st, 1)
        on_lo, on_hi = st.trial_q == narrow.q_lo[None, :], st.trial_q == narrow.q_hi[None, :]
        cl = (on_lo | on_hi).any(axis=1)                              # the oracle's trial point is clamped
        if not cl.any():
            continue
        n_clamped += int(cl.sum())
        assert np.abs(g["trial_q"] - st.trial_q)[cl].max() <= H.TOL_Q
        assert np.array_equal(g["trial_q"][on_lo], np.broadcast_to(lo32, on_lo.shape)[on_lo])
        assert np.array_equal(g["trial_q"][on_hi], np.broadcast_to(hi32, on_hi.shape)[on_hi])
        # |r+| agrees to the fp32 floor of the pose (1e-6) plus what the difference of the two trial points explains
        # (|dr| <= |J|_2 |dq|_2 < 8 |dq|_inf on this arm)
        dtr = np.abs(g["trial_q"] - st.trial_q).max(axis=1)
        assert np.all(np.abs(np.sqrt(g["F_trial"]) - np.sqrt(st.F_trial))[cl] <= 1e-6 + 8 * dtr[cl])
        dec = cl & H.decisive(st.F_before, st.F_trial)
        acc_g = (g["mask"] & np.uint64(1)) == 1
        assert np.array_equal(acc_g[dec], (st.accepted == 1)[dec])
        n_decided += int(dec.sum())
        both = dec & acc_g
        assert np.all(g["status"][both] & lm.LM_ST_CLAMPED) and np.all(st.status[both] & 16)
        n_acc_clamped += int(both.sum())
    s.close()
    assert n_clamped >= 100 and n_decided >= 50 and n_acc_clamped >= 10, (n_clamped, n_decided, n_acc_clamped)


@pytest.mark.parametrize("d", [1, 2, 3, 4, 5, 6])
def test_low_dof_chains(lm, d):
    rng = np.random.default_rng(40 + d)
    ch = wl.Chain(f"gen{d}", d, (rng.random(d) < 0.25).astype(np.int32), rng.uniform(-0.3, 0.3, d),
                  rng.choice([0.0, np.pi / 2, -np.pi / 2, 0.7], d), rng.uniform(0.0, 0.3, d), rng.uniform(-1, 1, d),
                  np.full(d, -2.0), np.full(d, 2.0), np.array([0.05, 0.0, 0.1, 1, 0, 0, 0.0]))
    truth = rng.uniform(-1.0, 1.0, size=(1, 90, d))
    w = wl._from_truth("low", ch, truth, 0.05, rng, H.oracle_fk(ch), 0.0, 10)
    g, o = H.run_gpu(w), H.run_oracle(w)
    assert np.array_equal(g["iters"], o.iters)
    # under-actuated chains (d < 6) sit at a least-squares point; lambda_min keeps it well conditioned
    assert np.abs(g["q"] - o.q).max() <= H.TOL_Q
    rel = np.abs(g["res_norm"] - o.res_norm) / np.maximum(o.res_norm, 1e-5)
    print("clamp free-running: max relative |r| difference over all waypoints", rel.max())
    assert rel.max() <= 0.05            # both sides sit in the same valley (not asserted to 1e-5: the sequences parted)


def test_solver_variants(lm, w_small):
    o = H.run_oracle(w_small)
    for kw in (dict(refine_steps=0), dict(refine_steps=2), dict(fast_sincos=1)):
        g = H.run_gpu(w_small, **kw)
        dq = np.abs(g["q"] - o.q).max(axis=1)
        assert np.all((g["status"] & 1) == 1)
        print("solver variant", kw, "max |dq|", dq.max())
        assert dq.max() <= H.TOL_Q, kw     # every waypoint (measured: 5.2e-5 without refinement, 8e-7 with two steps, 6.1e-5 fast sincos)


def test_api_errors_on_device(lm, w_small):
    s = H.make_solver(w_small)
    with pytest.raises(lm.LmError):
        lm.lm_run(s._ctx, 65)
    with pytest.raises(lm.LmError):
        lm.lm_set_option(s._ctx, lm.LM_OPT_BLOCK_THREADS, 40)
    with pytest.raises(lm.LmError):
        lm.lm_set_option(s._ctx, 99, 1)
    with pytest.raises(lm.LmError):
        lm.lm_fk(s._ctx, 0, 10, 0, 0)
    n0 = lm.lm_launch_count()
    s.run(3)
    assert lm.lm_launch_count() == n0 + 1   # the whole LM loop is ONE launch
    s.close()


def test_specialised_kernels_equal_generic(lm):
    """Chains whose structure is registered in csrc/lm_specs.cuh run a compile-time specialised
    kernel; it must return the generic kernel's values (only multiplications by exact 0 / +-1 and
    additions of exact 0 are removed; the sign of a zero may differ, nothing else)."""
    cases = [("panda7", wl.config2(H.oracle_fk(wl.panda_chain()), B=5, n=131)),
             ("rand8", wl.config3(H.oracle_fk(wl.random_chain_8dof(3)), B=5, n=131)),
             ("panda7", wl.config4(H.oracle_fk(wl.panda_chain()), B=5, n=131))]
    for name, w in cases:
        s = H.make_solver(w)
        assert s.kernel_name == name
        s.run(w.max_iters)
        a = s.fetch()
        s.use_generic_kernel(True)
        assert s.kernel_name == "generic"
        s.reset()
        s.run(w.max_iters)
        b = s.fetch()
        s.close()
        for k in ("q", "res_norm", "lam"):
            assert np.array_equal(a[k], b[k]), (name, k)   # value equality (+0 == -0)
        for k in ("iters", "mask", "status"):
            assert np.array_equal(a[k], b[k]), (name, k)
    # anything else runs the generic kernel: other robots, a rotated tool, a theta offset
    other = wl.panda_chain()
    other.theta = other.theta + np.array([0, 0, 0.1, 0, 0, 0, 0])
    s = H.make_solver(wl.Workload("o", other, 1, 4, cases[0][1].target_pos[:4], cases[0][1].target_quat[:4],
                                  cases[0][1].seeds[:4], 0.0, 2))
    assert s.kernel_name == "generic"
    s.close()
    c5 = wl.random_chain_8dof(5)   # same recipe, different structure
    s = H.make_solver(wl.Workload("o", c5, 1, 4, cases[1][1].target_pos[:4], cases[1][1].target_quat[:4],
                                  cases[1][1].seeds[:4], 0.0, 2))
    assert s.kernel_name == "generic"
    s.close()


@pytest.mark.gpu
@pytest.mark.parametrize("chunks", [1, 3, 8])
def test_solve_host_pipelined_equals_the_stepwise_path(chunks):
    """lm_solve_host (host arrays, chunked + pipelined over streams) returns exactly what
    lm_init + lm_run + lm_fetch return: waypoints are independent."""
    import torch
    from paper_2309_09102_b200 import lm, workloads as wl
    from oracle import lm_oracle as orc
    ch = wl.panda_chain()
    w = wl.config2(lambda q: orc.fk(ch, q), B=13, n=37)
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol)
    ref_s = lm.Solver(ch, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm)
    ref_s.run(w.max_iters)
    ref = ref_s.fetch()
    ref_s.close()
    d, W = 7, w.W
    soa = lambda x: torch.from_numpy(np.ascontiguousarray(np.asarray(x, np.float32).T)).pin_memory()
    tp, tq, seeds = soa(w.target_pos), soa(w.target_quat), soa(w.seeds)
    nbytes = lm.lm_solve_host_workspace_bytes(d, w.B, w.n, chunks)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    ptr = (ws.data_ptr() + 255) // 256 * 256
    cchain, keep = lm.make_chain(ch)
    q = torch.empty((d, W), dtype=torch.float32).pin_memory()
    res = torch.empty(W, dtype=torch.float32).pin_memory()
    its = torch.empty(W, dtype=torch.int32).pin_memory()
    sts = torch.empty(W, dtype=torch.int32).pin_memory()
    msk = torch.empty(W, dtype=torch.int64).pin_memory()
    conv = torch.empty(w.B, dtype=torch.uint8).pin_memory()
    pb = lm.LmProblem(w.B, w.n, tp.data_ptr(), tq.data_ptr(), 0, seeds.data_ptr(), lm.LM_MEM_HOST, ptr, nbytes)
    st = lm.LmStats(res.data_ptr(), None, None, None, its.data_ptr(), msk.data_ptr(), sts.data_ptr(), conv.data_ptr(), None, 0, 0)
    lm.lm_solve_host(cchain, pb, prm, w.max_iters, chunks, q.data_ptr(), st)
    assert np.array_equal(q.numpy().T, ref["q"])
    assert np.array_equal(res.numpy(), ref["res_norm"])
    assert np.array_equal(its.numpy(), ref["iters"])
    assert np.array_equal(msk.numpy().view(np.uint64), ref["mask"])
    assert np.array_equal(sts.numpy().view(np.uint32), ref["status"])
    assert np.array_equal(conv.numpy(), ref["traj_converged"])
    assert st.total_waypoint_iters == ref["total_waypoint_iters"]
    assert st.converged_trajectories == ref["converged_trajectories"]
    with pytest.raises(lm.LmError):
        lm.lm_solve_host(cchain, pb, prm, w.max_iters, w.B + 1, q.data_ptr(), st)
    # the same through a kept handle (lm_pipe_*), twice, on a caller's stream that still has the production of the host
    # inputs queued: the pipeline must start after it and later work on the stream after the pipeline
    pipe = lm.lm_pipe_create(8)
    stream = torch.cuda.Stream()
    dev_seeds = torch.from_numpy(np.ascontiguousarray(w.seeds.T)).cuda()
    for rep in range(2):
        q.zero_(); res.zero_(); seeds.zero_()
        with torch.cuda.stream(stream):
            seeds.copy_(dev_seeds, non_blocking=True)           # inputs arrive on the caller's stream
            lm.lm_pipe_solve(pipe, cchain, pb, prm, w.max_iters, chunks, q.data_ptr(), st, int(stream.cuda_stream))
        assert np.array_equal(q.numpy().T, ref["q"]) and np.array_equal(res.numpy(), ref["res_norm"])
        assert st.total_waypoint_iters == ref["total_waypoint_iters"]
    with pytest.raises(lm.LmError):                              # more chunks than the handle was created for
        lm.lm_pipe_solve(pipe, cchain, pb, prm, w.max_iters, 9, q.data_ptr(), st)
    lm.lm_pipe_destroy(pipe)


# ------------------------------------------------------------------ the iteration limit of the ABI (LM_MAX_ITERS = 64)

def test_iteration_limit_64(lm):
    """lm_run(ctx, 64) with tol = 0: iteration 63 is bit 63 of the 64-bit accept mask and the 8-bit counter packed next
    to the frozen flag reaches 64.  (a) lambda0 = 100, nu_down = 1.01: 64 small damped steps, EVERY one a decisive
    accept in the oracle (checked below from the oracle alone) -> iters == 64, mask == 2^64 - 1 bit for bit, status
    MAXITER, joints within the bar.  (b) the default constants: the run reaches the fp32 floor long before 64, where
    decisions are noise -> iters == 64 both sides, joints within the bar, decisive bits equal.  (c) 64 x lm_step
    returns the bits of lm_run(64); 65 is rejected."""
    ch = wl.panda_chain()
    c1 = wl.config1(H.oracle_fk(ch))
    wa = wl.Workload("lim64a", ch, c1.B, c1.n, c1.target_pos, c1.target_quat, c1.seeds, 0.0, 64, 100.0)
    tr = H.oracle_trace(wa, 64, nu_down=1.01)
    Fb, Ft = np.stack([a.F_before for _, a in tr], 1), np.stack([a.F_trial for _, a in tr], 1)
    assert H.decisive(Fb, Ft).all() and all((a.accepted == 1).all() for _, a in tr)
    o = H.run_oracle(wa, nu_down=1.01)
    g = H.run_gpu(wa, nu_down=1.01)
    assert np.all(o.iters == 64) and np.all(g["iters"] == 64)
    assert np.all(o.mask == np.uint64(0xFFFFFFFFFFFFFFFF)) and np.array_equal(g["mask"], o.mask)
    assert np.all(g["status"] & lm.LM_ST_MAXITER) and not np.any(g["status"] & lm.LM_ST_FROZEN)
    assert np.array_equal(g["status"] & 3, o.status & 3)
    assert np.abs(g["q"] - o.q).max() <= H.TOL_Q
    assert np.abs(g["lam"] / o.lam - 1.0).max() <= 1e-5            # lambda0 / 1.01^64, 64 roundings
    assert np.abs(g["res_norm"] - o.res_norm).max() <= 2e-6
    # (c) on the same problem
    s = H.make_solver(wa, nu_down=1.01)
    for _ in range(64):
        s.step()
    same_bits(s.fetch(), g, keys=("q", "res_norm", "lam", "iters", "mask"))
    s.step()                                                       # a 65th iteration has no mask bit: nothing executes
    same_bits(s.fetch(), g, keys=("q", "res_norm", "lam", "iters", "mask"))
    with pytest.raises(lm.LmError):
        lm.lm_run(s._ctx, 65)
    s.close()
    # (b)
    wb = wl.Workload("lim64b", ch, c1.B, c1.n, c1.target_pos, c1.target_quat, c1.seeds, 0.0, 64, c1.lambda0)
    o, g = H.run_oracle(wb), H.run_gpu(wb)
    assert np.all(o.iters == 64) and np.all(g["iters"] == 64) and np.all(g["status"] & lm.LM_ST_MAXITER)
    assert np.abs(g["q"] - o.q).max() <= H.TOL_Q
    compared, bad = H.decisive_mismatches(wb, g, 64)
    assert compared >= 100 and bad == 0, (compared, bad)
