"""Memory-safety and race checks of our own (SURVEY.md section 5 "Race detection / sanitizers").

compute-sanitizer is CLOSED on this GPU pool (gpurun answers "compute-sanitizer is closed on this pool and stays
closed: runs under it have left GPUs needing a reset", profiles/r2_sanitizers.md), so memcheck / initcheck / racecheck
are replaced by what can be observed from outside the kernels:

  * out-of-bounds WRITES: every workspace gets 4 KiB guard bands filled with 0xA5 (GuardedSolver below); after every
    kernel of the library has run on ragged sizes the bands must be intact;
  * reads of UNWRITTEN scratch: the workspace interior is poisoned with 0xFF bytes (fp32 NaN / int -1) instead of
    whatever the allocator hands out; all outputs must be bit-identical to the unpoisoned run;
  * RACES in the hand-rolled producer / consumer mbarrier rings (tl_solve_kernel) and the st.async + remote-mbarrier
    layer hand-off (search_dp_kernel): a race shows as timing dependence, so the same call is repeated while another
    stream keeps every SM busy with a large lm_run (the "SM shared with another stream's kernel" scenario of ADVICE r1):
    every repetition must return the same bits as the quiet run, and must return at all (pytest-timeout).
"""
import numpy as np
import pytest

from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(600)]


def problem(ch, B, n, seed, sigma=0.03):
    rng = np.random.default_rng(seed)
    truth = wl.smooth_joint_paths(ch, B, n, 3, 0.3, rng)
    return wl._from_truth("G", ch, truth, sigma, rng, lambda q: orc.fk(ch, q), 0.0, 8)


def guarded_solver_class():
    """lm.Solver with every workspace it allocates wrapped in guard bands (the stand-in for compute-sanitizer's memcheck /
    initcheck, which is closed on this pool): 4 KiB filled with 0xA5 on either side -- an out-of-bounds WRITE of any
    kernel shows up in guards_intact() -- and the interior poisoned with 0xFF bytes (fp32 NaN, int -1) so that a read
    of memory no kernel has written ends up in the outputs.  Test equipment: it lives here, not in the binding."""
    from paper_2309_09102_b200 import lm

    class GuardedSolver(lm.Solver):
        GUARD_BYTES = 4096

        def __init__(self, *a, **kw):
            self._guards = []
            super().__init__(*a, **kw)

        def _alloc_ws(self, nbytes: int):
            torch, G = self.torch, self.GUARD_BYTES
            t = torch.full((nbytes + 2 * G + 256,), 0xA5, dtype=torch.uint8, device=self.device)
            ptr = (t.data_ptr() + G + 255) // 256 * 256
            off = ptr - t.data_ptr()
            t[off:off + nbytes] = 0xFF
            self._guards.append((t, off, nbytes))
            return t, ptr

        def guards_intact(self) -> bool:
            self.torch.cuda.synchronize(self.device)
            ok = True
            for t, off, nbytes in self._guards:
                ok = ok and bool((t[:off] == 0xA5).all().item()) and bool((t[off + nbytes:] == 0xA5).all().item())
            return ok

    return GuardedSolver


def everything(ch, w, guarded, rows=True):
    """Every entry point of the library on one problem; returns all outputs (numpy) and the solver's guard verdict."""
    from paper_2309_09102_b200 import lm
    out = {}
    cls = guarded_solver_class() if guarded else lm.Solver
    s = cls(ch, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=0.0))
    s.enable_trace()
    s.run(3)
    s.step()
    out["pose"] = s.fetch()
    s.use_generic_kernel(True)
    s.reset()
    s.run(4)
    out["pose_generic"] = s.fetch(host=False)
    s.use_generic_kernel(False)
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=0.3))
    s.traj_enable_trace()
    s.traj_run(2)
    out["traj_plain"] = s.traj_fetch()
    if rows and ch.dof == 7:
        s.traj_set_capsules(wl.panda_capsules(), 1.0, 0.3)
        s.traj_set_obstacles(wl.panda_scene(), 1.0, 0.3)
        s.traj_run(2)
        out["traj_rows"] = s.traj_fetch()
    s.plan_attach(lm.lm_plan_default_params(pose_iters=4))
    s.plan_run(2)
    out["plan"] = s.plan_fetch()
    out["q_after_plan"] = s.fetch()
    if w.B <= 1024:
        out["search"] = s.search()
        if rows and ch.dof == 7:
            out["search_clear"] = s.search(lm.lm_search_default_params(use_clearance=1))
    intact = s.guards_intact() if guarded else True
    s.close()
    return out, intact


def flatten(o, prefix=""):
    for k, v in o.items():
        if isinstance(v, dict):
            yield from flatten(v, prefix + k + ".")
        else:
            yield prefix + k, v


@pytest.mark.parametrize("chain_name,B,n", [("panda", 33, 13), ("panda", 5, 301), ("rand8", 9, 40), ("panda", 1, 1)])
def test_guard_bands_intact_and_no_read_of_unwritten_scratch(chain_name, B, n):
    ch = wl.panda_chain() if chain_name == "panda" else wl.random_chain_8dof(3)
    w = problem(ch, B, n, 700 + B)
    plain, _ = everything(ch, w, guarded=False)
    guarded, intact = everything(ch, w, guarded=True)
    assert intact, "a kernel wrote outside its workspace"
    for (k, a), (k2, b) in zip(flatten(plain), flatten(guarded)):
        assert k == k2
        if isinstance(a, np.ndarray):
            assert np.array_equal(a, b, equal_nan=True), f"{k}: depends on unwritten workspace memory"
        else:
            assert a == b or (a != a and b != b), k


def test_solve_host_guard_bands():
    import torch
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    w = problem(ch, 11, 29, 710)
    W, d, G = w.W, 7, 4096
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a.T)).pin_memory()
    tp, tq, sd = pin(w.target_pos), pin(w.target_quat), pin(w.seeds)
    results = []
    for chunks, poison in ((1, 0x00), (4, 0xFF)):
        nbytes = lm.lm_solve_host_workspace_bytes(d, w.B, w.n, chunks)
        t = torch.full((nbytes + 2 * G + 256,), 0xA5, dtype=torch.uint8, device="cuda:0")
        ptr = (t.data_ptr() + G + 255) // 256 * 256
        off = ptr - t.data_ptr()
        t[off:off + nbytes] = poison
        # host outputs with guard elements of their own
        q = torch.full((d * W + 64,), 7.0, dtype=torch.float32).pin_memory()
        it = torch.full((W + 64,), -7, dtype=torch.int32).pin_memory()
        st = lm.LmStats(None, None, None, None, it.data_ptr() + 128, None, None, None, None, 0, 0)
        cchain, keep = lm.make_chain(ch)
        pb = lm.LmProblem(w.B, w.n, tp.data_ptr(), tq.data_ptr(), 0, sd.data_ptr(), lm.LM_MEM_HOST, ptr, nbytes)
        lm.lm_solve_host(cchain, pb, lm.lm_default_params(tol=0.0), 6, chunks, q.data_ptr() + 128, st)
        torch.cuda.synchronize()
        assert bool((t[:off] == 0xA5).all().item()) and bool((t[off + nbytes:] == 0xA5).all().item())
        assert (q[:32] == 7.0).all() and (q[32 + d * W:] == 7.0).all() and (it[:32] == -7).all() and (it[32 + W:] == -7).all()
        results.append((q[32:32 + d * W].numpy().copy(), it[32:32 + W].numpy().copy()))
    assert np.array_equal(results[0][0], results[1][0]) and np.array_equal(results[0][1], results[1][1])
    assert np.all(results[0][1] == 6)


def test_results_do_not_depend_on_timing():
    """tl_solve_kernel's mbarrier rings and search_dp_kernel's st.async hand-off, repeated while a second stream keeps
    the SMs busy: identical bits every time."""
    import torch
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    big = problem(ch, 2048, 100, 720)
    heavy = lm.Solver(ch, big.B, big.n, big.target_pos, big.target_quat, big.seeds, params=lm.lm_default_params(tol=0.0),
                      stream=torch.cuda.Stream())
    w = problem(ch, 70, 57, 721)
    s = lm.Solver(ch, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=lm.lm_default_params(tol=0.0))
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=0.3))
    s.traj_enable_trace()

    def one_traj():
        s.set_state(w.seeds)
        s.traj_reset()
        s.traj_run(3)
        t = s.traj_fetch()
        return s.fetch()["q"].copy(), t["trial_q"].copy(), t["cost"].copy()

    quiet = None
    for mode in (2, 1):  # the copy-fed rings (unfused) and the rings the producer warps compute into (fused, round 2)
        s.traj_set_fused(mode)
        first = one_traj()
        if quiet is None:
            quiet = first
        for a, b in zip(quiet, first):
            assert np.array_equal(a, b), "fused and unfused trajectory-level step differ"
        for rep in range(25):
            heavy.reset()
            heavy.run(30 + rep)                  # asynchronous, on its own stream: varies what shares the SMs
            got = one_traj()
            for a, b in zip(quiet, got):
                assert np.array_equal(a, b), f"trajectory-level step differs in repetition {rep} (fused mode {mode})"
    s.close()
    for K, n in ((3, 40), (9, 40), (24, 60), (175, 80), (600, 180)):
        q = wl.search_candidates(ch, K, n, 730 + K, limit_frac=0.02)
        ss = lm.Solver(ch, K, n, np.zeros((K * n, 3), np.float32), np.tile(np.array([[1, 0, 0, 0]], np.float32), (K * n, 1)),
                       q.reshape(K * n, 7))
        ref = ss.search()
        for rep in range(12):
            heavy.reset()
            heavy.run(20 + 3 * rep)
            g = ss.search()
            assert np.array_equal(g["choice"], ref["choice"]) and g["cost"] == ref["cost"], (K, n, rep)
        ss.close()
    heavy.close()
