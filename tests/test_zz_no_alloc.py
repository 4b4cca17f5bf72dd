"""lm_search_static (include/lm.h): the global discrete search for callers that cannot allocate device memory.

Who needs it: a re-planning loop that must answer inside a time budget (cudaMalloc / cudaFree take driver-wide locks,
may wait for the whole device and have no latency bound), and a process whose GPU memory belongs to somebody else's
pool (a simulator, a learning framework, a fixed start-up budget), where a fresh cudaMalloc fails or is not allowed.
For them the search keeps its intermediate arrays in a fixed 16 MiB array inside the library instead of a caller's
workspace.  The array is shared by every call and keeps the previous call's contents, so this test makes two calls
in a row of DIFFERENT shapes (the second smaller: it runs on top of the first one's leftovers), then the first shape
again, and compares each with the existing path, lm_search on a caller-allocated workspace.  The search is integer /
argmin work decided in fp32 by both paths with the same kernels, so the bar is the one tests/test_gpu_search.py uses:
bit for bit (choice, xi, cost, mjac).

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests), and
passes both alone in a fresh process -- where its first call is the one that looks up the array's device address --
and after the rest of the suite."""
import numpy as np
import pytest

from paper_2309_09102_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def existing_path(ch, q32):
    """lm_search through a context and a torch-allocated workspace: the path the other tests pin to the oracle."""
    from oracle import lm_oracle as orc
    from paper_2309_09102_b200 import lm
    K, n, d = q32.shape
    p, R = orc.fk(ch, q32[0].astype(np.float64))                   # targets are irrelevant to the search; any pose does
    tp = np.tile(p.astype(np.float32), (K, 1))
    tq = np.tile(wl._R_to_quat_wxyz(R).astype(np.float32), (K, 1))
    s = lm.Solver(ch, K, n, tp, tq, q32.reshape(K * n, d))
    g = s.search()
    s.close()
    return g


class StaticCall:
    """Inputs and outputs of one lm_search_static call, all allocated up front (the call itself allocates nothing)."""

    def __init__(self, ch, q32):
        import torch
        K, n, d = q32.shape
        self.ch, self.K, self.n, self.d = ch, K, n, d
        self.q = torch.from_numpy(np.ascontiguousarray(q32.reshape(K * n, d).T)).to("cuda:0")   # [d][K * n]
        self.choice = torch.full((n,), -1, dtype=torch.int32, device="cuda:0")
        self.xi = torch.full((d, n), float("nan"), dtype=torch.float32, device="cuda:0")
        self.res = torch.full((2,), float("nan"), dtype=torch.float32, device="cuda:0")

    def run(self):
        import torch
        from paper_2309_09102_b200 import lm
        self.choice.fill_(-1); self.xi.fill_(float("nan")); self.res.fill_(float("nan"))
        lm.lm_search_static(self.ch, self.K, self.n, self.q.data_ptr(), lm.lm_search_default_params(),
                            torch.cuda.current_stream().cuda_stream, self.choice.data_ptr(), self.xi.data_ptr(), self.res.data_ptr())
        r = self.res.cpu().numpy()
        return {"choice": self.choice.cpu().numpy(), "xi": np.ascontiguousarray(self.xi.cpu().numpy().T), "cost": float(r[0]), "mjac": float(r[1])}


def same_bits(a, b):
    assert np.array_equal(a["choice"], b["choice"])
    assert np.array_equal(a["xi"].view(np.uint32), b["xi"].view(np.uint32))
    assert np.float32(a["cost"]).view(np.uint32) == np.float32(b["cost"]).view(np.uint32)
    assert np.float32(a["mjac"]).view(np.uint32) == np.float32(b["mjac"]).view(np.uint32)


def test_static_search_equals_the_workspace_search_on_two_calls_in_a_row():
    import torch
    from paper_2309_09102_b200 import lm
    torch.cuda.set_device(0)
    panda, fetch_like = wl.panda_chain(), wl.random_chain_8dof(3)   # 7 revolute joints; 8 joints, one prismatic
    qa = wl.search_candidates(panda, 175, 120, 21, limit_frac=0.03)                  # the paper's K; 15.5 of the 16 MiB
    qb = wl.search_candidates(fetch_like, 33, 45, 22, limit_frac=0.3)                # smaller: sits inside qa's leftovers
    qb[:, 20, 1] = np.float32(fetch_like.q_hi[1]) - np.float32(0.001)                # a layer of unavoidable penalties
    assert lm.lm_search_static_fits(7, 175, 120) and lm.lm_search_static_fits(8, 33, 45)
    want_a, want_b = existing_path(panda, qa), existing_path(fetch_like, qb)
    assert len(set(want_a["choice"].tolist())) > 1 and want_b["cost"] >= 10.0        # neither problem is trivial
    a, b = StaticCall(panda, qa), StaticCall(fetch_like, qb)
    a.run()                                                         # start-up call: address look-up, kernel loading
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    got_a = a.run()                                                 # two calls in a row on the shared array ...
    got_b = b.run()
    got_a2 = a.run()                                                # ... and the first shape once more on top of them
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before              # the device's free memory did not shrink
    same_bits(got_a, want_a)
    same_bits(got_b, want_b)
    same_bits(got_a2, want_a)


def test_static_search_rejects_what_does_not_fit():
    import torch
    from paper_2309_09102_b200 import lm
    torch.cuda.set_device(0)
    ch = wl.panda_chain()
    assert not lm.lm_search_static_fits(7, 175, 300)                # the paper's K = 175 at n = 300 needs 40 MB: lm_search
    assert lm.lm_search_static_fits(7, 175, 124) and not lm.lm_search_static_fits(7, 175, 125)
    assert not lm.lm_search_static_fits(7, 1025, 2) and not lm.lm_search_static_fits(9, 4, 4)
    big = StaticCall(ch, np.zeros((175, 125, 7), np.float32))
    with pytest.raises(lm.LmError) as e:
        big.run()
    assert e.value.code == lm.LM_ECAPACITY and "fixed scratch" in str(e.value)
    assert (big.choice.cpu().numpy() == -1).all()                   # nothing was launched, nothing written
    ok = StaticCall(ch, wl.search_candidates(ch, 4, 6, 23))
    host_q = np.zeros((7, 24), np.float32)
    with pytest.raises(lm.LmError) as e:                            # q must be device memory
        lm.lm_search_static(ch, 4, 6, host_q.ctypes.data, lm.lm_search_default_params(), 0, None, None, None)
    assert e.value.code == lm.LM_EINVAL
    with pytest.raises(lm.LmError) as e:                            # the clearance penalty needs a context
        lm.lm_search_static(ch, 4, 6, ok.q.data_ptr(), lm.lm_search_default_params(use_clearance=1), 0, None, None, None)
    assert e.value.code == lm.LM_EINVAL
    same_bits(ok.run(), existing_path(ch, wl.search_candidates(ch, 4, 6, 23)))       # and the array still works afterwards
