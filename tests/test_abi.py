"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol that
include/lm.h declares; host-only entry points behave as documented (CPU only, no compute calls)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2309_09102_b200 import build as lm_build
from paper_2309_09102_b200 import lm, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    lm_build.build()
    return lm.lib()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "lm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lm_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    names = declared_functions()
    assert set(names) == set(lm.SYMBOLS), (names, lm.SYMBOLS)
    for n in names:
        assert hasattr(L, n), n


def test_library_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", lm_build.LIB_PATH], stdout=subprocess.PIPE, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, out


def test_default_params_and_strerror(L):
    p = lm.lm_default_params()
    assert (p.lambda0, p.nu_up, p.nu_down) == (np.float32(1e-3), 10.0, 10.0)
    assert p.lambda_min == np.float32(1e-4) and p.lambda_max == np.float32(1e7)
    assert p.tol == 0.0 and p.w_pos == 1.0 and p.w_rot == 1.0 and p.refine_steps == 1 and p.fast_sincos == 0
    assert L.lm_default_params(None) == lm.LM_EINVAL
    assert lm.lm_strerror(0) == "ok" and "invalid" in lm.lm_strerror(lm.LM_EINVAL)
    assert "workspace" in lm.lm_strerror(lm.LM_ENOMEM) and lm.lm_strerror(-99).startswith("unknown")


def test_workspace_bytes(L):
    assert lm.lm_workspace_bytes(0, 1, 1) == 0 and lm.lm_workspace_bytes(9, 1, 1) == 0
    assert lm.lm_workspace_bytes(7, 0, 10) == 0
    a = lm.lm_workspace_bytes(7, 4096, 300)
    W = 4096 * 300
    assert a >= W * (4 * 7 + 4 * 5 + 8 + 8) and a % 256 == 0
    assert a < W * 80
    h = lm.lm_workspace_bytes(7, 4096, 300, 0, lm.LM_MEM_HOST)
    assert h >= a + W * 4 * (7 + 7)
    hs = lm.lm_workspace_bytes(7, 4096, 300, 1, lm.LM_MEM_HOST)
    assert hs < h


def test_init_validation_without_gpu(L):
    ch, keep = lm.make_chain(wl.panda_chain())
    prm = lm.lm_default_params()
    fake = 0x10000  # never dereferenced: every case below must fail validation first
    nbytes = lm.lm_workspace_bytes(7, 2, 5)

    def init(chain=ch, B=2, n=5, tp=fake, tq=fake, seeds=fake, mem=lm.LM_MEM_DEVICE, ws=fake, wsb=nbytes, params=prm):
        ctx = C.c_void_p()
        pb = lm.LmProblem(B, n, tp, tq, 0, seeds, mem, ws, wsb)
        return L.lm_init(C.byref(ctx), C.byref(chain), C.byref(pb), C.byref(params), None), ctx

    assert init(B=0)[0] == lm.LM_EINVAL
    assert init(tp=None)[0] == lm.LM_EINVAL
    assert init(seeds=fake + 4)[0] == lm.LM_EINVAL          # misaligned device pointer
    assert init(ws=fake + 16)[0] == lm.LM_EINVAL            # workspace not 256-byte aligned
    assert init(mem=7)[0] == lm.LM_EINVAL
    assert init(wsb=nbytes - 1)[0] == lm.LM_ENOMEM
    bad, keep2 = lm.make_chain(wl.panda_chain())
    bad.dof = 9
    assert init(chain=bad)[0] == lm.LM_EINVAL
    c2 = wl.panda_chain()
    c2.q_lo = c2.q_hi + 1.0
    bad2, keep3 = lm.make_chain(c2)
    assert init(chain=bad2)[0] == lm.LM_EINVAL
    assert init(params=lm.lm_default_params(refine_steps=3))[0] == lm.LM_EINVAL
    assert init(params=lm.lm_default_params(lambda0=0.0))[0] == lm.LM_EINVAL
    # null handles
    assert L.lm_specialize(None) == lm.LM_EINVAL
    assert L.lm_step(None) == lm.LM_EINVAL and L.lm_run(None, 5) == lm.LM_EINVAL
    assert L.lm_fetch(None, None, None) == lm.LM_EINVAL and L.lm_reset(None) == lm.LM_EINVAL
    # a well-formed device-memory problem binds without touching the device; max_iters is checked
    rc, ctx = init()
    assert rc == lm.LM_OK and ctx.value
    assert L.lm_run(ctx, 65) == lm.LM_EINVAL and L.lm_run(ctx, -1) == lm.LM_EINVAL
    assert L.lm_set_option(ctx, lm.LM_OPT_BLOCK_THREADS, 48) == lm.LM_EINVAL
    assert L.lm_set_option(ctx, lm.LM_OPT_BLOCK_THREADS, 64) == lm.LM_OK
    assert L.lm_set_option(ctx, 77, 1) == lm.LM_EINVAL
    # the Panda table's structure is registered: a specialised kernel is selected at lm_init
    assert L.lm_kernel_name(ctx) == b"panda7"
    assert L.lm_set_option(ctx, lm.LM_OPT_GENERIC_KERNEL, 1) == lm.LM_OK and L.lm_kernel_name(ctx) == b"generic"
    L.lm_free(ctx)


def test_pipe_handle_validation_without_a_device():
    """lm_pipe_* (include/lm.h): argument checks come before any CUDA call, null handles are harmless, and a handle is an
    independent object (two creations never share state: on a box without a GPU both fail in CUDA, not in the library)."""
    import ctypes as C
    L = lm.lib()
    assert L.lm_pipe_create(None, 4) == lm.LM_EINVAL
    h = C.c_void_p()
    assert L.lm_pipe_create(C.byref(h), 0) == lm.LM_EINVAL and not h.value
    assert L.lm_pipe_create(C.byref(h), 257) == lm.LM_EINVAL and not h.value
    L.lm_pipe_destroy(None)
    assert L.lm_pipe_solve(None, None, None, None, None, 1, 1, None, None) == lm.LM_EINVAL
    import torch
    handles = []
    for _ in range(2):  # one per "device slot" of a multi-GPU process: independent objects, no process-global state
        h = C.c_void_p()
        rc = L.lm_pipe_create(C.byref(h), 8)
        if torch.cuda.is_available():
            assert rc == lm.LM_OK and h.value
            handles.append(h)
        else:
            assert rc == lm.LM_ECUDA and not h.value
    assert len({x.value for x in handles}) == len(handles)
    for x in handles:
        # a handle rejects malformed problems before touching its streams
        assert L.lm_pipe_solve(x, None, None, None, None, 1, 1, None, None) == lm.LM_EINVAL
        L.lm_pipe_destroy(x)


def test_product_has_no_oracle_dependency():
    """The package never imports oracle/ (no CPU fallback): grep the sources."""
    pkg = os.path.join(ROOT, "paper_2309_09102_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "lm_oracle" not in txt and "import oracle" not in txt and "from oracle" not in txt, f


def test_solver_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    ch = wl.panda_chain()
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        lm.Solver(ch, 1, 1, np.zeros((1, 3)), np.array([[1, 0, 0, 0.0]]), np.zeros((1, 7)))
