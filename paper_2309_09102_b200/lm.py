"""Thin ctypes binding of include/lm.h (liblm_b200.so): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device
memory (``torch.empty(..., device="cuda")``) and the stream handle, nothing else.  There is no
CPU fallback: if the library has not been built (``python -m paper_2309_09102_b200.build``) or
no CUDA device is present, the calls raise.

The functions ``lm_*`` mirror the C entry points one to one; ``Solver`` bundles the buffers of
one problem (it owns the torch tensors the library borrows).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from .build import LIB_PATH

LM_MAX_DOF = 8
LM_MAX_ITERS = 64
LM_OK, LM_EINVAL, LM_ENOMEM, LM_ECUDA, LM_ECAPACITY = 0, -1, -2, -3, -4
LM_SEARCH_STATIC_BYTES = 16 << 20
LM_MEM_DEVICE, LM_MEM_HOST = 0, 1
LM_OPT_BLOCK_THREADS, LM_OPT_GENERIC_KERNEL, LM_OPT_LANES_PER_WAYPOINT, LM_OPT_TRAJ_FUSED, LM_OPT_TRAJ_COST_LANES = 1, 2, 3, 4, 5
LM_ST_FROZEN, LM_ST_MAXITER, LM_ST_BREAKDOWN, LM_ST_NONFINITE, LM_ST_CLAMPED = 1, 2, 4, 8, 16

# every symbol include/lm.h declares (checked by tests/test_abi.py)
SYMBOLS = ("lm_workspace_bytes", "lm_default_params", "lm_init", "lm_step", "lm_run", "lm_fetch",
           "lm_reset", "lm_set_state", "lm_set_trace", "lm_set_option", "lm_kernel_name", "lm_fk", "lm_fp32_peak", "lm_free",
           "lm_strerror", "lm_launch_count",
           "lm_traj_workspace_bytes", "lm_traj_default_params", "lm_traj_attach", "lm_traj_run", "lm_traj_reset",
           "lm_traj_fetch", "lm_traj_set_trace", "lm_traj_set_capsules", "lm_traj_set_obstacles",
           "lm_solve_host_workspace_bytes", "lm_solve_host", "lm_pipe_create", "lm_pipe_solve", "lm_pipe_destroy", "lm_specialize",
           "lm_plan_workspace_bytes", "lm_plan_default_params", "lm_plan_attach", "lm_plan_run", "lm_plan_fetch",
           "lm_search_workspace_bytes", "lm_search_default_params", "lm_search",
           "lm_search_static_fits", "lm_search_static")
LM_SOLVER_PRIMAL, LM_SOLVER_DUAL = 0, 1
LM_ROT_LOG, LM_ROT_RPY = 0, 1


class LmChain(C.Structure):
    _fields_ = [("dof", C.c_int32), ("joint_type", C.POINTER(C.c_uint8)), ("dh", C.POINTER(C.c_double)),
                ("q_lo", C.POINTER(C.c_double)), ("q_hi", C.POINTER(C.c_double)), ("tool", C.c_double * 7)]


class LmProblem(C.Structure):
    _fields_ = [("B", C.c_int64), ("n", C.c_int64), ("target_pos", C.c_void_p), ("target_quat", C.c_void_p),
                ("shared_targets", C.c_int32), ("seeds", C.c_void_p), ("memory", C.c_int32),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class LmParams(C.Structure):
    _fields_ = [("lambda0", C.c_float), ("nu_up", C.c_float), ("nu_down", C.c_float),
                ("lambda_min", C.c_float), ("lambda_max", C.c_float), ("tol", C.c_float),
                ("w_pos", C.c_float), ("w_rot", C.c_float), ("refine_steps", C.c_int32),
                ("fast_sincos", C.c_int32), ("solver", C.c_int32), ("rot_residual", C.c_int32)]


class LmStats(C.Structure):
    _fields_ = [("res_norm", C.c_void_p), ("pos_err", C.c_void_p), ("rot_err", C.c_void_p),
                ("lambda_", C.c_void_p), ("iters", C.c_void_p), ("accept_mask", C.c_void_p),
                ("status", C.c_void_p), ("traj_converged", C.c_void_p), ("traj_iters", C.c_void_p),
                ("total_waypoint_iters", C.c_int64), ("converged_trajectories", C.c_int64)]


class LmTrajParams(C.Structure):
    _fields_ = [("w_pose", C.c_float), ("w_diff", C.c_float), ("lambda0", C.c_float), ("nu_up", C.c_float),
                ("nu_down", C.c_float), ("lambda_min", C.c_float), ("lambda_max", C.c_float),
                ("refine_steps", C.c_int32)]


class LmTrajStats(C.Structure):
    _fields_ = [("cost", C.c_void_p), ("cost_pose", C.c_void_p), ("cost_diff", C.c_void_p), ("cost_coll", C.c_void_p),
                ("lambda_", C.c_void_p), ("iters", C.c_void_p), ("accept_mask", C.c_void_p),
                ("status", C.c_void_p), ("total_traj_iters", C.c_int64)]


class LmCapsules(C.Structure):
    _fields_ = [("ncaps", C.c_int32), ("link", C.POINTER(C.c_int32)), ("a", C.POINTER(C.c_float)), ("b", C.POINTER(C.c_float)),
                ("radius", C.POINTER(C.c_float)), ("npairs", C.c_int32), ("pairs", C.POINTER(C.c_int32)),
                ("w_coll", C.c_float), ("d_safe", C.c_float)]


class LmObstacles(C.Structure):
    _fields_ = [("nobs", C.c_int32), ("pose", C.POINTER(C.c_float)), ("pmin", C.POINTER(C.c_float)),
                ("pmax", C.POINTER(C.c_float)), ("npairs", C.c_int32), ("pairs", C.POINTER(C.c_int32)),
                ("w_env", C.c_float), ("d_safe", C.c_float)]


class LmPlanParams(C.Structure):
    _fields_ = [("pos_tol", C.c_float), ("rot_tol", C.c_float), ("mjac_rev", C.c_float), ("mjac_pris", C.c_float),
                ("pose_iters", C.c_int32), ("min_clearance", C.c_float)]


class LmPlanStats(C.Structure):
    _fields_ = [("valid", C.c_void_p), ("first_valid_cycle", C.c_void_p), ("records", C.c_void_p),
                ("length", C.c_void_p), ("max_pos_err", C.c_void_p), ("max_rot_err", C.c_void_p),
                ("mjac_rev", C.c_void_p), ("mjac_pris", C.c_void_p), ("cur_length", C.c_void_p),
                ("min_clearance", C.c_void_p), ("valid_trajectories", C.c_int64)]


class LmSearchParams(C.Structure):
    _fields_ = [("margin_rev", C.c_float), ("margin_pris", C.c_float), ("pen_limit", C.c_float),
                ("pen_collision", C.c_float), ("use_clearance", C.c_int32)]


class LmError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {lm_strerror(code)} ({code})")


_lib = None


def lib() -> C.CDLL:
    """Load liblm_b200.so; fails loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2309_09102_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.lm_workspace_bytes.argtypes = [C.c_int32, C.c_int64, C.c_int64, C.c_int32, C.c_int32]
        L.lm_workspace_bytes.restype = C.c_size_t
        L.lm_default_params.argtypes = [C.POINTER(LmParams)]
        L.lm_init.argtypes = [C.POINTER(C.c_void_p), C.POINTER(LmChain), C.POINTER(LmProblem),
                              C.POINTER(LmParams), C.c_void_p]
        L.lm_step.argtypes = [C.c_void_p]
        L.lm_run.argtypes = [C.c_void_p, C.c_int32]
        L.lm_fetch.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(LmStats)]
        L.lm_reset.argtypes = [C.c_void_p]
        L.lm_set_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.lm_set_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.lm_set_option.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        L.lm_specialize.argtypes = [C.c_void_p]
        L.lm_kernel_name.argtypes = [C.c_void_p]
        L.lm_kernel_name.restype = C.c_char_p
        L.lm_fk.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.lm_fp32_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.lm_free.argtypes = [C.c_void_p]
        L.lm_free.restype = None
        L.lm_strerror.argtypes = [C.c_int]
        L.lm_strerror.restype = C.c_char_p
        L.lm_launch_count.restype = C.c_int64
        L.lm_traj_workspace_bytes.argtypes = [C.c_int32, C.c_int64, C.c_int64]
        L.lm_traj_workspace_bytes.restype = C.c_size_t
        L.lm_traj_default_params.argtypes = [C.POINTER(LmTrajParams)]
        L.lm_traj_attach.argtypes = [C.c_void_p, C.POINTER(LmTrajParams), C.c_void_p, C.c_size_t]
        L.lm_traj_run.argtypes = [C.c_void_p, C.c_int32]
        L.lm_traj_reset.argtypes = [C.c_void_p, C.c_void_p]
        L.lm_traj_fetch.argtypes = [C.c_void_p, C.POINTER(LmTrajStats)]
        L.lm_traj_set_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.lm_traj_set_capsules.argtypes = [C.c_void_p, C.POINTER(LmCapsules)]
        L.lm_traj_set_obstacles.argtypes = [C.c_void_p, C.POINTER(LmObstacles)]
        L.lm_solve_host_workspace_bytes.argtypes = [C.c_int32, C.c_int64, C.c_int64, C.c_int32]
        L.lm_solve_host_workspace_bytes.restype = C.c_size_t
        L.lm_solve_host.argtypes = [C.POINTER(LmChain), C.POINTER(LmProblem), C.POINTER(LmParams), C.c_int32, C.c_int32,
                                    C.c_void_p, C.POINTER(LmStats)]
        L.lm_pipe_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32]
        L.lm_pipe_solve.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(LmChain), C.POINTER(LmProblem), C.POINTER(LmParams), C.c_int32,
                                    C.c_int32, C.c_void_p, C.POINTER(LmStats)]
        L.lm_pipe_destroy.argtypes = [C.c_void_p]
        L.lm_pipe_destroy.restype = None
        L.lm_plan_workspace_bytes.argtypes = [C.c_int32, C.c_int64, C.c_int64]
        L.lm_plan_workspace_bytes.restype = C.c_size_t
        L.lm_plan_default_params.argtypes = [C.POINTER(LmPlanParams)]
        L.lm_plan_attach.argtypes = [C.c_void_p, C.POINTER(LmPlanParams), C.c_void_p, C.c_size_t]
        L.lm_plan_run.argtypes = [C.c_void_p, C.c_int32]
        L.lm_plan_fetch.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(LmPlanStats)]
        L.lm_search_workspace_bytes.argtypes = [C.c_int32, C.c_int64, C.c_int64]
        L.lm_search_workspace_bytes.restype = C.c_size_t
        L.lm_search_default_params.argtypes = [C.POINTER(LmSearchParams)]
        L.lm_search.argtypes = [C.c_void_p, C.POINTER(LmSearchParams), C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p, C.c_void_p]
        L.lm_search_static_fits.argtypes = [C.c_int32, C.c_int64, C.c_int64]
        L.lm_search_static.argtypes = [C.POINTER(LmChain), C.c_int64, C.c_int64, C.c_void_p, C.POINTER(LmSearchParams), C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _check(rc: int, where: str) -> None:
    if rc != LM_OK:
        raise LmError(rc, where)


# ------------------------------------------------------------------ 1:1 wrappers

def lm_strerror(code: int) -> str:
    return lib().lm_strerror(int(code)).decode()


def lm_launch_count() -> int:
    return int(lib().lm_launch_count())


def lm_workspace_bytes(dof: int, B: int, n: int, shared_targets: int = 0, memory: int = LM_MEM_DEVICE) -> int:
    return int(lib().lm_workspace_bytes(dof, B, n, shared_targets, memory))


def lm_default_params(**overrides) -> LmParams:
    p = LmParams()
    _check(lib().lm_default_params(C.byref(p)), "lm_default_params")
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


def make_chain(chain) -> tuple:
    """Marshal a workloads.Chain-like object into an LmChain (returns the struct and the arrays it
    points to, which must outlive the lm_init call)."""
    d = int(chain.dof)
    jt = np.ascontiguousarray(np.asarray(chain.joint_type), dtype=np.uint8)
    dh = np.ascontiguousarray(np.stack([chain.a, chain.alpha, chain.d, chain.theta], axis=1), dtype=np.float64)
    lo = np.ascontiguousarray(chain.q_lo, dtype=np.float64)
    hi = np.ascontiguousarray(chain.q_hi, dtype=np.float64)
    c = LmChain()
    c.dof = d
    c.joint_type = jt.ctypes.data_as(C.POINTER(C.c_uint8))
    c.dh = dh.ctypes.data_as(C.POINTER(C.c_double))
    c.q_lo = lo.ctypes.data_as(C.POINTER(C.c_double))
    c.q_hi = hi.ctypes.data_as(C.POINTER(C.c_double))
    for i, v in enumerate(np.asarray(chain.tool, dtype=np.float64)):
        c.tool[i] = float(v)
    return c, (jt, dh, lo, hi)


def lm_init(chain: LmChain, problem: LmProblem, params: LmParams, cuda_stream: int = 0) -> int:
    ctx = C.c_void_p()
    _check(lib().lm_init(C.byref(ctx), C.byref(chain), C.byref(problem), C.byref(params),
                         C.c_void_p(cuda_stream)), "lm_init")
    return ctx.value


def lm_step(ctx: int) -> None:
    _check(lib().lm_step(ctx), "lm_step")


def lm_run(ctx: int, max_iters: int) -> None:
    _check(lib().lm_run(ctx, int(max_iters)), "lm_run")


def lm_reset(ctx: int) -> None:
    _check(lib().lm_reset(ctx), "lm_reset")


def lm_fetch(ctx: int, q_out_ptr: Optional[int], stats: Optional[LmStats]) -> None:
    _check(lib().lm_fetch(ctx, q_out_ptr, C.byref(stats) if stats is not None else None), "lm_fetch")


def lm_set_state(ctx: int, q_ptr: int, lambda_ptr: Optional[int]) -> None:
    _check(lib().lm_set_state(ctx, q_ptr, lambda_ptr), "lm_set_state")


def lm_set_trace(ctx: int, trial_q_ptr: Optional[int], trial_F_ptr: Optional[int]) -> None:
    _check(lib().lm_set_trace(ctx, trial_q_ptr, trial_F_ptr), "lm_set_trace")


def lm_set_option(ctx: int, option: int, value: int) -> None:
    _check(lib().lm_set_option(ctx, int(option), int(value)), "lm_set_option")


def lm_kernel_name(ctx: int) -> str:
    return lib().lm_kernel_name(ctx).decode()


def lm_fk(ctx: int, q_ptr: int, count: int, pos_ptr: int, rot_ptr: int) -> None:
    _check(lib().lm_fk(ctx, q_ptr, int(count), pos_ptr, rot_ptr), "lm_fk")


def lm_fp32_peak(cuda_stream: int = 0) -> float:
    out = C.c_double(0.0)
    _check(lib().lm_fp32_peak(C.c_void_p(cuda_stream), C.byref(out)), "lm_fp32_peak")
    return float(out.value)


def lm_traj_workspace_bytes(dof: int, B: int, n: int) -> int:
    return int(lib().lm_traj_workspace_bytes(dof, B, n))


def lm_traj_default_params(**overrides) -> LmTrajParams:
    p = LmTrajParams()
    _check(lib().lm_traj_default_params(C.byref(p)), "lm_traj_default_params")
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


def lm_traj_attach(ctx: int, params: LmTrajParams, workspace_ptr: int, workspace_bytes: int) -> None:
    _check(lib().lm_traj_attach(ctx, C.byref(params), workspace_ptr, workspace_bytes), "lm_traj_attach")


def lm_traj_run(ctx: int, iters: int) -> None:
    _check(lib().lm_traj_run(ctx, int(iters)), "lm_traj_run")


def lm_traj_reset(ctx: int, lambda_ptr: Optional[int]) -> None:
    _check(lib().lm_traj_reset(ctx, lambda_ptr), "lm_traj_reset")


def lm_traj_fetch(ctx: int, stats: LmTrajStats) -> None:
    _check(lib().lm_traj_fetch(ctx, C.byref(stats)), "lm_traj_fetch")


def lm_traj_set_capsules(ctx: int, model, w_coll: float = 1.0, d_safe: float = 0.05) -> None:
    """model: a workloads.CapsuleModel-like object (link, a, b, radius, pairs) or None to remove the rows."""
    if model is None:
        _check(lib().lm_traj_set_capsules(ctx, None), "lm_traj_set_capsules")
        return
    link = np.ascontiguousarray(model.link, dtype=np.int32)
    a = np.ascontiguousarray(model.a, dtype=np.float32)
    b = np.ascontiguousarray(model.b, dtype=np.float32)
    rad = np.ascontiguousarray(model.radius, dtype=np.float32)
    pairs = np.ascontiguousarray(model.pairs, dtype=np.int32)
    m = LmCapsules(len(link), link.ctypes.data_as(C.POINTER(C.c_int32)), a.ctypes.data_as(C.POINTER(C.c_float)),
                   b.ctypes.data_as(C.POINTER(C.c_float)), rad.ctypes.data_as(C.POINTER(C.c_float)), len(pairs),
                   pairs.ctypes.data_as(C.POINTER(C.c_int32)), float(w_coll), float(d_safe))
    _check(lib().lm_traj_set_capsules(ctx, C.byref(m)), "lm_traj_set_capsules")


def lm_traj_set_obstacles(ctx: int, scene, w_env: float = 1.0, d_safe: float = 0.05) -> None:
    """scene: a workloads.ObstacleScene-like object (pose [M, 7] = xyz + unit quaternion w, x, y, z of each box frame, as
    lm_obstacles takes it; pmin, pmax [M, 3]; pairs [Q, 2]) or None to remove the rows."""
    if scene is None:
        _check(lib().lm_traj_set_obstacles(ctx, None), "lm_traj_set_obstacles")
        return
    pose = np.ascontiguousarray(scene.pose, dtype=np.float32)
    pmin = np.ascontiguousarray(scene.pmin, dtype=np.float32)
    pmax = np.ascontiguousarray(scene.pmax, dtype=np.float32)
    pairs = np.ascontiguousarray(scene.pairs, dtype=np.int32)
    fp = C.POINTER(C.c_float)
    o = LmObstacles(len(pose), pose.ctypes.data_as(fp), pmin.ctypes.data_as(fp), pmax.ctypes.data_as(fp), len(pairs),
                    pairs.ctypes.data_as(C.POINTER(C.c_int32)), float(w_env), float(d_safe))
    _check(lib().lm_traj_set_obstacles(ctx, C.byref(o)), "lm_traj_set_obstacles")


def lm_traj_set_trace(ctx: int, trial_q_ptr: Optional[int], trial_F_ptr: Optional[int]) -> None:
    _check(lib().lm_traj_set_trace(ctx, trial_q_ptr, trial_F_ptr), "lm_traj_set_trace")


def lm_solve_host_workspace_bytes(dof: int, B: int, n: int, chunks: int) -> int:
    return int(lib().lm_solve_host_workspace_bytes(dof, B, n, chunks))


def lm_solve_host(chain: LmChain, problem: LmProblem, params: LmParams, max_iters: int, chunks: int,
                  q_out_ptr: Optional[int], stats: Optional[LmStats]) -> None:
    _check(lib().lm_solve_host(C.byref(chain), C.byref(problem), C.byref(params), int(max_iters), int(chunks),
                               q_out_ptr, C.byref(stats) if stats is not None else None), "lm_solve_host")


def lm_pipe_create(max_chunks: int) -> C.c_void_p:
    """Streams / events / pinned totals of the host-data pipeline on the CURRENT device (include/lm.h)."""
    out = C.c_void_p()
    _check(lib().lm_pipe_create(C.byref(out), int(max_chunks)), "lm_pipe_create")
    return out


def lm_pipe_solve(pipe, chain: LmChain, problem: LmProblem, params: LmParams, max_iters: int, chunks: int,
                  q_out_ptr: Optional[int], stats: Optional[LmStats], cuda_stream: int = 0) -> None:
    _check(lib().lm_pipe_solve(pipe, C.c_void_p(cuda_stream), C.byref(chain), C.byref(problem), C.byref(params), int(max_iters),
                               int(chunks), q_out_ptr, C.byref(stats) if stats is not None else None), "lm_pipe_solve")


def lm_pipe_destroy(pipe) -> None:
    lib().lm_pipe_destroy(pipe)


def lm_plan_workspace_bytes(dof: int, B: int, n: int) -> int:
    return int(lib().lm_plan_workspace_bytes(dof, B, n))


def lm_plan_default_params(**overrides) -> LmPlanParams:
    p = LmPlanParams()
    _check(lib().lm_plan_default_params(C.byref(p)), "lm_plan_default_params")
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


def lm_plan_attach(ctx: int, params: LmPlanParams, workspace_ptr: int, workspace_bytes: int) -> None:
    _check(lib().lm_plan_attach(ctx, C.byref(params), workspace_ptr, workspace_bytes), "lm_plan_attach")


def lm_plan_run(ctx: int, cycles: int) -> None:
    _check(lib().lm_plan_run(ctx, int(cycles)), "lm_plan_run")


def lm_plan_fetch(ctx: int, q_valid_ptr: Optional[int], stats: Optional[LmPlanStats]) -> None:
    _check(lib().lm_plan_fetch(ctx, q_valid_ptr, C.byref(stats) if stats is not None else None), "lm_plan_fetch")


def lm_search_workspace_bytes(dof: int, K: int, n: int) -> int:
    return int(lib().lm_search_workspace_bytes(dof, K, n))


def lm_search_default_params(**overrides) -> LmSearchParams:
    p = LmSearchParams()
    _check(lib().lm_search_default_params(C.byref(p)), "lm_search_default_params")
    for k, v in overrides.items():
        if not hasattr(p, k):
            raise AttributeError(k)
        setattr(p, k, v)
    return p


def lm_search(ctx: int, params: LmSearchParams, workspace_ptr: int, workspace_bytes: int, choice_ptr: Optional[int],
              xi_ptr: Optional[int], result_ptr: Optional[int]) -> None:
    _check(lib().lm_search(ctx, C.byref(params), workspace_ptr, workspace_bytes, choice_ptr, xi_ptr, result_ptr), "lm_search")


def lm_search_static_fits(dof: int, K: int, n: int) -> bool:
    return bool(lib().lm_search_static_fits(dof, K, n))


def lm_search_static(chain, K: int, n: int, q_ptr: int, params: LmSearchParams, cuda_stream: int, choice_ptr: Optional[int],
                     xi_ptr: Optional[int], result_ptr: Optional[int]) -> None:
    """include/lm.h, lm_search_static: the search for callers that cannot allocate device memory (a re-planning loop
    with a deadline, a process whose GPU memory belongs to somebody else's pool).  Its scratch is a fixed 16 MiB array
    inside the library, shared by all calls; nothing is allocated here either: `chain` is marshalled on the host,
    q_ptr is the caller's device array [d][K * n], the three outputs are the caller's (device or host) buffers."""
    cstruct, keep = make_chain(chain)
    rc = lib().lm_search_static(C.byref(cstruct), K, n, q_ptr, C.byref(params), C.c_void_p(cuda_stream), choice_ptr, xi_ptr, result_ptr)
    del keep
    _check(rc, "lm_search_static")


def lm_free(ctx: int) -> None:
    lib().lm_free(ctx)


# ------------------------------------------------------------------ buffer bundle

class Solver:
    """Owns the torch device tensors of one problem and the lm_ctx that borrows them.

    ``target_pos [W,3]``, ``target_quat [W,4]`` (``[n,.]`` when shared), ``seeds [W,d]`` are
    waypoint-major numpy arrays (as produced by ``workloads``); they are transposed to the
    library's SoA layout here.  ``host_inputs=True`` hands the library pinned HOST arrays instead
    (LM_MEM_HOST: the host->device copies happen inside lm_init).
    """

    def __init__(self, chain, B: int, n: int, target_pos, target_quat, seeds, params: Optional[LmParams] = None,
                 shared_targets: bool = False, host_inputs: bool = False, device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the batched-LM path has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.chain, self.B, self.n, self.W, self.d = chain, int(B), int(n), int(B) * int(n), int(chain.dof)
        self.params = params if params is not None else lm_default_params()
        self.shared = bool(shared_targets)
        self.host_inputs = bool(host_inputs)
        self.stream = stream
        self._ctx = None
        Wt = self.n if self.shared else self.W
        assert np.shape(target_pos) == (Wt, 3) and np.shape(target_quat) == (Wt, 4) and np.shape(seeds) == (self.W, self.d)

        def soa(x):
            t = torch.from_numpy(np.ascontiguousarray(np.asarray(x, dtype=np.float32).T))
            return t.pin_memory() if self.host_inputs else t.to(self.device)

        with torch.cuda.device(self.device), self._on_stream():
            self.tp, self.tq, self.seeds = soa(target_pos), soa(target_quat), soa(seeds)
            mem = LM_MEM_HOST if self.host_inputs else LM_MEM_DEVICE
            nbytes = lm_workspace_bytes(self.d, self.B, self.n, int(self.shared), mem)
            self.workspace, ws_ptr = self._alloc_ws(nbytes)
            self._cchain, self._keep = make_chain(chain)
            pb = LmProblem(self.B, self.n, self.tp.data_ptr(), self.tq.data_ptr(), int(self.shared),
                           self.seeds.data_ptr(), mem, ws_ptr, nbytes)
            s = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._stream_handle = int(s.cuda_stream)
            self._ctx = lm_init(self._cchain, pb, self.params, self._stream_handle)

    def _alloc_ws(self, nbytes: int):
        """Device scratch of `nbytes`: (the tensor that owns it, a 256-byte aligned pointer into it)."""
        t = self.torch.empty(nbytes + 256, dtype=self.torch.uint8, device=self.device)
        return t, (t.data_ptr() + 255) // 256 * 256

    def _on_stream(self):
        """Uploads and allocations happen on the stream the library launches on: with a caller-supplied
        (possibly non-blocking) stream nothing else orders an H2D upload before the library's use of it, or the
        caching allocator's reuse of a freed block after it."""
        import contextlib
        if self.stream is None:
            return contextlib.nullcontext()
        return self.torch.cuda.stream(self.stream)

    # -- the hot path
    def step(self) -> None:
        lm_step(self._ctx)

    def run(self, max_iters: int) -> None:
        lm_run(self._ctx, max_iters)

    def reset(self) -> None:
        lm_reset(self._ctx)

    def set_launch(self, block_threads: int) -> None:
        lm_set_option(self._ctx, LM_OPT_BLOCK_THREADS, block_threads)

    def use_generic_kernel(self, on: bool = True) -> None:
        lm_set_option(self._ctx, LM_OPT_GENERIC_KERNEL, int(on))

    def specialize(self) -> None:
        """lm_specialize: compile (NVRTC, once per chain structure) and use a kernel specialised to this chain."""
        _check(lib().lm_specialize(self._ctx), "lm_specialize")

    def set_lanes_per_waypoint(self, lanes: int) -> None:
        """1 (default), 2 or 4 lanes per waypoint block (the measured lane-group alternative, include/lm.h)."""
        lm_set_option(self._ctx, LM_OPT_LANES_PER_WAYPOINT, int(lanes))

    @property
    def kernel_name(self) -> str:
        return lm_kernel_name(self._ctx)

    def set_state(self, q, lam=None) -> None:
        """q [W,d], lam [W] numpy (waypoint-major)."""
        torch = self.torch
        with self._on_stream():
            self._q_in = torch.from_numpy(np.ascontiguousarray(np.asarray(q, dtype=np.float32).T)).to(self.device)
            self._lam_in = None if lam is None else torch.from_numpy(np.ascontiguousarray(lam, dtype=np.float32)).to(self.device)
        lm_set_state(self._ctx, self._q_in.data_ptr(), None if lam is None else self._lam_in.data_ptr())

    def enable_trace(self) -> None:
        torch = self.torch
        with self._on_stream():
            self.trace_q = torch.full((self.d, self.W), float("nan"), dtype=torch.float32, device=self.device)
            self.trace_F = torch.full((2, self.W), float("nan"), dtype=torch.float32, device=self.device)
        lm_set_trace(self._ctx, self.trace_q.data_ptr(), self.trace_F.data_ptr())

    def fetch(self, host: bool = True) -> dict:
        """lm_fetch into fresh buffers; returns numpy arrays (host=True: the library writes pinned
        host memory directly; host=False: device tensors copied back by torch afterwards)."""
        torch = self.torch
        W, B, d = self.W, self.B, self.d

        def buf(shape, dtype):
            if host:
                return torch.empty(shape, dtype=dtype).pin_memory()
            with self._on_stream():
                return torch.empty(shape, dtype=dtype, device=self.device)

        out = {"q": buf((d, W), torch.float32), "res_norm": buf((W,), torch.float32),
               "pos_err": buf((W,), torch.float32), "rot_err": buf((W,), torch.float32),
               "lam": buf((W,), torch.float32), "iters": buf((W,), torch.int32),
               "mask": buf((W,), torch.int64), "status": buf((W,), torch.int32),
               "traj_converged": buf((B,), torch.uint8), "traj_iters": buf((B,), torch.int32)}
        st = LmStats(out["res_norm"].data_ptr(), out["pos_err"].data_ptr(), out["rot_err"].data_ptr(),
                     out["lam"].data_ptr(), out["iters"].data_ptr(), out["mask"].data_ptr(),
                     out["status"].data_ptr(), out["traj_converged"].data_ptr(), out["traj_iters"].data_ptr(), 0, 0)
        lm_fetch(self._ctx, out["q"].data_ptr(), st)      # synchronises the library's stream
        res = {k: v.cpu().numpy() for k, v in out.items()}
        res["q"] = np.ascontiguousarray(res["q"].T)
        res["mask"] = res["mask"].view(np.uint64)
        res["status"] = res["status"].view(np.uint32)
        res["total_waypoint_iters"] = int(st.total_waypoint_iters)
        res["converged_trajectories"] = int(st.converged_trajectories)
        if getattr(self, "trace_q", None) is not None:
            res["trial_q"] = np.ascontiguousarray(self.trace_q.cpu().numpy().T)
            tf = self.trace_F.cpu().numpy()
            res["F_before"], res["F_trial"] = tf[0], tf[1]
        return res

    # -- trajectory-level step (include/lm.h, lm_traj_*)
    def traj_attach(self, tparams: Optional[LmTrajParams] = None) -> None:
        torch = self.torch
        self.tparams = tparams if tparams is not None else lm_traj_default_params()
        nbytes = lm_traj_workspace_bytes(self.d, self.B, self.n)
        with self._on_stream():
            self.traj_workspace, ptr = self._alloc_ws(nbytes)
        lm_traj_attach(self._ctx, self.tparams, ptr, nbytes)

    def traj_set_fused(self, mode: int) -> None:
        """LM_OPT_TRAJ_FUSED: 0 = chosen by tile count, 1 = fused solve kernels, 2 = per-waypoint kernels through HBM."""
        lm_set_option(self._ctx, LM_OPT_TRAJ_FUSED, int(mode))

    def traj_set_cost_lanes(self, mode: int) -> None:
        """LM_OPT_TRAJ_COST_LANES: 0 = by shared_targets, 1 = a warp takes one waypoint of 32 trajectories, 2 = 32 waypoints of one."""
        lm_set_option(self._ctx, LM_OPT_TRAJ_COST_LANES, int(mode))

    def traj_set_capsules(self, model, w_coll: float = 1.0, d_safe: float = 0.05) -> None:
        lm_traj_set_capsules(self._ctx, model, w_coll, d_safe)

    def traj_set_obstacles(self, scene, w_env: float = 1.0, d_safe: float = 0.05) -> None:
        lm_traj_set_obstacles(self._ctx, scene, w_env, d_safe)

    def traj_run(self, iters: int) -> None:
        lm_traj_run(self._ctx, iters)

    def traj_reset(self, lam=None) -> None:
        """lam [B] numpy or None (= lambda0)."""
        if lam is None:
            lm_traj_reset(self._ctx, None)
        else:
            with self._on_stream():
                self._tlam_in = self.torch.from_numpy(np.ascontiguousarray(lam, dtype=np.float32)).to(self.device)
            lm_traj_reset(self._ctx, self._tlam_in.data_ptr())

    def traj_enable_trace(self) -> None:
        torch = self.torch
        with self._on_stream():
            self.ttrace_q = torch.full((self.d, self.W), float("nan"), dtype=torch.float32, device=self.device)
            self.ttrace_F = torch.full((2, self.B), float("nan"), dtype=torch.float32, device=self.device)
        lm_traj_set_trace(self._ctx, self.ttrace_q.data_ptr(), self.ttrace_F.data_ptr())

    def traj_fetch(self) -> dict:
        """lm_traj_fetch into pinned host buffers -> numpy; q comes from fetch()."""
        torch = self.torch
        B = self.B

        def buf(dtype):
            return torch.empty((B,), dtype=dtype).pin_memory()

        out = {"cost": buf(torch.float32), "cost_pose": buf(torch.float32), "cost_diff": buf(torch.float32),
               "cost_coll": buf(torch.float32), "lam": buf(torch.float32), "iters": buf(torch.int32), "mask": buf(torch.int64),
               "status": buf(torch.int32)}
        st = LmTrajStats(out["cost"].data_ptr(), out["cost_pose"].data_ptr(), out["cost_diff"].data_ptr(),
                         out["cost_coll"].data_ptr(), out["lam"].data_ptr(), out["iters"].data_ptr(), out["mask"].data_ptr(),
                         out["status"].data_ptr(), 0)
        lm_traj_fetch(self._ctx, st)
        res = {k: v.numpy().copy() for k, v in out.items()}
        res["mask"] = res["mask"].view(np.uint64)
        res["status"] = res["status"].view(np.uint32)
        res["total_traj_iters"] = int(st.total_traj_iters)
        if getattr(self, "ttrace_q", None) is not None:
            res["trial_q"] = np.ascontiguousarray(self.ttrace_q.cpu().numpy().T)
            tf = self.ttrace_F.cpu().numpy()
            res["F_before"], res["F_trial"] = tf[0], tf[1]
        return res

    # -- non-stationary schedule with anytime bookkeeping (include/lm.h, lm_plan_*)
    def plan_attach(self, pparams: Optional[LmPlanParams] = None) -> None:
        torch = self.torch
        self.pparams = pparams if pparams is not None else lm_plan_default_params()
        nbytes = lm_plan_workspace_bytes(self.d, self.B, self.n)
        with self._on_stream():
            self.plan_workspace, ptr = self._alloc_ws(nbytes)
        lm_plan_attach(self._ctx, self.pparams, ptr, nbytes)

    def plan_run(self, cycles: int) -> None:
        lm_plan_run(self._ctx, cycles)

    def plan_fetch(self) -> dict:
        torch = self.torch
        B = self.B

        def buf(dtype):
            return torch.empty((B,), dtype=dtype).pin_memory()

        qv = torch.empty((self.d, self.W), dtype=torch.float32).pin_memory()
        out = {"valid": buf(torch.uint8), "first_valid_cycle": buf(torch.int32), "records": buf(torch.int32),
               "length": buf(torch.float32), "max_pos_err": buf(torch.float32), "max_rot_err": buf(torch.float32),
               "mjac_rev": buf(torch.float32), "mjac_pris": buf(torch.float32), "cur_length": buf(torch.float32),
               "min_clearance": buf(torch.float32)}
        st = LmPlanStats(*[out[k].data_ptr() for k in ("valid", "first_valid_cycle", "records", "length", "max_pos_err",
                                                       "max_rot_err", "mjac_rev", "mjac_pris", "cur_length", "min_clearance")], 0)
        lm_plan_fetch(self._ctx, qv.data_ptr(), st)
        res = {k: v.numpy().copy() for k, v in out.items()}
        res["valid"] = res["valid"].astype(bool)
        res["q_valid"] = np.ascontiguousarray(qv.numpy().T)
        res["valid_trajectories"] = int(st.valid_trajectories)
        return res

    # -- global discrete search over the B = K candidates of one path (include/lm.h, lm_search)
    def search(self, sparams: Optional[LmSearchParams] = None, to_host: bool = True) -> dict:
        torch = self.torch
        sparams = sparams if sparams is not None else lm_search_default_params()
        nbytes = lm_search_workspace_bytes(self.d, self.B, self.n)
        if getattr(self, "search_workspace", None) is None or self._search_ws_bytes < nbytes:
            with self._on_stream():
                self.search_workspace, self._search_ws_ptr = self._alloc_ws(nbytes)
            self._search_ws_bytes = nbytes
        ptr = self._search_ws_ptr
        if not to_host:
            lm_search(self._ctx, sparams, ptr, nbytes, None, None, None)
            return {}
        choice = torch.empty((self.n,), dtype=torch.int32).pin_memory()
        xi = torch.empty((self.d, self.n), dtype=torch.float32).pin_memory()
        res = torch.empty((2,), dtype=torch.float32).pin_memory()
        lm_search(self._ctx, sparams, ptr, nbytes, choice.data_ptr(), xi.data_ptr(), res.data_ptr())
        return {"choice": choice.numpy().copy(), "xi": np.ascontiguousarray(xi.numpy().T), "cost": float(res[0]), "mjac": float(res[1])}

    def fetch_totals(self) -> tuple:
        """lm_fetch of the two scalar totals only (synchronises the stream)."""
        st = LmStats()
        lm_fetch(self._ctx, None, st)
        return int(st.total_waypoint_iters), int(st.converged_trajectories)

    def fk(self, q) -> tuple:
        """Device FK of q [count, d] -> (pos [count,3], R [count,3,3]) float64 numpy."""
        torch = self.torch
        q = np.asarray(q, dtype=np.float32)
        count = q.shape[0]
        with self._on_stream():
            qd = torch.from_numpy(np.ascontiguousarray(q.T)).to(self.device)
            pos = torch.empty((3, count), dtype=torch.float32, device=self.device)
            rot = torch.empty((9, count), dtype=torch.float32, device=self.device)
        lm_fk(self._ctx, qd.data_ptr(), count, pos.data_ptr(), rot.data_ptr())
        torch.cuda.synchronize(self.device)
        return (pos.cpu().numpy().T.astype(np.float64),
                rot.cpu().numpy().T.reshape(count, 3, 3).astype(np.float64))

    def close(self) -> None:
        if self._ctx is not None:
            self.torch.cuda.synchronize(self.device)
            lm_free(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def device_fk(chain, device: str = "cuda:0"):
    """An ``fk`` callable for workloads.*: FK on the GPU through lm_fk (S1 of the hot path)."""
    dummy = Solver(chain, 1, 1, np.zeros((1, 3), np.float32), np.array([[1, 0, 0, 0]], np.float32),
                   np.zeros((1, chain.dof), np.float32), device=device)

    def fk(q):
        q = np.asarray(q, dtype=np.float64)
        flat = q.reshape(-1, chain.dof)
        pos, R = dummy.fk(flat)
        return pos.reshape(q.shape[:-1] + (3,)), R.reshape(q.shape[:-1] + (3, 3))

    return fk
