"""ctypes wrapper around the fp64 CPU oracle (oracle/lm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the
paper_2309_09102_b200 package and the package imports nothing from here.

Arrays are waypoint-major (``q[W, d]``, ``target_pos[W, 3]``, ``target_quat[W, 4]``), fp64.
Citations: PAPER.md line numbers; "DESIGN R<n>" = readings listed in DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lm_oracle.c")
_HDR = os.path.join(_HERE, "lm_oracle.h")
_SRCS = [_SRC, os.path.join(_HERE, "lm_traj_oracle.c"), os.path.join(_HERE, "lm_coll_oracle.c")]  # one shared object
_DEPS = _SRCS + [_HDR, os.path.join(_HERE, "lm_traj_oracle.h"), os.path.join(_HERE, "lm_coll_oracle.h")]
# LM_ORACLE_SANITIZE=1: the same sources built with AddressSanitizer + UndefinedBehaviorSanitizer into a library of
# their own.  Run the CPU pins under it with
#   LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 LM_ORACLE_SANITIZE=1 \
#       python -m pytest tests -m "not gpu" -q
# (libasan must be loaded before python; leak detection is off because the interpreter itself "leaks").
_SANITIZE = os.environ.get("LM_ORACLE_SANITIZE", "") not in ("", "0")
_LIB = os.path.join(_HERE, "liblm_oracle_asan.so" if _SANITIZE else "liblm_oracle.so")
MAX_DOF = 8


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C11 + OpenMP for the timing leg)."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < max(os.path.getmtime(p) for p in _DEPS)
    if force or stale:
        tmp = _LIB + f".tmp{os.getpid()}"
        opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] \
            if _SANITIZE else ["-O2"]
        subprocess.check_call(["gcc"] + opt + ["-std=c11", "-Wall", "-Wextra", "-fPIC", "-fopenmp",
                               "-shared"] + _SRCS + ["-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Chain(C.Structure):
    _fields_ = [("dof", C.c_int32), ("joint_type", C.c_int32 * MAX_DOF),
                ("a", C.c_double * MAX_DOF), ("alpha", C.c_double * MAX_DOF),
                ("d", C.c_double * MAX_DOF), ("theta", C.c_double * MAX_DOF),
                ("q_lo", C.c_double * MAX_DOF), ("q_hi", C.c_double * MAX_DOF),
                ("tool_p", C.c_double * 3), ("tool_q", C.c_double * 4)]


class _Params(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("lambda0", "nu_up", "nu_down", "lambda_min", "lambda_max", "tol", "w_pos", "w_rot")] + [("rot_mode", C.c_int32)]


@dataclass
class Params:
    """LM constants, DESIGN R5/R7 (the paper gives none)."""
    lambda0: float = 1e-3
    nu_up: float = 10.0
    nu_down: float = 10.0
    lambda_min: float = 1e-4
    lambda_max: float = 1e7
    tol: float = 0.0
    w_pos: float = 1.0
    w_rot: float = 1.0
    rot_mode: int = 0   # 0: rotation-vector residual (DESIGN R2); 1: the paper's literal roll-pitch-yaw differences (variant)

    def _c(self) -> _Params:
        return _Params(self.lambda0, self.nu_up, self.nu_down, self.lambda_min, self.lambda_max,
                       self.tol, self.w_pos, self.w_rot, int(self.rot_mode))


def _chain_c(chain) -> _Chain:
    """`chain` is any object with dof, joint_type, a, alpha, d, theta, q_lo, q_hi, tool (xyz+wxyz)."""
    c = _Chain()
    n = int(chain.dof)
    assert 1 <= n <= MAX_DOF
    c.dof = n
    for name in ("a", "alpha", "d", "theta", "q_lo", "q_hi"):
        arr = np.asarray(getattr(chain, name), dtype=np.float64)
        assert arr.shape == (n,), name
        for j in range(n):
            getattr(c, name)[j] = float(arr[j])
    jt = np.asarray(chain.joint_type)
    for j in range(n):
        c.joint_type[j] = int(jt[j])
    tool = np.asarray(chain.tool, dtype=np.float64)
    for i in range(3):
        c.tool_p[i] = float(tool[i])
    for i in range(4):
        c.tool_q[i] = float(tool[3 + i])
    return c


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_fk.argtypes = [C.POINTER(_Chain), _dp, _dp, _dp, _dp, _dp]
        L.orc_fk.restype = None
        L.orc_quat_to_R.argtypes = [_dp, _dp]
        L.orc_log_so3.argtypes = [_dp, _dp]
        L.orc_residual.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, _dp]
        L.orc_rpy.argtypes = [_dp, _dp]
        L.orc_rpy.restype = None
        L.orc_residual_rpy.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, _dp]
        L.orc_residual_rpy.restype = None
        L.orc_jacobian_to_rpy.argtypes = [C.c_int, _dp, _dp]
        L.orc_jacobian_to_rpy.restype = None
        L.orc_jacobian.argtypes = [C.POINTER(_Chain), _dp, _dp]
        L.orc_lu_solve.argtypes = [C.c_int, _dp, _dp, _dp]
        L.orc_lu_solve.restype = C.c_int
        L.orc_lm_delta.argtypes = [C.c_int, _dp, _dp, C.c_double, _dp]
        L.orc_lm_delta.restype = C.c_int
        L.orc_lm_advance.argtypes = [C.POINTER(_Chain), C.POINTER(_Params), C.c_int64, _dp, _dp,
                                     _dp, _dp, C.POINTER(C.c_int32), C.POINTER(C.c_uint64),
                                     C.POINTER(C.c_uint32), C.c_int32, C.c_int32, _dp, _dp, _dp,
                                     _dp, _dp, _dp, C.POINTER(C.c_int32), C.c_int32]
        L.orc_lm_advance.restype = C.c_int64
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _f64(x, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


# --------------------------------------------------------------------------- single pieces

def fk(chain, q):
    """FK(q).  q: [..., d] -> p [..., 3], R [..., 3, 3]."""
    c = _chain_c(chain)
    q = _f64(q)
    flat = q.reshape(-1, chain.dof)
    p = np.empty((flat.shape[0], 3))
    R = np.empty((flat.shape[0], 9))
    L = lib()
    for i in range(flat.shape[0]):
        L.orc_fk(C.byref(c), _p(flat[i]), _p(p[i]), _p(R[i]), None, None)
    return p.reshape(q.shape[:-1] + (3,)), R.reshape(q.shape[:-1] + (3, 3))


def fk_axes(chain, q):
    """FK for one q, with joint axes z[d,3] and frame origins o[d,3]."""
    c = _chain_c(chain)
    q = _f64(q, (chain.dof,))
    p, R = np.empty(3), np.empty(9)
    z, o = np.empty((chain.dof, 3)), np.empty((chain.dof, 3))
    lib().orc_fk(C.byref(c), _p(q), _p(p), _p(R), _p(z), _p(o))
    return p, R.reshape(3, 3), z, o


def quat_to_R(quat):
    quat = _f64(quat, (4,))
    R = np.empty(9)
    lib().orc_quat_to_R(_p(quat), _p(R))
    return R.reshape(3, 3)


def log_so3(E):
    E = _f64(E, (3, 3))
    w = np.empty(3)
    lib().orc_log_so3(_p(E), _p(w))
    return w


def residual(p, R, target_pos, target_quat, w_pos=1.0, w_rot=1.0):
    r = np.empty(6)
    lib().orc_residual(_p(_f64(p, (3,))), _p(_f64(R, (3, 3))), _p(_f64(target_pos, (3,))),
                       _p(_f64(target_quat, (4,))), w_pos, w_rot, _p(r))
    return r


def rpy(R):
    """(roll, pitch, yaw) of R = Rz(yaw) Ry(pitch) Rx(roll)."""
    out = np.empty(3)
    lib().orc_rpy(_p(_f64(R, (3, 3))), _p(out))
    return out


def residual_rpy(p, R, target_pos, target_quat, w_pos=1.0, w_rot=1.0):
    r = np.empty(6)
    lib().orc_residual_rpy(_p(_f64(p, (3,))), _p(_f64(R, (3, 3))), _p(_f64(target_pos, (3,))),
                           _p(_f64(target_quat, (4,))), w_pos, w_rot, _p(r))
    return r


def jacobian_rpy(chain, q):
    """6 x d Jacobian of (x, y, z, roll, pitch, yaw) of the flange wrt q: rows 3..5 = E(rpy)^-1 J_w."""
    J = jacobian(chain, q)
    _, R = fk(chain, _f64(q, (chain.dof,)))
    lib().orc_jacobian_to_rpy(chain.dof, _p(_f64(R, (3, 3))), _p(J))
    return J


def jacobian(chain, q):
    """6 x d geometric Jacobian (DESIGN R3)."""
    c = _chain_c(chain)
    q = _f64(q, (chain.dof,))
    J = np.empty((6, chain.dof))
    lib().orc_jacobian(C.byref(c), _p(q), _p(J))
    return J


def lu_solve(A, b):
    A = _f64(A)
    n = A.shape[0]
    b = _f64(b, (n,))
    x = np.empty(n)
    rc = lib().orc_lu_solve(n, _p(A), _p(b), _p(x))
    if rc != 0:
        raise np.linalg.LinAlgError("singular")
    return x


def lm_delta(J, r, lam):
    """delta = -(J^T J + lam I)^-1 J^T r (DESIGN R4)."""
    J = _f64(J)
    n = J.shape[1]
    delta = np.empty(n)
    rc = lib().orc_lm_delta(n, _p(J), _p(_f64(r, (6,))), float(lam), _p(delta))
    if rc != 0:
        raise np.linalg.LinAlgError("singular")
    return delta


# --------------------------------------------------------------------------- batched LM

@dataclass
class State:
    """Per-waypoint LM state (waypoint-major)."""
    q: np.ndarray
    lam: np.ndarray
    iters: np.ndarray
    mask: np.ndarray
    status: np.ndarray
    res_norm: np.ndarray = field(default=None)
    pos_err: np.ndarray = field(default=None)
    rot_err: np.ndarray = field(default=None)
    # trace of the last iteration executed by the latest advance() call
    trial_q: np.ndarray = field(default=None)
    F_before: np.ndarray = field(default=None)
    F_trial: np.ndarray = field(default=None)
    accepted: np.ndarray = field(default=None)
    executed: int = 0

    def copy(self) -> "State":
        return State(**{k: (v.copy() if isinstance(v, np.ndarray) else v)
                        for k, v in self.__dict__.items()})


def init_state(seeds, params: Params) -> State:
    q = _f64(seeds).copy()
    W = q.shape[0]
    return State(q=q, lam=np.full(W, params.lambda0), iters=np.zeros(W, np.int32),
                 mask=np.zeros(W, np.uint64), status=np.zeros(W, np.uint32))


def advance(chain, params: Params, target_pos, target_quat, st: State, max_total_iters: int,
            at_most: int = -1, nthreads: int = 0) -> State:
    """Run LM on every waypoint until frozen / max_total_iters / at_most more iterations.

    Modifies and returns `st`.  The algorithm is the pseudo-code of DESIGN section "oracle"."""
    c = _chain_c(chain)
    W, d = st.q.shape
    assert d == chain.dof
    tp = _f64(target_pos, (W, 3))
    tq = _f64(target_quat, (W, 4))
    st.res_norm, st.pos_err, st.rot_err = np.empty(W), np.empty(W), np.empty(W)
    st.trial_q = np.full((W, d), np.nan)
    st.F_before, st.F_trial = np.full(W, np.nan), np.full(W, np.nan)
    st.accepted = np.full(W, -1, np.int32)
    prm = params._c()
    st.executed = int(lib().orc_lm_advance(
        C.byref(c), C.byref(prm), W, _p(tp), _p(tq), _p(st.q), _p(st.lam),
        st.iters.ctypes.data_as(C.POINTER(C.c_int32)), st.mask.ctypes.data_as(C.POINTER(C.c_uint64)),
        st.status.ctypes.data_as(C.POINTER(C.c_uint32)), int(max_total_iters), int(at_most),
        _p(st.res_norm), _p(st.pos_err), _p(st.rot_err), _p(st.trial_q), _p(st.F_before),
        _p(st.F_trial), st.accepted.ctypes.data_as(C.POINTER(C.c_int32)), int(nthreads)))
    return st


def lm_run(chain, params: Params, target_pos, target_quat, seeds, max_iters: int,
           nthreads: int = 0) -> State:
    return advance(chain, params, target_pos, target_quat, init_state(seeds, params), max_iters,
                   nthreads=nthreads)


def num_threads() -> int:
    return int(lib().orc_num_threads())
