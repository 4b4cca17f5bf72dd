"""ctypes wrapper around the fp64 CPU oracle of the trajectory-level LM step (oracle/lm_traj_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/lm_oracle.py): only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import it.

Arrays are trajectory-major fp64: ``q[B, n, d]``, ``target_pos[B, n, 3]``, ``target_quat[B, n, 4]``
(single-trajectory functions take ``[n, ...]``).  Stacked residual of one trajectory
(Fig. 6):  r = [w_pose r_pose ; w_diff (q_{k+1} - q_k)_{k=1..n-1}].
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass, field

import numpy as np

from . import lm_coll_oracle as _co
from . import lm_oracle as _o

_dp = C.POINTER(C.c_double)


class _TParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("w_pose", "w_diff", "lambda0", "nu_up", "nu_down", "lambda_min", "lambda_max")] + [("caps", C.c_void_p)]


@dataclass
class TrajParams:
    """Weights and LM constants of the trajectory-level step (DESIGN T1/T3; the paper gives none)."""
    w_pose: float = 1.0
    w_diff: float = 1.0
    lambda0: float = 1e-3
    nu_up: float = 10.0
    nu_down: float = 10.0
    lambda_min: float = 1e-4
    lambda_max: float = 1e7
    caps: object = None   # lm_coll_oracle.Capsules or None: self-collision hinge rows

    def _c(self) -> _TParams:
        t = _TParams(self.w_pose, self.w_diff, self.lambda0, self.nu_up, self.nu_down,
                     self.lambda_min, self.lambda_max, None)
        if self.caps is not None:
            t._caps_keep = self.caps._c()          # keep the struct alive as long as the params struct
            t.caps = C.addressof(t._caps_keep)
        return t


_ready = False


def _lib():
    global _ready
    L = _o.lib()
    if not _ready:
        ch, pp, tp = C.POINTER(_o._Chain), C.POINTER(_o._Params), C.POINTER(_TParams)
        L.orc_traj_rows.argtypes = [C.c_int32, C.c_int64]
        L.orc_traj_rows.restype = C.c_int64
        L.orc_traj_rows_all.argtypes = [tp, C.c_int32, C.c_int64]
        L.orc_traj_rows_all.restype = C.c_int64
        L.orc_traj_residual.argtypes = [ch, pp, tp, C.c_int64, _dp, _dp, _dp, _dp]
        L.orc_traj_residual.restype = None
        L.orc_traj_jacobian.argtypes = [ch, pp, tp, C.c_int64, _dp, _dp]
        L.orc_traj_jacobian.restype = None
        for f in (L.orc_traj_delta_dense, L.orc_traj_delta_banded):
            f.argtypes = [ch, pp, tp, C.c_int64, _dp, _dp, _dp, C.c_double, _dp]
            f.restype = C.c_int
        L.orc_traj_lm_advance.argtypes = [ch, pp, tp, C.c_int64, C.c_int64, _dp, _dp, _dp, _dp,
                                          C.POINTER(C.c_int32), C.POINTER(C.c_uint64), C.POINTER(C.c_uint32),
                                          C.c_int32, C.c_int32, _dp, _dp, _dp, _dp, _dp, _dp,
                                          C.POINTER(C.c_int32), C.c_int32, C.c_int32]
        L.orc_traj_lm_advance.restype = C.c_int64
        _ready = True
    return L


def _p(a):
    return a.ctypes.data_as(_dp)


def rows(dof: int, n: int, tparams: "TrajParams" = None) -> int:
    if tparams is None:
        return int(_lib().orc_traj_rows(dof, n))
    tp = tparams._c()
    return int(_lib().orc_traj_rows_all(C.byref(tp), dof, n))


def residual(chain, pose_params: _o.Params, tparams: TrajParams, target_pos, target_quat, q):
    """Stacked residual r[6n + d(n-1)] of one trajectory q[n, d]."""
    q = _o._f64(q)
    n, d = q.shape
    c, pp, tp = _o._chain_c(chain), pose_params._c(), tparams._c()
    r = np.empty(rows(d, n, tparams))
    _lib().orc_traj_residual(C.byref(c), C.byref(pp), C.byref(tp), n, _p(_o._f64(target_pos, (n, 3))),
                             _p(_o._f64(target_quat, (n, 4))), _p(q), _p(r))
    return r


def jacobian(chain, pose_params: _o.Params, tparams: TrajParams, q):
    """Dense Jacobian [6n + d(n-1), n d] of the stacked residual as the paper states it (L121, L123)."""
    q = _o._f64(q)
    n, d = q.shape
    c, pp, tp = _o._chain_c(chain), pose_params._c(), tparams._c()
    J = np.empty((rows(d, n, tparams), n * d))
    _lib().orc_traj_jacobian(C.byref(c), C.byref(pp), C.byref(tp), n, _p(q), _p(J))
    return J


def delta(chain, pose_params: _o.Params, tparams: TrajParams, target_pos, target_quat, q, lam: float,
          dense: bool = False):
    """LM step delta[n, d] = -(J^T J + lam I)^-1 J^T r of one trajectory (dense LU or banded Cholesky)."""
    q = _o._f64(q)
    n, d = q.shape
    c, pp, tp = _o._chain_c(chain), pose_params._c(), tparams._c()
    out = np.empty((n, d))
    f = _lib().orc_traj_delta_dense if dense else _lib().orc_traj_delta_banded
    rc = f(C.byref(c), C.byref(pp), C.byref(tp), n, _p(_o._f64(target_pos, (n, 3))),
           _p(_o._f64(target_quat, (n, 4))), _p(q), float(lam), _p(out))
    if rc != 0:
        raise np.linalg.LinAlgError("singular / not positive definite")
    return out


@dataclass
class TrajState:
    """Per-trajectory LM state."""
    q: np.ndarray          # [B, n, d]
    lam: np.ndarray        # [B]
    iters: np.ndarray
    mask: np.ndarray
    status: np.ndarray
    F_total: np.ndarray = field(default=None)
    F_pose: np.ndarray = field(default=None)
    F_diff: np.ndarray = field(default=None)
    trial_q: np.ndarray = field(default=None)
    F_before: np.ndarray = field(default=None)
    F_trial: np.ndarray = field(default=None)
    accepted: np.ndarray = field(default=None)
    executed: int = 0

    def copy(self) -> "TrajState":
        return TrajState(**{k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in self.__dict__.items()})


def init_state(q0, tparams: TrajParams) -> TrajState:
    q = _o._f64(q0).copy()
    B = q.shape[0]
    return TrajState(q=q, lam=np.full(B, tparams.lambda0), iters=np.zeros(B, np.int32),
                     mask=np.zeros(B, np.uint64), status=np.zeros(B, np.uint32))


def advance(chain, pose_params: _o.Params, tparams: TrajParams, target_pos, target_quat, st: TrajState,
            max_total_iters: int, at_most: int = -1, dense: bool = False, nthreads: int = 0) -> TrajState:
    """Trajectory-level LM on every trajectory until max_total_iters / at_most more iterations."""
    B, n, d = st.q.shape
    assert d == chain.dof
    c, pp, tp = _o._chain_c(chain), pose_params._c(), tparams._c()
    tpos = _o._f64(target_pos, (B, n, 3))
    tq = _o._f64(target_quat, (B, n, 4))
    st.F_total, st.F_pose, st.F_diff = np.empty(B), np.empty(B), np.empty(B)
    st.trial_q = np.full((B, n, d), np.nan)
    st.F_before, st.F_trial = np.full(B, np.nan), np.full(B, np.nan)
    st.accepted = np.full(B, -1, np.int32)
    st.executed = int(_lib().orc_traj_lm_advance(
        C.byref(c), C.byref(pp), C.byref(tp), B, n, _p(tpos), _p(tq), _p(st.q), _p(st.lam),
        st.iters.ctypes.data_as(C.POINTER(C.c_int32)), st.mask.ctypes.data_as(C.POINTER(C.c_uint64)),
        st.status.ctypes.data_as(C.POINTER(C.c_uint32)), int(max_total_iters), int(at_most),
        _p(st.F_total), _p(st.F_pose), _p(st.F_diff), _p(st.trial_q), _p(st.F_before), _p(st.F_trial),
        st.accepted.ctypes.data_as(C.POINTER(C.c_int32)), int(bool(dense)), int(nthreads)))
    return st


def lm_run(chain, pose_params: _o.Params, tparams: TrajParams, target_pos, target_quat, q0, max_iters: int,
           dense: bool = False, nthreads: int = 0) -> TrajState:
    return advance(chain, pose_params, tparams, target_pos, target_quat, init_state(q0, tparams), max_iters,
                   dense=dense, nthreads=nthreads)
