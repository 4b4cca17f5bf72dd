"""ctypes wrapper around the fp64 CPU oracle of the capsule-capsule collision residual
(oracle/lm_coll_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT."""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import lm_oracle as _o

MAX_CAPS, MAX_PAIRS, MAX_OBS = 16, 32, 8
_dp = C.POINTER(C.c_double)


class _Caps(C.Structure):
    _fields_ = [("ncaps", C.c_int32), ("link", C.c_int32 * MAX_CAPS), ("a", (C.c_double * 3) * MAX_CAPS),
                ("b", (C.c_double * 3) * MAX_CAPS), ("c", C.c_double * MAX_CAPS), ("npairs", C.c_int32),
                ("pair", (C.c_int32 * 2) * MAX_PAIRS), ("w_coll", C.c_double), ("d_safe", C.c_double),
                ("nobs", C.c_int32), ("Ro", (C.c_double * 9) * MAX_OBS), ("to", (C.c_double * 3) * MAX_OBS),
                ("pmin", (C.c_double * 3) * MAX_OBS), ("pmax", (C.c_double * 3) * MAX_OBS), ("nenv", C.c_int32),
                ("env_pair", (C.c_int32 * 2) * MAX_PAIRS), ("w_env", C.c_double), ("d_safe_env", C.c_double)]


@dataclass
class Capsules:
    """Capsule model of a robot (readings C1, C2, C4 of lm_coll_oracle.h): `model` is any object with
    link [K], a [K,3], b [K,3], radius [K], pairs [P,2] (e.g. workloads.CapsuleModel)."""
    model: object
    w_coll: float = 1.0
    d_safe: float = 0.05
    scene: object = None     # obstacles: R [M,3,3] (box axes as columns), t [M,3], pmin [M,3], pmax [M,3], pairs [Q,2] (capsule, obstacle)
    w_env: float = 0.0
    d_safe_env: float = 0.05

    def _c(self) -> _Caps:
        m = self.model
        s = _Caps()
        K, P = len(m.link), len(m.pairs)
        assert K <= MAX_CAPS and P <= MAX_PAIRS
        s.ncaps, s.npairs = K, P
        for k in range(K):
            s.link[k] = int(m.link[k])
            s.c[k] = float(m.radius[k])
            for i in range(3):
                s.a[k][i] = float(m.a[k][i])
                s.b[k][i] = float(m.b[k][i])
        for p in range(P):
            s.pair[p][0], s.pair[p][1] = int(m.pairs[p][0]), int(m.pairs[p][1])
        s.w_coll, s.d_safe = float(self.w_coll), float(self.d_safe)
        if self.scene is not None:
            sc = self.scene
            M, Q = len(sc.t), len(sc.pairs)
            assert M <= MAX_OBS and Q <= MAX_PAIRS
            s.nobs, s.nenv = M, Q
            for o in range(M):
                for i in range(9):
                    s.Ro[o][i] = float(np.asarray(sc.R[o]).reshape(9)[i])
                for i in range(3):
                    s.to[o][i], s.pmin[o][i], s.pmax[o][i] = float(sc.t[o][i]), float(sc.pmin[o][i]), float(sc.pmax[o][i])
            for p in range(Q):
                s.env_pair[p][0], s.env_pair[p][1] = int(sc.pairs[p][0]), int(sc.pairs[p][1])
            s.w_env, s.d_safe_env = float(self.w_env), float(self.d_safe_env)
        return s


_ready = False


def _lib():
    global _ready
    L = _o.lib()
    if not _ready:
        ch, cp = C.POINTER(_o._Chain), C.POINTER(_Caps)
        L.orc_segment_distance.argtypes = [_dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_segment_distance.restype = C.c_double
        L.orc_segment_box_distance.argtypes = [_dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_segment_box_distance.restype = C.c_double
        L.orc_coll_rows.argtypes = [cp]
        L.orc_coll_rows.restype = C.c_int
        L.orc_capsule_world.argtypes = [ch, cp, _dp, _dp, _dp]
        L.orc_capsule_world.restype = None
        L.orc_coll_residual.argtypes = [ch, cp, _dp, _dp, _dp]
        L.orc_coll_residual.restype = None
        L.orc_coll_jacobian.argtypes = [ch, cp, _dp, _dp]
        L.orc_coll_jacobian.restype = None
        L.orc_fk_frames.argtypes = [ch, _dp, _dp, _dp]
        L.orc_fk_frames.restype = None
        _ready = True
    return L


def _p(a):
    return a.ctypes.data_as(_dp)


def segment_distance(a1, b1, a2, b2):
    """(min distance, t1, t2) of the QP of PAPER.md:L163-166."""
    t1, t2 = C.c_double(), C.c_double()
    a1, b1, a2, b2 = (_o._f64(x, (3,)) for x in (a1, b1, a2, b2))
    d = _lib().orc_segment_distance(_p(a1), _p(b1), _p(a2), _p(b2), C.byref(t1), C.byref(t2))
    return float(d), float(t1.value), float(t2.value)


def segment_box_distance(a, b, pmin, pmax):
    """(min distance, t, p[3]) of the QP of PAPER.md:L176-178 (box frame)."""
    t = C.c_double()
    p = np.empty(3)
    a, b, pmin, pmax = (_o._f64(x, (3,)) for x in (a, b, pmin, pmax))
    d = _lib().orc_segment_box_distance(_p(a), _p(b), _p(pmin), _p(pmax), C.byref(t), _p(p))
    return float(d), float(t.value), p


def fk_frames(chain, q):
    c = _o._chain_c(chain)
    q = _o._f64(q, (chain.dof,))
    R, o = np.empty((chain.dof, 3, 3)), np.empty((chain.dof, 3))
    _lib().orc_fk_frames(C.byref(c), _p(q), _p(R), _p(o))
    return R, o


def capsule_world(chain, caps: Capsules, q):
    c, m = _o._chain_c(chain), caps._c()
    q = _o._f64(q, (chain.dof,))
    wa, wb = np.empty((m.ncaps, 3)), np.empty((m.ncaps, 3))
    _lib().orc_capsule_world(C.byref(c), C.byref(m), _p(q), _p(wa), _p(wb))
    return wa, wb


def residual(chain, caps: Capsules, q):
    """(dist [P], r [P]) at one configuration."""
    c, m = _o._chain_c(chain), caps._c()
    q = _o._f64(q, (chain.dof,))
    rows = int(_lib().orc_coll_rows(C.byref(m)))
    dist, r = np.empty(rows), np.empty(rows)
    _lib().orc_coll_residual(C.byref(c), C.byref(m), _p(q), _p(dist), _p(r))
    return dist, r


def jacobian(chain, caps: Capsules, q):
    c, m = _o._chain_c(chain), caps._c()
    q = _o._f64(q, (chain.dof,))
    J = np.empty((int(_lib().orc_coll_rows(C.byref(m))), chain.dof))
    _lib().orc_coll_jacobian(C.byref(c), C.byref(m), _p(q), _p(J))
    return J
