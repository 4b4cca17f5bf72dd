"""Shared helpers of the parity tests: run the oracle / the CUDA path on one Workload and compare."""
from __future__ import annotations

import numpy as np

from oracle import lm_oracle as orc
from paper_2309_09102_b200 import workloads as wl

TOL_Q = 1e-4      # rad (m for prismatic) per joint        -- BASELINE.json north_star
TOL_POS = 1e-5    # m, pose error after a fixed iteration count
TOL_ROT = 1e-4    # rad


def oracle_fk(chain):
    return lambda q: orc.fk(chain, q)


def oracle_params(w: wl.Workload, **kw) -> orc.Params:
    return orc.Params(lambda0=w.lambda0, tol=w.tol, **kw)


def run_oracle(w: wl.Workload, max_iters=None, **kw) -> orc.State:
    return orc.lm_run(w.chain, oracle_params(w, **kw), w.target_pos.astype(np.float64),
                      w.target_quat.astype(np.float64), w.seeds.astype(np.float64),
                      w.max_iters if max_iters is None else max_iters)


def make_solver(w: wl.Workload, **kw):
    from paper_2309_09102_b200 import lm
    pkw = {k: kw.pop(k) for k in list(kw) if k in ("lambda_min", "lambda_max", "nu_up", "nu_down", "w_pos",
                                                    "w_rot", "refine_steps", "fast_sincos", "solver", "rot_residual")}
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol, **pkw)
    return lm.Solver(w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, **kw)


def run_gpu(w: wl.Workload, max_iters=None, **kw) -> dict:
    s = make_solver(w, **kw)
    s.run(w.max_iters if max_iters is None else max_iters)
    out = s.fetch()
    s.close()
    return out


def pose_errors_by_oracle(w: wl.Workload, q: np.ndarray):
    """Position / rotation error of joint values q against the targets, evaluated by the ORACLE's
    fp64 FK and residual (so the GPU's own fp32 FK error is part of what is measured)."""
    p, R = orc.fk(w.chain, q.astype(np.float64))
    pe, re = np.empty(w.W), np.empty(w.W)
    for i in range(w.W):
        r = orc.residual(p[i], R[i], w.target_pos[i].astype(np.float64), w.target_quat[i].astype(np.float64))
        pe[i], re[i] = np.linalg.norm(r[:3]), np.linalg.norm(r[3:])
    return pe, re


def mask_bits(mask: np.ndarray, n: int) -> np.ndarray:
    """[W] uint64 -> [W, n] bool"""
    return ((mask[:, None] >> np.arange(n, dtype=np.uint64)[None, :]) & np.uint64(1)).astype(bool)


def oracle_trace(w: wl.Workload, n_iters: int, **kw):
    """Oracle stepped one iteration at a time: list of (state_before, state_after) copies."""
    prm = oracle_params(w, **kw)
    st = orc.init_state(w.seeds.astype(np.float64), prm)
    tp, tq = w.target_pos.astype(np.float64), w.target_quat.astype(np.float64)
    # res_norm of the seeds (iteration 0 "before" state)
    out = []
    for _ in range(n_iters):
        before = st.copy()
        orc.advance(w.chain, prm, tp, tq, st, n_iters, at_most=1)
        out.append((before, st.copy()))
    return out


def decisive_mismatches(w: wl.Workload, gpu: dict, n_iters: int, floor: float = 1e-5, margin: float = 1e-3, **kw):
    """Compare accept/reject bits on the decisive iterations (P10): both sides
    executed iteration k, the oracle's sqrt(F) before it was >= floor, and the oracle's own
    decision had relative margin |F - F+| / F > margin.  Stops at the first mismatch of a
    waypoint (after it the two sequences are different problems).
    Returns (number of decisive decisions compared, number of waypoints with a mismatch)."""
    tr = oracle_trace(w, n_iters, **kw)
    gbits = mask_bits(gpu["mask"], n_iters)
    alive = np.ones(w.W, bool)
    compared, bad = 0, np.zeros(w.W, bool)
    for k, (b, a) in enumerate(tr):
        ran_o = a.accepted >= 0                      # oracle executed iteration k
        ran_g = gpu["iters"] > k
        Fb, Ft = a.F_before, a.F_trial
        with np.errstate(invalid="ignore", divide="ignore"):
            dec = ran_o & ran_g & alive & (np.sqrt(Fb) >= floor) & (np.abs(Fb - Ft) > margin * Fb)
        mism = dec & ((a.accepted == 1) != gbits[:, k])
        compared += int(dec.sum())
        bad |= mism
        # once the sequences part (decisive or not) later bits are not comparable
        alive &= ~(ran_o & ran_g & ((a.accepted == 1) != gbits[:, k]))
        alive &= ran_o & ran_g
    return compared, int(bad.sum())
