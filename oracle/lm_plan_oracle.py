"""fp64 CPU ORACLE of the optimiser's non-stationary schedule with anytime bookkeeping
(CppFlow, arxiv 2309.09102 sec. III-C).

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as oracle/lm_oracle.py).  Plain Python / numpy
around the two C oracles, in the paper's order:

  "the optimizer optimizes for pose error exclusively until the positional and rotational error of
   the end effector is below the respective specified threshold at every timestep.  A trajectory
   length and obstacle avoidance optimization step is then taken, after which the optimizer switches
   back to pose only, and the cycle continues."
  "The optimizer keeps track of the latest valid solution"

Validity of a trajectory: positional error < 0.1 mm and rotational
(geodesic) error < 0.1 deg at every timestep, joints inside their limits (enforced by clamping,
L170), and no joint changes by more than 7 deg (revolute) / 2 cm (prismatic) across a timestep.
Trajectory length: "the cumulative change in configuration-space across a
trajectory (measured in radians and meters)" = sum_i sum_j |q_{i+1}[j] - q_i[j]|.
mjac: max_i max_j |q_{i+1}[j] - q_i[j]|, here kept per joint type because the two
limits have different units.  With a capsule model (lm_coll_oracle.py, synthetic) a valid trajectory is also
collision free: "At no timestep in the trajectory can the robot collide with itself or the environment" (L49).

Readings: P1 a pose-only phase is lm_run from fresh LM state (lambda0,
0 iterations) with the per-waypoint freeze |r|_2 < tol, capped at `pose_iters`; P2 the
trajectory-level step is ONE iteration of the stacked-residual LM and only
trajectories that are pose-valid at that moment take it; its lambda persists across cycles;
P3 "latest valid" = the most recent trajectory that passed the validity test, recorded right
after a pose phase; P4 after the last cycle one more pose phase and one more record.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import lm_coll_oracle as corc
from . import lm_oracle as orc
from . import lm_traj_oracle as torc

DEG = np.pi / 180.0


@dataclass
class PlanParams:
    pos_tol: float = 1e-4          # m,
    rot_tol: float = 0.1 * DEG     # rad
    mjac_rev: float = 7.0 * DEG    # rad
    mjac_pris: float = 0.02        # m,
    pose_iters: int = 10           # cap of each pose-only phase (reading P1)
    min_clearance: float = 0.0     # m: with a capsule model, every listed pair keeps at least this clearance


def trajectory_length(q: np.ndarray) -> np.ndarray:
    """q [B, n, d] -> [B]: cumulative change in configuration space."""
    return np.abs(np.diff(q, axis=1)).sum(axis=(1, 2))


def mjac(q: np.ndarray, joint_type: np.ndarray):
    """q [B, n, d] -> (max change of a revolute joint [B], of a prismatic joint [B]) across a timestep."""
    B, n, d = q.shape
    if n < 2:
        return np.zeros(B), np.zeros(B)
    dq = np.abs(np.diff(q, axis=1))
    rev, pris = joint_type == 0, joint_type == 1
    mr = dq[:, :, rev].max(axis=(1, 2)) if rev.any() else np.zeros(B)
    mp = dq[:, :, pris].max(axis=(1, 2)) if pris.any() else np.zeros(B)
    return mr, mp


@dataclass
class PlanResult:
    q: np.ndarray                   # [B, n, d] current trajectory at the end
    q_valid: np.ndarray             # [B, n, d] latest valid trajectory (NaN where none)
    valid: np.ndarray               # [B] bool: a valid trajectory has been recorded
    first_valid_cycle: np.ndarray   # [B] int (-1 = never); cycle 0 = after the first pose phase
    length: np.ndarray              # [B] trajectory length of the recorded trajectory (NaN where none)
    records: np.ndarray             # [B] how many times a valid trajectory was recorded
    max_pos_err: np.ndarray         # [B] of the current trajectory, after the last pose phase
    max_rot_err: np.ndarray
    mjac_rev: np.ndarray
    mjac_pris: np.ndarray
    traj_mask: np.ndarray           # [B] uint64 accept bits of the trajectory-level steps taken
    traj_iters: np.ndarray          # [B] trajectory-level steps taken
    history: list = field(default_factory=list)  # per record point: dict(valid_now, margins)


def min_clearance(chain, caps, q: np.ndarray) -> np.ndarray:
    """q [B, n, d] -> [B]: smallest clearance over all listed capsule pairs and all waypoints."""
    B, n, _ = q.shape
    return np.array([min(corc.residual(chain, caps, q[b, i])[0].min() for i in range(n)) for b in range(B)])


def plan(chain, pose_params: orc.Params, tparams: torc.TrajParams, pparams: PlanParams, target_pos, target_quat,
         seeds, cycles: int, nthreads: int = 0) -> PlanResult:
    """target_pos [B, n, 3], target_quat [B, n, 4], seeds [B, n, d] (fp64).  With tparams.caps set, the collision
    rows are part of the trajectory-level step and a valid trajectory must also be collision free."""
    q = np.array(seeds, dtype=np.float64)
    B, n, d = q.shape
    tp = np.asarray(target_pos, np.float64).reshape(B * n, 3)
    tq = np.asarray(target_quat, np.float64).reshape(B * n, 4)
    jt = np.asarray(chain.joint_type)
    tst = torc.init_state(q, tparams)           # per-trajectory lambda / mask persist across cycles (P2)
    q_valid = np.full_like(q, np.nan)
    valid = np.zeros(B, bool)
    first = np.full(B, -1, np.int64)
    length = np.full(B, np.nan)
    records = np.zeros(B, np.int64)
    hist = []
    pe = re_ = None
    for c in range(cycles + 1):
        # ---- pose-only phase from fresh LM state (P1)
        st = orc.lm_run(chain, pose_params, tp, tq, q.reshape(B * n, d), pparams.pose_iters, nthreads=nthreads)
        q = st.q.reshape(B, n, d)
        pe = st.pos_err.reshape(B, n).max(axis=1)
        re_ = st.rot_err.reshape(B, n).max(axis=1)
        mr, mp = mjac(q, jt)
        ok = (pe < pparams.pos_tol) & (re_ < pparams.rot_tol) & (mr <= pparams.mjac_rev) & (mp <= pparams.mjac_pris)
        clr = None
        if tparams.caps is not None:
            clr = min_clearance(chain, tparams.caps, q)
            ok &= clr >= pparams.min_clearance
        # ---- anytime bookkeeping (P3)
        q_valid[ok] = q[ok]
        length[ok] = trajectory_length(q[ok])
        first[ok & ~valid] = c
        valid |= ok
        records += ok
        hist.append({"valid_now": ok.copy(), "pos": pe.copy(), "rot": re_.copy(), "mjac_rev": mr.copy(), "mjac_pris": mp.copy(),
                     "clearance": None if clr is None else clr.copy()})
        if c == cycles:
            break
        # ---- one trajectory-level step for the trajectories that are pose-valid now (P2)
        pose_ok = (pe < pparams.pos_tol) & (re_ < pparams.rot_tol)
        if pose_ok.any():
            sub = torc.TrajState(q=np.ascontiguousarray(q[pose_ok]), lam=tst.lam[pose_ok].copy(), iters=tst.iters[pose_ok].copy(),
                                 mask=tst.mask[pose_ok].copy(), status=tst.status[pose_ok].copy())
            torc.advance(chain, orc.Params(w_pos=pose_params.w_pos, w_rot=pose_params.w_rot), tparams,
                         tp.reshape(B, n, 3)[pose_ok], tq.reshape(B, n, 4)[pose_ok], sub, 64, at_most=1, nthreads=nthreads)
            q[pose_ok] = sub.q
            tst.lam[pose_ok], tst.iters[pose_ok], tst.mask[pose_ok], tst.status[pose_ok] = sub.lam, sub.iters, sub.mask, sub.status
    mr, mp = mjac(q, jt)
    return PlanResult(q=q, q_valid=q_valid, valid=valid, first_valid_cycle=first, length=length, records=records,
                      max_pos_err=pe, max_rot_err=re_, mjac_rev=mr, mjac_pris=mp, traj_mask=tst.mask.copy(),
                      traj_iters=tst.iters.copy(), history=hist)
