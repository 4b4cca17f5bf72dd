"""Seeded synthetic inputs for the batched-LM hot path.

This module serves BOTH the CUDA path and the oracle's tests and therefore holds none of the
method's arithmetic: no forward kinematics, residual, Jacobian or solver.  Target poses are
obtained through an ``fk`` callable passed in by the caller (tests pass the oracle's FK; bench.py
passes the library's device FK): ``fk(q[W, d] float64) -> (pos[W, 3], R[W, 3, 3])``.

The inputs stand in for the paper's 13 planning problems, whose target paths,
scenes and robot models are not available: they keep the shapes the paper states -- 7-/8-DoF
serial arms (L190), smooth n-pose SE(3) paths (L85), seeds "in close vicinity to a valid
solution" (L109).  Sizes follow BASELINE.json configs[0..4].

Everything is drawn in fp64 from ``numpy.random.default_rng(seed)`` and rounded to fp32 ONCE;
both sides read the same rounded values.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np
from scipy.spatial.transform import Rotation

PI = np.pi


@dataclass
class Chain:
    """Serial chain in modified-DH (Craig) form, DESIGN R1 (config data, no arithmetic)."""
    name: str
    dof: int
    joint_type: np.ndarray  # [d] 0 revolute, 1 prismatic
    a: np.ndarray           # [d] a_{j-1}  (m)
    alpha: np.ndarray       # [d] alpha_{j-1} (rad)
    d: np.ndarray           # [d] d_j (m)
    theta: np.ndarray       # [d] theta offset (rad)
    q_lo: np.ndarray
    q_hi: np.ndarray
    tool: np.ndarray        # [7] xyz + quaternion wxyz


def panda_chain() -> Chain:
    """Franka Panda, modified DH from the manufacturer's public documentation (BASELINE.json
    configs[0] "standard Franka Panda DH table"); flange offset 0.107 m."""
    return Chain(
        name="panda", dof=7, joint_type=np.zeros(7, np.int32),
        a=np.array([0, 0, 0, 0.0825, -0.0825, 0, 0.088]),
        alpha=np.array([0, -PI / 2, PI / 2, PI / 2, -PI / 2, PI / 2, PI / 2]),
        d=np.array([0.333, 0, 0.316, 0, 0.384, 0, 0]),
        theta=np.zeros(7),
        q_lo=np.array([-2.8973, -1.7628, -2.8973, -3.0718, -2.8973, -0.0175, -2.8973]),
        q_hi=np.array([2.8973, 1.7628, 2.8973, -0.0698, 2.8973, 3.7525, 2.8973]),
        tool=np.array([0, 0, 0.107, 1, 0, 0, 0], dtype=np.float64))


def random_chain_8dof(seed: int = 3) -> Chain:
    """8-DoF chain of BASELINE.json configs[2]: joint 1 prismatic along z (range 0..0.38 m, like
    the Fetch torso lift), joints 2-8 revolute with one of (a, d) ~ U[0.05, 0.4] m
    and alpha drawn from {0, +-pi/2}, theta offsets ~ U(-pi, pi); limits +-2.5 rad.  No two
    consecutive alpha = 0 so the arm is spatial, not planar; the theta offsets move the mid-range
    configuration away from the all-zero (stretched, near-singular) pose."""
    rng = np.random.default_rng(seed)
    d_ = 8
    a = np.zeros(d_)
    dd = np.zeros(d_)
    alpha = np.zeros(d_)
    prev_zero = True  # joint 1 has alpha = 0
    for j in range(1, d_):
        length = rng.uniform(0.05, 0.4)
        if rng.random() < 0.5:
            a[j] = length
        else:
            dd[j] = length
        choices = [-PI / 2, PI / 2] if prev_zero else [0.0, -PI / 2, PI / 2]
        alpha[j] = choices[rng.integers(len(choices))]
        prev_zero = alpha[j] == 0.0
    theta = rng.uniform(-PI, PI, size=d_)
    theta[0] = 0.0
    jt = np.zeros(d_, np.int32)
    jt[0] = 1
    lo = np.full(d_, -2.5)
    hi = np.full(d_, 2.5)
    lo[0], hi[0] = 0.0, 0.38
    return Chain(name=f"rand8_{seed}", dof=d_, joint_type=jt, a=a, alpha=alpha, d=dd,
                 theta=theta, q_lo=lo, q_hi=hi,
                 tool=np.array([0, 0, 0.1, 1, 0, 0, 0], dtype=np.float64))


@dataclass
class CapsuleModel:
    """Capsules rigidly attached to link frames and the pairs to check -- config data.
    link[k] = -1 for the base (world) frame, j for the frame that joint j (0-based) moves."""
    name: str
    link: np.ndarray     # [K] int
    a: np.ndarray        # [K, 3] endpoint in the link frame (m)
    b: np.ndarray        # [K, 3]
    radius: np.ndarray   # [K] (m)
    pairs: np.ndarray    # [P, 2] capsule indices


def panda_capsules() -> CapsuleModel:
    """SYNTHETIC capsule model for the Panda DH chain (the paper fits capsules to the link meshes, which are
    not available): one capsule per major link placed along the link's extent in its modified-DH frame --
    base column, shoulder, upper arm, elbow, forearm, wrist, hand -- and the 9 pairs of non-adjacent links
    that can actually meet."""
    link = np.array([-1, 0, 2, 3, 4, 5, 6])
    a = np.array([[0, 0, 0.0], [0, 0, -0.10], [0, 0, -0.25], [0, 0, -0.03], [0, 0, -0.30], [0, 0, -0.02], [0, 0, 0.02]], float)
    b = np.array([[0, 0, 0.25], [0, 0, 0.0], [0, 0, -0.05], [0, 0, 0.03], [0, 0, -0.05], [0, 0, 0.05], [0, 0, 0.17]], float)
    radius = np.array([0.09, 0.08, 0.07, 0.07, 0.06, 0.06, 0.05])
    pairs = np.array([[0, 4], [0, 5], [0, 6], [1, 4], [1, 5], [1, 6], [2, 5], [2, 6], [3, 6]])
    return CapsuleModel("panda_synthetic", link, a, b, radius, pairs)


def chain_capsules(chain: "Chain", radius: float = 0.05) -> CapsuleModel:
    """SYNTHETIC capsule model for any chain: one capsule per joint frame along its z axis (+-6 cm), one on the
    base, all pairs at least three links apart."""
    d = chain.dof
    link = np.arange(-1, d)
    a = np.tile(np.array([0, 0, -0.06]), (d + 1, 1)).astype(float)
    b = np.tile(np.array([0, 0, 0.06]), (d + 1, 1)).astype(float)
    pairs = np.array([[i, j] for i in range(d + 1) for j in range(i + 3, d + 1)])
    return CapsuleModel(f"{chain.name}_synthetic", link, a, b, np.full(d + 1, radius), pairs)


@dataclass
class ObstacleScene:
    """Cuboid obstacles "with arbitrary spatial positioning": frame of each box in the world
    (R = box axes as columns, t = origin), extents pmin / pmax in that frame, and the (capsule, obstacle)
    pairs to check -- config data."""
    name: str
    R: np.ndarray      # [M, 3, 3]
    t: np.ndarray      # [M, 3]
    pmin: np.ndarray   # [M, 3]
    pmax: np.ndarray   # [M, 3]
    pairs: np.ndarray  # [Q, 2] (capsule index, obstacle index)

    @property
    def pose(self) -> np.ndarray:
        """[M, 7] xyz + unit quaternion (w, x, y, z) of every box frame: the form include/lm.h's lm_obstacles takes."""
        return np.concatenate([np.asarray(self.t, dtype=np.float64), _R_to_quat_wxyz(np.asarray(self.R, dtype=np.float64))], axis=1)


def panda_scene(seed: int = 7) -> ObstacleScene:
    """SYNTHETIC scene for the Panda capsule model (the paper's obstacle scenes are not available): a table slab in
    front of the robot, a tilted post beside it and a small box above the table; forearm, wrist and hand capsules
    are checked against all three, the elbow against the post."""
    rng = np.random.default_rng(seed)
    R = np.stack([np.eye(3), Rotation.from_rotvec([0.2, -0.1, 0.5]).as_matrix(),
                  Rotation.from_rotvec(rng.normal(size=3) * 0.4).as_matrix()])
    t = np.array([[0.55, 0.0, 0.15], [0.25, 0.45, 0.35], [0.45, -0.25, 0.45]])
    half = np.array([[0.30, 0.40, 0.02], [0.05, 0.05, 0.35], [0.08, 0.06, 0.10]])
    pairs = np.array([[4, 0], [5, 0], [6, 0], [4, 1], [5, 1], [6, 1], [3, 1], [4, 2], [5, 2], [6, 2]])
    return ObstacleScene("panda_synthetic_scene", R, t, -half, half, pairs)


@dataclass
class Workload:
    name: str
    chain: Chain
    B: int
    n: int
    target_pos: np.ndarray   # [W, 3] float32
    target_quat: np.ndarray  # [W, 4] float32, w x y z
    seeds: np.ndarray        # [W, d] float32, inside the joint limits
    tol: float               # DESIGN R7/R8: 0 = fixed iteration count
    max_iters: int
    lambda0: float = 1e-3
    truth: Optional[np.ndarray] = field(default=None)  # [W, d] float64 (None for config 4)

    @property
    def W(self) -> int:
        return self.B * self.n

    def subset(self, traj: slice) -> "Workload":
        """Trajectories traj.start..traj.stop as their own workload (waypoint w = b*n + i)."""
        b0, b1, _ = traj.indices(self.B)
        s = slice(b0 * self.n, b1 * self.n)
        return Workload(self.name, self.chain, b1 - b0, self.n, self.target_pos[s], self.target_quat[s],
                        self.seeds[s], self.tol, self.max_iters, self.lambda0,
                        None if self.truth is None else self.truth[s])


FkFn = Callable[[np.ndarray], tuple]


def _R_to_quat_wxyz(R: np.ndarray) -> np.ndarray:
    xyzw = Rotation.from_matrix(R).as_quat()
    return np.concatenate([xyzw[:, 3:4], xyzw[:, 0:3]], axis=1)


def smooth_joint_paths(chain: Chain, B: int, n: int, n_sin: int, amp: float,
                       rng: np.random.Generator) -> np.ndarray:
    """q*[B, n, d]: q*_j(t) = c_j + sum_m a_jm sin(2 pi f_jm t + phi_jm), t in [0, 1], c = mid-range,
    sum_m |a_jm| = amp (capped at 40 % of the joint's range), f ~ U[0.5, 3], phi ~ U[0, 2 pi)."""
    d = chain.dof
    t = np.linspace(0.0, 1.0, n)
    mid = 0.5 * (chain.q_lo + chain.q_hi)
    amp_j = np.minimum(amp, 0.4 * (chain.q_hi - chain.q_lo))
    wts = rng.uniform(0.2, 1.0, size=(B, d, n_sin)) * rng.choice([-1.0, 1.0], size=(B, d, n_sin))
    wts *= (amp_j[None, :, None] / np.abs(wts).sum(axis=2, keepdims=True))
    f = rng.uniform(0.5, 3.0, size=(B, d, n_sin))
    phi = rng.uniform(0.0, 2 * PI, size=(B, d, n_sin))
    arg = 2 * PI * f[:, None, :, :] * t[None, :, None, None] + phi[:, None, :, :]
    return mid[None, None, :] + (wts[:, None, :, :] * np.sin(arg)).sum(axis=3)


def _noisy_seeds(chain: Chain, base: np.ndarray, sigma: float, rng: np.random.Generator) -> np.ndarray:
    """base + N(0, sigma) rad on revolute joints, N(0, sigma/10) m on prismatic ones (a paper-free
    choice, DESIGN input recipe), clamped to the joint limits and rounded to fp32 so that the
    rounded value is still inside the limits."""
    sig = np.where(chain.joint_type == 1, sigma / 10.0, sigma)
    s = base + rng.normal(size=base.shape) * sig
    lo32 = np.nextafter(chain.q_lo.astype(np.float32), np.float32(np.inf))
    hi32 = np.nextafter(chain.q_hi.astype(np.float32), np.float32(-np.inf))
    return np.clip(s.astype(np.float32), lo32, hi32)


def _from_truth(name, chain, truth, sigma, rng, fk: FkFn, tol, max_iters, lambda0=1e-3) -> Workload:
    B, n, d = truth.shape
    flat = truth.reshape(B * n, d)
    pos, R = fk(flat)
    return Workload(name=name, chain=chain, B=B, n=n,
                    target_pos=np.asarray(pos, np.float64).astype(np.float32),
                    target_quat=_R_to_quat_wxyz(np.asarray(R, np.float64)).astype(np.float32),
                    seeds=_noisy_seeds(chain, flat, sigma, rng), tol=tol, max_iters=max_iters,
                    lambda0=lambda0, truth=flat)


def config1(fk: FkFn, seed_offset: int = 0) -> Workload:
    """BASELINE.json configs[0]: 1 x 50, Panda, 3 sinusoids amp 0.3, seeds N(0, 0.05), 20 iters."""
    rng = np.random.default_rng(1 + seed_offset)
    ch = panda_chain()
    return _from_truth("C1", ch, smooth_joint_paths(ch, 1, 50, 3, 0.3, rng), 0.05, rng, fk, 0.0, 20)


def config2(fk: FkFn, B: int = 512, n: int = 300, seed_offset: int = 0) -> Workload:
    """configs[1]: 512 x 300, Panda, 5 sinusoids amp 0.5, seeds N(0, 0.1), tol 1e-5, <= 50 iters."""
    rng = np.random.default_rng(2 + seed_offset)
    ch = panda_chain()
    return _from_truth("C2", ch, smooth_joint_paths(ch, B, n, 5, 0.5, rng), 0.1, rng, fk, 1e-5, 50)


def config3(fk: FkFn, B: int = 2048, n: int = 300, seed_offset: int = 0) -> Workload:
    """configs[2]: 2048 x 300, 8-DoF chain with one prismatic joint, seeds N(0, 0.15)."""
    ch = random_chain_8dof(3)
    rng = np.random.default_rng(4 + seed_offset)
    return _from_truth("C3", ch, smooth_joint_paths(ch, B, n, 5, 0.5, rng), 0.15, rng, fk, 1e-5, 50)


def config5(fk: FkFn, B: int, n: int, seed_offset: int = 0) -> Workload:
    """configs[4] sweep point: B x n, Panda, paths as config 2, fixed 20 iterations."""
    rng = np.random.default_rng(6 + seed_offset)
    ch = panda_chain()
    return _from_truth(f"C5_{B}x{n}", ch, smooth_joint_paths(ch, B, n, 5, 0.5, rng), 0.1, rng, fk, 0.0, 20)


def config4(fk: FkFn, B: int = 4096, n: int = 300, seed_offset: int = 0) -> Workload:
    """configs[3]: 4096 x 300, Panda; SE(3) lines / circles (radius U[0.1, 0.3] m), orientation
    slerp over <= 90 deg; seeds = anchor configuration + N(0, 0.2) at every waypoint; 50 iters.
    Reachability of the far end of a path is NOT guaranteed -- that is the workload."""
    rng = np.random.default_rng(5 + seed_offset)
    ch = panda_chain()
    d = ch.dof
    mid = 0.5 * (ch.q_lo + ch.q_hi)
    half = 0.5 * (ch.q_hi - ch.q_lo)
    q_c = mid + 0.6 * half * rng.uniform(-1.0, 1.0, size=(B, d))  # central 60 % of each range
    p0, R0 = fk(q_c)
    p0 = np.asarray(p0, np.float64)
    R0 = np.asarray(R0, np.float64)
    t = np.linspace(0.0, 1.0, n)
    rho = rng.uniform(0.1, 0.3, size=B)
    # random orthonormal pair (u, v) spanning the path's plane
    u = rng.normal(size=(B, 3))
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    v = rng.normal(size=(B, 3))
    v -= (v * u).sum(axis=1, keepdims=True) * u
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    is_circle = rng.random(B) < 0.5
    ang = 2 * PI * t[None, :]
    circle = rho[:, None, None] * ((np.cos(ang) - 1.0)[:, :, None] * u[:, None, :]
                                   + np.sin(ang)[:, :, None] * v[:, None, :])  # through p0 at t=0
    line = (2.0 * rho[:, None] * t[None, :])[:, :, None] * u[:, None, :]        # length 2 rho
    pos = p0[:, None, :] + np.where(is_circle[:, None, None], circle, line)
    axis = rng.normal(size=(B, 3))
    axis /= np.linalg.norm(axis, axis=1, keepdims=True)
    phi = rng.uniform(0.0, PI / 2, size=B)
    rotvec = (t[None, :, None] * phi[:, None, None]) * axis[:, None, :]         # [B, n, 3]
    Rt = Rotation.from_rotvec(rotvec.reshape(-1, 3)).as_matrix().reshape(B, n, 3, 3) @ R0[:, None]
    quat = _R_to_quat_wxyz(Rt.reshape(-1, 3, 3))
    base = np.repeat(q_c[:, None, :], n, axis=1).reshape(B * n, d)
    return Workload(name="C4", chain=ch, B=B, n=n, target_pos=pos.reshape(-1, 3).astype(np.float32),
                    target_quat=quat.astype(np.float32), seeds=_noisy_seeds(ch, base, 0.2, rng),
                    tol=0.0, max_iters=50, truth=None)


def to_soa(x: np.ndarray) -> np.ndarray:
    """[W, k] waypoint-major -> [k, W] structure-of-arrays (the device layout, include/lm.h)."""
    return np.ascontiguousarray(x.T)


def search_candidates(ch: Chain, K: int, n: int, seed: int, jump: float = 0.8, quant=None, limit_frac: float = 0.0) -> np.ndarray:
    """Input of the global discrete search (synthetic stand-in for K IK-generated motion plans of one
    path): q [K, n, d] fp32.  K candidate trajectories of one path as the search stage sees them: smooth pieces on different self-motion
    branches, each with a few pieces on another branch (a jump in, a jump out); optionally quantised (many exact ties) and with some values pushed to a limit."""
    rng = np.random.default_rng(seed)
    base = smooth_joint_paths(ch, 1, n, 3, 0.3, rng)[0]
    t = np.linspace(0.0, 1.0, n)[None, :, None]
    q = base[None] + 0.03 * np.sin(2 * np.pi * (t * rng.uniform(0.5, 2.0, (K, 1, ch.dof)) + rng.random((K, 1, ch.dof))))
    for k in range(K):
        for _ in range(int(rng.integers(1, 4)) if K > 1 else 0):    # every candidate jumps somewhere: no single one is smooth
            i0 = int(rng.integers(1, max(n, 2)))
            i1 = i0 + 1 + int(rng.integers(0, max(n // 3, 1)))
            q[k, i0:i1, :] += rng.normal(size=ch.dof) * jump * (rng.random(ch.dof) < 0.4)
    span = ch.q_hi - ch.q_lo
    q = np.clip(q, ch.q_lo + 0.05 * span, ch.q_hi - 0.05 * span)
    if limit_frac > 0:
        hit = rng.random(q.shape[:2]) < limit_frac
        j = rng.integers(0, ch.dof, size=q.shape[:2])
        side = rng.random(q.shape[:2]) < 0.5
        for k, i in zip(*np.nonzero(hit)):
            jj = j[k, i]
            marg = 0.01 if ch.joint_type[jj] == 1 else np.deg2rad(0.5)
            q[k, i, jj] = ch.q_lo[jj] + marg if side[k, i] else ch.q_hi[jj] - marg
    if quant:
        q = np.round(q / quant) * quant
        q = np.clip(q, np.ceil((ch.q_lo + 0.05 * span) / quant) * quant, np.floor((ch.q_hi - 0.05 * span) / quant) * quant)
    return q.astype(np.float32)
