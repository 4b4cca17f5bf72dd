"""GPU parity of the global discrete search (lm_search, NEXT-4 iii) against oracle/lm_search_oracle.py
(PAPER.md:L93-99).  Two checks on every case:

(1) VALIDITY, independent of the kernel's precision: the S1 cost of the GPU's path, re-evaluated in fp64 by the
    definition (sorc.path_cost), is the fp64 oracle's optimum (sorc.search in fp64: pinned to brute force over all
    K^n paths) within twice the rounding bound of DESIGN.md section 15 -- (1 + L) * 2^-24 relative, L = number of
    layers holding a penalised node; the reported cost and mjac are those of that path to one rounding.
(2) The choice is an argmin decided by floating point, so it is ALSO compared bit for bit (choice, xi, cost, mjac)
    with the oracle's fp32 mode (every subtraction / addition rounded to fp32; pinned against the fp64 mode on
    inputs where rounding matters, tests/test_oracle_search.py).

Inputs are the seeds (fp32), never anything read back from the GPU."""
import numpy as np
import pytest

from oracle import lm_coll_oracle as corc
from oracle import lm_oracle as orc
from oracle import lm_search_oracle as sorc
from paper_2309_09102_b200 import workloads as wl

pytestmark = pytest.mark.gpu


candidates = wl.search_candidates


def make_solver(ch, q32, **kw):
    from paper_2309_09102_b200 import lm
    K, n, d = q32.shape
    p, R = orc.fk(ch, q32[0].astype(np.float64))
    tp = np.tile(p.astype(np.float32), (K, 1))
    tq = np.tile(wl._R_to_quat_wxyz(R).astype(np.float32), (K, 1))
    return lm.Solver(ch, K, n, tp, tq, q32.reshape(K * n, d), **kw)


def check(ch, q32, clearance=None, solver=None, sparams=None):
    from paper_2309_09102_b200 import lm
    s = solver if solver is not None else make_solver(ch, q32)
    g = s.search(sparams)
    assert np.array_equal(s.fetch()["q"].reshape(q32.shape), q32)      # the search ran on exactly the seeds
    if solver is None:
        s.close()
    pen = sorc.penalties(q32, ch.q_lo.astype(np.float32), ch.q_hi.astype(np.float32), ch.joint_type, clearance,
                         margin_rev=np.float32(np.deg2rad(1.5)), margin_pris=np.float32(0.03))
    choice, xi, cost, mj = sorc.search(q32, pen, dtype=np.float32)
    assert np.array_equal(g["choice"], choice)
    assert np.array_equal(g["xi"], xi)
    assert np.float32(g["cost"]) == np.float32(cost)
    assert np.float32(g["mjac"]) == np.float32(mj)
    validity(q32, pen, g)
    return g, pen


U32 = 2.0 ** -24


def validity(q32, pen, g):
    """The fp64 path cost of the GPU's choice against the fp64 optimum (no fp32 oracle mode involved).  The penalty
    table is an integer-valued INPUT of the DP (decided once, in fp32, by both sides)."""
    K, n, d = q32.shape
    q64, pen64 = q32.astype(np.float64), pen.astype(np.float64)
    best = sorc.search(q64, pen64, dtype=np.float64)[2]
    bound = 1.01 * (1 + int((pen64 != 0).any(axis=1).sum())) * U32
    choice = np.asarray(g["choice"])
    assert choice.shape == (n,) and choice.min() >= 0 and choice.max() < K
    pc = sorc.path_cost(q64, pen64, choice)
    assert best <= pc <= best * (1 + 2 * bound), (best, pc)
    assert abs(float(g["cost"]) - pc) <= bound * pc
    xi64 = q64[choice, np.arange(n)]
    assert np.array_equal(g["xi"].astype(np.float64), xi64)
    mj = np.abs(np.diff(xi64, axis=0)).max() if n > 1 else 0.0
    assert abs(float(g["mjac"]) - mj) <= U32 * mj


def test_search_matches_the_oracle_panda():
    ch = wl.panda_chain()
    q = candidates(ch, 24, 60, 1)
    g, pen = check(ch, q)
    assert len(set(g["choice"].tolist())) > 1                       # the path really switches candidates
    single = min(np.abs(np.diff(q[k].astype(np.float64), axis=0)).max() for k in range(24))
    assert g["mjac"] < 0.5 * single                                 # much smoother than the best single candidate


def test_search_paper_size_175_candidates_300_waypoints():
    ch = wl.panda_chain()
    q = candidates(ch, 175, 300, 2, limit_frac=0.02)
    g, pen = check(ch, q)
    assert pen.max() == 10.0 and g["cost"] < 10.0                   # penalised nodes exist and are all avoided


def test_search_ties_go_to_the_lowest_candidate():
    ch = wl.panda_chain()
    q = candidates(ch, 40, 50, 3, quant=0.125)                      # steps are multiples of 1/8: many exact ties
    q[7] = q[3]                                                     # two identical candidates
    g, _ = check(ch, q)
    assert 7 not in g["choice"]


def test_search_prismatic_margins_and_unavoidable_penalties():
    ch = wl.random_chain_8dof(3)
    q = candidates(ch, 33, 45, 4, limit_frac=0.3)
    q[:, 20, 1] = np.float32(ch.q_hi[1]) - np.float32(0.001)        # every node of timestep 20 is near a limit
    g, pen = check(ch, q)
    assert (pen[20] == 10.0).all() and 10.0 <= g["cost"] < 20.0


def test_search_shapes():
    ch = wl.panda_chain()
    for K, n, seed in ((1, 1, 5), (1, 40, 6), (5, 1, 7), (3, 2, 8), (257, 9, 9), (1024, 5, 10), (600, 220, 11)):
        check(ch, candidates(ch, K, n, seed))                       # (600, 220): predecessors do not fit in shared memory


def test_search_collision_penalty():
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    caps, scene = wl.panda_capsules(), wl.panda_scene()
    K, n = 30, 40
    q = candidates(ch, K, n, 12)
    ocaps = corc.Capsules(caps, w_coll=1.0, d_safe=0.05, scene=scene, w_env=1.0, d_safe_env=0.05)
    clr = np.array([[corc.residual(ch, ocaps, q[k, i].astype(np.float64))[0].min() for i in range(n)] for k in range(K)])
    assert (clr < 0).any() and (clr > 0).any() and np.abs(clr).min() > 1e-5
    s = make_solver(ch, q)
    s.traj_attach(lm.lm_traj_default_params())
    s.traj_set_capsules(caps, 1.0, 0.05)
    s.traj_set_obstacles(scene, 1.0, 0.05)
    check(ch, q, clearance=clr, solver=s, sparams=lm.lm_search_default_params(use_clearance=1))
    s.close()


def test_search_rejects_bad_arguments():
    from paper_2309_09102_b200 import lm
    ch = wl.panda_chain()
    s = make_solver(ch, candidates(ch, 4, 6, 13))
    with pytest.raises(lm.LmError):
        s.search(lm.lm_search_default_params(use_clearance=1))      # no capsule model
    with pytest.raises(lm.LmError):
        s.search(lm.lm_search_default_params(margin_rev=-1.0))
    nbytes = lm.lm_search_workspace_bytes(7, 4, 6)
    ptr = (s.search_workspace.data_ptr() + 255) // 256 * 256 if getattr(s, "search_workspace", None) is not None else 256
    with pytest.raises(lm.LmError):
        lm.lm_search(s._ctx, lm.lm_search_default_params(), ptr + 4, nbytes, None, None, None)
    s.close()
    assert lm.lm_search_workspace_bytes(7, 1025, 10) == 0 and lm.lm_search_workspace_bytes(9, 10, 10) == 0


def test_search_random_shapes():
    """Twelve seeded (K, n) pairs on both chains, with near-limit nodes and (every fourth) quantised inputs: the GPU's
    choice / xi / cost / mjac stay bit-identical to the fp32 oracle whatever the cluster slicing (KC, G, padding)."""
    chains = (wl.panda_chain(), wl.random_chain_8dof(3))
    for seed in range(100, 112):
        rng = np.random.default_rng(seed)
        K, n = int(rng.integers(1, 200)), int(rng.integers(1, 120))
        ch = chains[seed % 2]
        check(ch, candidates(ch, K, n, seed, limit_frac=0.05 * (seed % 3), quant=(0.125 if seed % 4 == 0 else None)))
