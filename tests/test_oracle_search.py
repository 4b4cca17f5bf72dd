"""Pins of the search oracle (oracle/lm_search_oracle.py; NEXT-4 iii) -- CPU only."""
import numpy as np

from oracle import lm_search_oracle as sorc
from paper_2309_09102_b200 import workloads as wl


def test_dp_equals_brute_force_over_all_paths():
    rng = np.random.default_rng(0)
    for K, n in ((2, 6), (3, 5), (4, 4)):
        for trial in range(20):
            q = rng.normal(size=(K, n, 3)) * 0.3
            pen = 10.0 * (rng.random((n, K)) < 0.2) + 100.0 * (rng.random((n, K)) < 0.05)
            choice, xi, cost, mj = sorc.search(q, pen)
            assert np.isclose(cost, sorc.brute_force(q, pen), atol=1e-12)
            # the returned path really has that cost and xi is the selected configurations
            c = pen[0, choice[0]]
            for i in range(1, n):
                c = max(c, np.abs(q[choice[i], i] - q[choice[i - 1], i - 1]).max()) + pen[i, choice[i]]
            assert np.isclose(c, cost, atol=1e-12)
            assert np.array_equal(xi, q[choice, np.arange(n)])
            assert np.isclose(mj, np.abs(np.diff(xi, axis=0)).max())


def test_search_stitches_the_smooth_pieces_together():
    """Two candidates that are each smooth on one half and jump on the other: the search switches between them once and
    returns a path whose mjac is the small step, not the jump (the purpose of the module)."""
    n, d = 40, 7
    t = np.linspace(0, 1, n)[:, None]
    smooth = 0.5 * np.sin(2 * np.pi * t + np.arange(d)[None, :])
    a, b = smooth.copy(), smooth.copy() + 0.004          # b is a slightly shifted copy
    a[n // 2:] += 1.0                                      # a jumps in the middle
    b[:n // 2] -= 1.0                                      # b has its jump on the other side
    q = np.stack([a, b])
    choice, xi, cost, mj = sorc.search(q, np.zeros((n, 2)))
    assert np.all(choice[:n // 2] == 0) and np.all(choice[n // 2:] == 1)
    step = np.abs(np.diff(smooth, axis=0)).max()
    assert mj <= step + 0.0041 and cost == mj
    assert np.abs(np.diff(a, axis=0)).max() > 0.9 and np.abs(np.diff(b, axis=0)).max() > 0.9


def test_penalties_match_the_paper():
    ch = wl.random_chain_8dof(3)
    q = np.tile(0.5 * (ch.q_lo + ch.q_hi), (2, 3, 1))
    q[0, 1, 2] = ch.q_hi[2] - np.deg2rad(1.0)             # revolute joint within 1.5 deg of its limit
    q[1, 2, 0] = ch.q_lo[0] + 0.02                        # prismatic joint within 3 cm
    q[1, 0, 3] = ch.q_lo[3] + np.deg2rad(2.0)             # 2 deg away: fine
    pen = sorc.penalties(q, ch.q_lo, ch.q_hi, ch.joint_type)
    expect = np.zeros((3, 2))
    expect[1, 0] = 10.0
    expect[2, 1] = 10.0
    assert np.array_equal(pen, expect)
    clr = np.full((2, 3), 0.1)
    clr[0, 0] = -0.01
    assert np.array_equal(sorc.penalties(q, ch.q_lo, ch.q_hi, ch.joint_type, clr), expect + 100.0 * (clr.T < 0))
    # a penalised node is avoided whenever an unpenalised path exists (10 > the largest possible mjac of pi)
    rng = np.random.default_rng(1)
    qq = rng.uniform(-1, 1, size=(3, 8, 4))
    pen = np.zeros((8, 3))
    pen[3, 0] = pen[3, 1] = 10.0
    choice, _, cost, _ = sorc.search(qq, pen)
    assert choice[3] == 2 and cost < 10.0


def test_invariants_of_the_optimal_cost():
    """Properties any correct minimax path search has: relabelling the candidates leaves the cost unchanged, more
    candidates never make it worse, reversing time (no penalties) gives the same cost, and the cost is never below the
    largest layer-to-layer gap min_{k,k'} step (every path crosses every layer)."""
    rng = np.random.default_rng(3)
    for trial in range(10):
        K, n, d = 6, 30, 4
        q = np.cumsum(rng.normal(size=(K, n, d)) * 0.05, axis=1) + rng.normal(size=(K, 1, d)) * 0.2
        for k in range(K):
            i0 = int(rng.integers(1, n))
            q[k, i0:] += rng.normal(size=d) * 0.5
        pen = 10.0 * (rng.random((n, K)) < 0.1)
        c0 = sorc.search(q, pen)[2]
        perm = rng.permutation(K)
        assert np.isclose(sorc.search(q[perm], pen[:, perm])[2], c0, atol=1e-12)
        extra = np.concatenate([q, q[:2] + 0.01 * rng.normal(size=(2, n, d))])
        assert sorc.search(extra, np.concatenate([pen, pen[:, :2]], axis=1))[2] <= c0 + 1e-12
        zero = np.zeros((n, K))
        cz = sorc.search(q, zero)[2]
        assert np.isclose(sorc.search(q[:, ::-1], zero)[2], cz, atol=1e-12)
        gap = max(np.abs(q[:, None, i] - q[None, :, i - 1]).max(axis=2).min() for i in range(1, n))
        assert cz >= gap - 1e-12
        assert cz <= min(np.abs(np.diff(q[k], axis=0)).max() for k in range(K)) + 1e-12     # a single candidate is a path


def test_fp32_mode_rounds_like_the_kernel():
    """dtype=np.float32: every difference and sum is an fp32 operation (what the CUDA path does with __fsub_rn /
    __fadd_rn); on inputs that are exactly representable and whose differences are too, both modes agree exactly."""
    rng = np.random.default_rng(4)
    q = (rng.integers(-64, 64, size=(5, 12, 3)) / 32.0).astype(np.float32)      # multiples of 1/32: exact arithmetic
    pen = 10.0 * (rng.random((12, 5)) < 0.2)
    a = sorc.search(q, pen, dtype=np.float32)
    b = sorc.search(q.astype(np.float64), pen, dtype=np.float64)
    assert np.array_equal(a[0], b[0]) and a[2] == b[2] and a[3] == b[3]
    assert a[1].dtype == np.float32


# ---------------------------------------------------------------- pins of the fp32 mode where rounding matters
U32 = 2.0 ** -24  # unit roundoff of fp32


def rounding_bound(pen):
    """Relative error bound of any fp32 node cost against its fp64 value ("Precision"): the
    inputs are fp32, a step |q_a - q_b| is ONE rounded subtraction (relative error <= u), max and min keep a relative
    bound, adding a non-zero penalty rounds once more (adding 0 is exact) => (1 + u)^(1 + L) - 1 with L = number of
    layers that hold a penalised node.  1 % slack for the second-order terms."""
    L = int((np.asarray(pen) != 0).any(axis=1).sum())
    return 1.01 * (1 + L) * U32


def clear_cut(q, pen, c):
    """True if no comparison the DP makes is between two DIFFERENT fp64 values closer than twice the rounding bound:
    per layer the compared values are the previous node costs and the K x K steps, at the end the last node costs."""
    K, n, _ = q.shape
    tol = 2.0 * rounding_bound(pen)
    for i in range(1, n + 1):
        vals = [c[i - 1]]
        if i < n:
            vals.append(np.abs(q[:, None, i, :] - q[None, :, i - 1, :]).max(axis=2).ravel())
        v = np.unique(np.concatenate(vals))
        if v.size > 1 and np.min(np.diff(v) / v[1:]) <= tol:
            return False
    return True


def test_fp32_mode_against_the_fp64_mode_on_inputs_where_rounding_matters():
    """Random fp32 inputs whose differences are NOT representable: the fp32 mode's cost stays within the rounding bound
    of the (brute-force-pinned, here exact) fp64 optimum, the path it returns is optimal within twice that bound when
    its cost is re-evaluated in fp64 by the definition, and on instances without near-ties it is the SAME path."""
    rng = np.random.default_rng(5)
    same, total, inexact = 0, 0, 0
    for trial in range(60):
        K, n, d = int(rng.integers(2, 14)), int(rng.integers(2, 18)), int(rng.integers(1, 8))
        if trial % 2:   # smooth candidates: neighbouring values are within a factor 2, their difference is exact (Sterbenz)
            q = (np.cumsum(rng.normal(size=(K, n, d)) * 0.07, axis=1) + rng.normal(size=(K, 1, d)) * 0.2).astype(np.float32)
        else:           # unrelated values of either sign: the subtraction rounds
            q = (rng.normal(size=(K, n, d)) * 0.3).astype(np.float32)
        pen = 10.0 * (rng.random((n, K)) < 0.15) + 100.0 * (rng.random((n, K)) < 0.03)
        if trial % 3 == 0:
            pen[int(rng.integers(0, n))] += 10.0            # a layer nobody can avoid: the addition rounds
        q64 = q.astype(np.float64)
        ch64, _, c64, _, table, _ = sorc.search(q64, pen, dtype=np.float64, return_table=True)
        ch32, xi32, c32, mj32 = sorc.search(q, pen, dtype=np.float32)
        b = rounding_bound(pen)
        assert abs(c32 - c64) <= b * c64
        pc = sorc.path_cost(q64, pen, ch32)
        assert c64 <= pc <= c64 * (1 + 2 * b)
        assert abs(pc - c32) <= b * pc                      # the reported cost is the (rounded) cost of the reported path
        assert np.array_equal(xi32, q[ch32, np.arange(n)])
        inexact += int(float(c32) != float(c64))
        if clear_cut(q64, pen, table):
            total += 1
            same += int(np.array_equal(ch32, ch64))
    assert total >= 40 and same == total
    assert inexact >= 20                                    # rounding really was exercised


def test_fp32_mode_against_brute_force():
    """Tiny K^n cases with fp32 inputs: the fp64 cost of the fp32 mode's path is the brute-force optimum over all
    paths, within twice the rounding bound."""
    rng = np.random.default_rng(6)
    for K, n in ((2, 6), (3, 5), (4, 4)):
        for trial in range(15):
            q = (rng.normal(size=(K, n, 3)) * 0.3).astype(np.float32)
            pen = 10.0 * (rng.random((n, K)) < 0.2) + 100.0 * (rng.random((n, K)) < 0.05)
            ch32 = sorc.search(q, pen, dtype=np.float32)[0]
            best = sorc.brute_force(q.astype(np.float64), pen)
            pc = sorc.path_cost(q, pen, ch32)
            assert best <= pc <= best * (1 + 2 * rounding_bound(pen))


def test_path_cost_is_the_definition():
    """path_cost on a hand-made instance: steps 0.5, 0.25 and a penalised node."""
    q = np.zeros((2, 3, 1))
    q[0, :, 0] = [0.0, 0.5, 0.75]
    q[1, :, 0] = [1.0, 1.0, 1.0]
    pen = np.zeros((3, 2))
    pen[1, 0] = 10.0
    assert sorc.path_cost(q, pen, [0, 0, 0]) == 10.5      # max(0, .5) + 10, then max(10.5, .25)
    assert sorc.path_cost(q, pen, [1, 1, 1]) == 0.0
    assert sorc.path_cost(q, pen, [0, 1, 1]) == 1.0
    assert sorc.path_cost(q, pen, [1, 1, 0]) == 0.25
