"""fp64 CPU ORACLE of the global discrete search over K candidate trajectories (CppFlow, arxiv 2309.09102
sec. III-B; SURVEY.md section 8f NEXT-4 iii).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

"The module first creates a directed graph from the K motion plans.  Each IK solution is considered a node.  Edges
 are connected from each IK solution to the K IK solutions at the following time step.  A dynamic-programming-based
 search procedure is run on the graph.  The cost at each node is set to the minimum mjac achievable if the node is
 included in the returned path. ... an additional cost of 10 ... is added to configurations that are within
 1.5 degrees/3 cm of their joint limits.  An additional cost of 100 is added to configurations that would lead to a
 collision. ... Upon completion, a backtracking procedure is executed, which returns xi_search."
 mjac = max_i max_j |q_{i+1}[j] - q_i[j]|

Readings: S1 node cost  c[i][k] = pen[i][k] + min_k' max(c[i-1][k'], step(i-1,k' -> i,k)),
c[0][k] = pen[0][k], step = max_j |dq_j| (radians and metres in one max, as the paper's formula has it);
S2 ties go to the lowest candidate index (first minimum); S3 the path ends at argmin_k c[n-1][k] and is read back
through the stored predecessors; S4 "would lead to a collision" = smallest capsule clearance of the node < 0
(only with a capsule model).
"""
from __future__ import annotations

import itertools

import numpy as np


def penalties(q, q_lo, q_hi, joint_type, clearance=None, margin_rev=np.deg2rad(1.5), margin_pris=0.03):
    """q [K, n, d] -> pen [n, K]: +10 near a joint limit, +100 in collision."""
    marg = np.where(np.asarray(joint_type) == 1, margin_pris, margin_rev)
    near = ((q - q_lo[None, None, :] < marg) | (q_hi[None, None, :] - q < marg)).any(axis=2)   # [K, n]
    pen = 10.0 * near.T.astype(np.float64)
    if clearance is not None:
        pen = pen + 100.0 * (np.asarray(clearance).T < 0.0)
    return pen


def search(q, pen, dtype=np.float64, return_table=False):
    """q [K, n, d], pen [n, K] -> (choice [n] int, xi [n, d], cost, mjac of xi).  Plain DP, S1-S3.
    dtype: the precision every subtraction and addition is rounded to (max and < are exact).  The choice is an
    argmin decided by floating point, so the bit-for-bit parity test takes the decision in the kernel's precision
    (dtype=np.float32 on fp32 inputs).  The fp64 mode is pinned to brute force over all K^n paths; the fp32 mode is
    pinned to the fp64 mode (tests/test_oracle_search.py: cost within the rounding bound, identical choices on
    instances without near-ties), and the GPU's choice is ALSO judged by its fp64 path cost (path_cost below).
    return_table: also return the node costs c [n, K] and predecessors pred [n, K]."""
    q = np.asarray(q, dtype)
    pen = np.asarray(pen, dtype)
    K, n, d = q.shape
    c = np.empty((n, K), dtype)
    pred = np.zeros((n, K), np.int64)
    c[0] = pen[0]
    for i in range(1, n):
        for k in range(K):
            step = np.abs(q[k, i][None, :] - q[:, i - 1, :]).max(axis=1)   # [K]: from every node k' of timestep i-1
            v = np.maximum(c[i - 1], step)
            arg = int(np.argmin(v))                                        # first minimum (S2)
            c[i, k] = v[arg] + pen[i, k]
            pred[i, k] = arg
    choice = np.empty(n, np.int64)
    choice[n - 1] = int(np.argmin(c[n - 1]))
    for i in range(n - 1, 0, -1):
        choice[i - 1] = pred[i, choice[i]]
    xi = q[choice, np.arange(n)]
    mj = float(np.abs(np.diff(xi, axis=0)).max()) if n > 1 else 0.0
    if return_table:
        return choice, xi, float(c[n - 1, choice[n - 1]]), mj, c, pred
    return choice, xi, float(c[n - 1, choice[n - 1]]), mj


def path_cost(q, pen, choice):
    """S1 cost of ONE given path (choice [n]) in fp64, straight from the definition: the running maximum of the
    steps plus the penalties of the nodes it visits.  Judges a path without trusting whoever found it."""
    q = np.asarray(q, np.float64)
    pen = np.asarray(pen, np.float64)
    n = q.shape[1]
    c = pen[0, choice[0]]
    for i in range(1, n):
        c = max(c, np.abs(q[choice[i], i] - q[choice[i - 1], i - 1]).max()) + pen[i, choice[i]]
    return float(c)


def brute_force(q, pen):
    """Smallest S1 path cost over ALL K^n paths (tiny K, n only): the definition the DP must reproduce."""
    K, n, d = q.shape
    best = np.inf
    for path in itertools.product(range(K), repeat=n):
        c = pen[0, path[0]]
        for i in range(1, n):
            c = max(c, np.abs(q[path[i], i] - q[path[i - 1], i - 1]).max()) + pen[i, path[i]]
        best = min(best, c)
    return best
