"""Pins of the collision oracle (oracle/lm_coll_oracle.c; NEXT-3) -- CPU only."""
import numpy as np
import pytest

from oracle import lm_coll_oracle as corc
from oracle import lm_oracle as orc
from oracle import lm_traj_oracle as torc
from paper_2309_09102_b200 import workloads as wl


def brute(a1, b1, a2, b2, m=401):
    t = np.linspace(0, 1, m)
    P1 = a1[None] + (b1 - a1)[None] * t[:, None]
    P2 = a2[None] + (b2 - a2)[None] * t[:, None]
    return np.sqrt(((P1[:, None, :] - P2[None, :, :]) ** 2).sum(-1)).min()


def test_segment_distance_is_the_qp_minimum():
    rng = np.random.default_rng(0)
    for k in range(300):
        a1, b1, a2, b2 = rng.normal(size=(4, 3))
        if k % 5 == 1:
            b2 = a2 + (b1 - a1) * rng.uniform(-2, 2)          # parallel
        if k % 7 == 2:
            b1 = a1.copy()                                    # a point
        if k % 11 == 3:
            a2 = a1 + 0.5 * (b1 - a1)                          # touching
        d, t1, t2 = corc.segment_distance(a1, b1, a2, b2)
        assert 0 <= t1 <= 1 and 0 <= t2 <= 1
        p = (a1 + (b1 - a1) * t1) - (a2 + (b2 - a2) * t2)
        assert np.isclose(np.linalg.norm(p), d, atol=1e-12)   # the reported minimiser attains it
        g = brute(a1, b1, a2, b2)
        assert d <= g + 1e-12                                  # no grid point is better
        assert g - d <= (np.linalg.norm(b1 - a1) + np.linalg.norm(b2 - a2)) / 400 + 1e-12


def test_segment_distance_closed_forms():
    # skew perpendicular segments crossing at height h
    d, t1, t2 = corc.segment_distance([-1, 0, 0], [1, 0, 0], [0, -1, 0.3], [0, 1, 0.3])
    assert np.isclose(d, 0.3) and np.isclose(t1, 0.5) and np.isclose(t2, 0.5)
    # parallel, overlapping in projection
    d, _, _ = corc.segment_distance([0, 0, 0], [1, 0, 0], [0.2, 0.4, 0], [0.9, 0.4, 0])
    assert np.isclose(d, 0.4)
    # collinear, apart: endpoint to endpoint
    d, t1, t2 = corc.segment_distance([0, 0, 0], [1, 0, 0], [1.5, 0, 0], [3, 0, 0])
    assert np.isclose(d, 0.5) and t1 == 1.0 and t2 == 0.0
    # endpoint of one against the interior of the other
    d, t1, t2 = corc.segment_distance([0, 0, 0], [2, 0, 0], [0.5, 1, 0], [0.5, 3, 0])
    assert np.isclose(d, 1.0) and np.isclose(t1, 0.25) and t2 == 0.0
    # intersecting
    d, _, _ = corc.segment_distance([-1, -1, 0], [1, 1, 0], [-1, 1, 0], [1, -1, 0])
    assert d < 1e-12


@pytest.mark.parametrize("ch", [wl.panda_chain(), wl.random_chain_8dof(3)], ids=lambda c: c.name)
def test_capsule_endpoints_ride_on_their_links(ch):
    """World endpoint of a capsule on link L = flange position of the chain truncated after joint L with
    the endpoint as tool offset (orc.fk is pinned in test_oracle_pins.py); base capsules do not move."""
    model = wl.chain_capsules(ch) if ch.dof == 8 else wl.panda_capsules()
    caps = corc.Capsules(model)
    rng = np.random.default_rng(1)
    q = 0.5 * (ch.q_lo + ch.q_hi) + 0.3 * (ch.q_hi - ch.q_lo) * rng.uniform(-1, 1, ch.dof)
    wa, wb = corc.capsule_world(ch, caps, q)
    for k in range(len(model.link)):
        L = int(model.link[k])
        if L < 0:
            assert np.array_equal(wa[k], model.a[k]) and np.array_equal(wb[k], model.b[k])
            continue
        for end, w in ((model.a[k], wa[k]), (model.b[k], wb[k])):
            sub = wl.Chain("sub", L + 1, ch.joint_type[:L + 1], ch.a[:L + 1], ch.alpha[:L + 1], ch.d[:L + 1],
                           ch.theta[:L + 1], ch.q_lo[:L + 1], ch.q_hi[:L + 1], np.r_[end, 1, 0, 0, 0])
            p, _ = orc.fk(sub, q[:L + 1])
            assert np.abs(p - w).max() < 1e-12


def folded_panda(rng, spread=0.15):
    """Configurations in which the hand comes back towards the base / shoulder (several pairs within 0.3 m)."""
    q = np.array([0.0, 1.2, 0.0, -2.9, 0.0, 2.2, 0.8]) + spread * rng.normal(size=7)
    ch = wl.panda_chain()
    return np.clip(q, ch.q_lo, ch.q_hi)


def test_hinge_residual_and_its_jacobian():
    ch = wl.panda_chain()
    model = wl.panda_capsules()
    rng = np.random.default_rng(2)
    checked = 0
    for trial in range(40):
        q = folded_panda(rng)
        caps = corc.Capsules(model, w_coll=1.7, d_safe=0.30)
        dist, r = corc.residual(ch, caps, q)
        wa, wb = corc.capsule_world(ch, caps, q)
        for p, (k1, k2) in enumerate(model.pairs):
            d, _, _ = corc.segment_distance(wa[k1], wb[k1], wa[k2], wb[k2])
            assert np.isclose(dist[p], d - model.radius[k1] - model.radius[k2], atol=1e-14)       # C3
            assert np.isclose(r[p], 1.7 * max(0.0, 0.30 - dist[p]), atol=1e-14)                    # C4
        J = corc.jacobian(ch, caps, q)
        assert np.all(J[r == 0.0] == 0.0)
        h = 1e-6
        Jfd = np.zeros_like(J)
        kink = np.zeros(len(r), bool)
        for j in range(7):
            e = np.zeros(7)
            e[j] = h
            dp, rp = corc.residual(ch, caps, q + e)
            dm, rm = corc.residual(ch, caps, q - e)
            Jfd[:, j] = (rp - rm) / (2 * h)
            kink |= (rp == 0) != (rm == 0)
        act = (r > 1e-3) & ~kink
        if act.any():
            assert np.abs(J[act] - Jfd[act]).max() < 2e-6, np.abs(J[act] - Jfd[act]).max()     # C5
            checked += int(act.sum())
    assert checked > 60


def test_trajectory_step_with_collision_rows():
    """The collision rows enter the stacked system like any other row: delta is still the damped least-squares
    solution (numpy lstsq on the oracle's own J, pinned above and in test_oracle_traj.py), dense = banded, and
    a few LM iterations push the closest pairs apart."""
    ch = wl.panda_chain()
    model = wl.panda_capsules()
    rng = np.random.default_rng(3)
    n = 8
    q0 = np.stack([folded_panda(rng, 0.05) for _ in range(n)])
    q0 = np.cumsum(np.r_[q0[:1], 0.01 * rng.normal(size=(n - 1, 7))], axis=0)
    q0 = np.clip(q0, ch.q_lo, ch.q_hi)
    p, R = orc.fk(ch, q0)
    tp, tq = p, wl._R_to_quat_wxyz(R)
    caps = corc.Capsules(model, w_coll=2.0, d_safe=0.25)
    pp = orc.Params()
    tprm = torc.TrajParams(w_pose=0.5, w_diff=0.3, caps=caps)
    assert torc.rows(7, n, tprm) == 6 * n + 7 * (n - 1) + len(model.pairs) * n
    r = torc.residual(ch, pp, tprm, tp, tq, q0)
    J = torc.jacobian(ch, pp, tprm, q0)
    assert (r[-len(model.pairs) * n:] > 0).sum() >= n          # hinges are active
    for lam in (1e-3, 1e-1):
        x = np.linalg.lstsq(np.vstack([J, np.sqrt(lam) * np.eye(7 * n)]), -np.r_[r, np.zeros(7 * n)], rcond=None)[0]
        dd = torc.delta(ch, pp, tprm, tp, tq, q0, lam, dense=True)
        db = torc.delta(ch, pp, tprm, tp, tq, q0, lam, dense=False)
        assert np.abs(dd.ravel() - x).max() < 1e-8 and np.abs(db - dd).max() < 1e-10
    # without the rows the step is different (they matter) ...
    d0 = torc.delta(ch, pp, torc.TrajParams(w_pose=0.5, w_diff=0.3), tp, tq, q0, 1e-3)
    assert np.abs(d0 - db).max() > 1e-3
    # ... and LM with them increases the smallest clearance while the cost goes down
    st = torc.lm_run(ch, pp, tprm, tp[None], tq[None], q0[None], 6)
    d_before = min(corc.residual(ch, caps, q0[i])[0].min() for i in range(n))
    d_after = min(corc.residual(ch, caps, st.q[0, i])[0].min() for i in range(n))
    assert d_after > d_before + 0.01
    assert st.F_total[0] < (r @ r) * 0.8
    assert np.isclose(st.F_total[0], np.sum(torc.residual(ch, pp, tprm, tp, tq, st.q[0]) ** 2), rtol=1e-12)


# ------------------------------------------------------------------ robot-environment rows

def brute_box(a, b, pmin, pmax, m=4001):
    t = np.linspace(0, 1, m)
    x = a[None] + (b - a)[None] * t[:, None]
    return np.sqrt(((x - np.clip(x, pmin, pmax)) ** 2).sum(-1)).min()


def test_segment_box_distance_is_the_qp_minimum():
    rng = np.random.default_rng(5)
    for k in range(400):
        half = rng.uniform(0.05, 0.5, size=3)
        a, b = rng.normal(size=(2, 3)) * rng.uniform(0.2, 1.5)
        if k % 4 == 1:
            b[rng.integers(3)] = a[rng.integers(3)]            # (partly) axis-parallel
        if k % 9 == 2:
            b = a.copy()
        d, t, p = corc.segment_box_distance(a, b, -half, half)
        assert 0 <= t <= 1 and np.all(p >= -half - 1e-15) and np.all(p <= half + 1e-15)
        x = a + (b - a) * t
        assert np.isclose(np.linalg.norm(x - p), d, atol=1e-12)                 # the minimiser attains it
        g = brute_box(a, b, -half, half)
        assert d <= g + 1e-12 and g - d <= np.linalg.norm(b - a) / 4000 + 1e-12
    # closed forms: above a face, beside an edge, beyond a corner, passing through
    assert np.isclose(corc.segment_box_distance([-1, 0, 0.7], [1, 0, 0.7], [-0.5] * 3, [0.5] * 3)[0], 0.2)
    assert np.isclose(corc.segment_box_distance([1, 1, -2], [1, 1, 2], [-0.5] * 3, [0.5] * 3)[0], np.sqrt(0.5))
    assert np.isclose(corc.segment_box_distance([1, 1, 1], [2, 2, 2], [-0.5] * 3, [0.5] * 3)[0], np.sqrt(0.75))
    assert corc.segment_box_distance([-1, 0.1, 0], [1, 0.2, 0.1], [-0.5] * 3, [0.5] * 3)[0] < 1e-15


def test_environment_rows_value_and_jacobian():
    ch, model, scene = wl.panda_chain(), wl.panda_capsules(), wl.panda_scene()
    rng = np.random.default_rng(6)
    caps = corc.Capsules(model, w_coll=0.0, scene=scene, w_env=1.3, d_safe_env=0.6)
    checked = 0
    for trial in range(30):
        q = np.clip(0.5 * (ch.q_lo + ch.q_hi) + 0.5 * rng.normal(size=7), ch.q_lo, ch.q_hi)
        dist, r = corc.residual(ch, caps, q)
        assert dist.shape == (len(scene.pairs),)
        wa, wb = corc.capsule_world(ch, caps, q)
        for p, (k, o) in enumerate(scene.pairs):
            ab = scene.R[o].T @ (wa[k] - scene.t[o])
            bb = scene.R[o].T @ (wb[k] - scene.t[o])
            d = corc.segment_box_distance(ab, bb, scene.pmin[o], scene.pmax[o])[0] - model.radius[k]
            assert np.isclose(dist[p], d, atol=1e-13)
            assert np.isclose(r[p], 1.3 * max(0.0, 0.6 - d), atol=1e-13)
        J = corc.jacobian(ch, caps, q)
        h = 1e-6
        Jfd = np.zeros_like(J)
        kink = np.zeros(len(r), bool)
        for j in range(7):
            e = np.zeros(7)
            e[j] = h
            dp, rp = corc.residual(ch, caps, q + e)
            dm, rm = corc.residual(ch, caps, q - e)
            Jfd[:, j] = (rp - rm) / (2 * h)
            kink |= (rp == 0) != (rm == 0)
        act = (r > 1e-3) & ~kink & (dist + model.radius[scene.pairs[:, 0]] > 1e-3)     # not penetrating the box itself
        if act.any():
            assert np.abs(J[act] - Jfd[act]).max() < 5e-6, np.abs(J[act] - Jfd[act]).max()
            checked += int(act.sum())
    assert checked > 100
    # both kinds of rows together: self rows first, then environment rows
    both = corc.Capsules(model, w_coll=1.0, d_safe=0.3, scene=scene, w_env=1.3, d_safe_env=0.6)
    q = np.array([0.0, 1.2, 0.0, -2.9, 0.0, 2.2, 0.8])
    d_all, r_all = corc.residual(ch, both, q)
    d_s, r_s = corc.residual(ch, corc.Capsules(model, w_coll=1.0, d_safe=0.3), q)
    d_e, r_e = corc.residual(ch, caps, q)
    assert np.array_equal(r_all, np.r_[r_s, r_e]) and np.array_equal(d_all, np.r_[d_s, d_e])
    assert np.array_equal(corc.jacobian(ch, both, q), np.vstack([corc.jacobian(ch, corc.Capsules(model, w_coll=1.0, d_safe=0.3), q),
                                                                 corc.jacobian(ch, caps, q)]))


def test_trajectory_step_with_environment_rows():
    ch, model, scene = wl.panda_chain(), wl.panda_capsules(), wl.panda_scene()
    rng = np.random.default_rng(7)
    n = 6
    q0 = np.clip(0.5 * (ch.q_lo + ch.q_hi) + np.cumsum(0.02 * rng.normal(size=(n, 7)), axis=0), ch.q_lo, ch.q_hi)
    p, R = orc.fk(ch, q0)
    tp, tq = p, wl._R_to_quat_wxyz(R)
    caps = corc.Capsules(model, w_coll=1.0, d_safe=0.2, scene=scene, w_env=1.5, d_safe_env=0.5)
    tprm = torc.TrajParams(w_pose=0.5, w_diff=0.3, caps=caps)
    rows = 6 * n + 7 * (n - 1) + (len(model.pairs) + len(scene.pairs)) * n
    r = torc.residual(ch, orc.Params(), tprm, tp, tq, q0)
    J = torc.jacobian(ch, orc.Params(), tprm, q0)
    assert r.shape == (rows,) and J.shape == (rows, 7 * n) and (r[-len(scene.pairs):] > 0).any()
    lam = 1e-2
    x = np.linalg.lstsq(np.vstack([J, np.sqrt(lam) * np.eye(7 * n)]), -np.r_[r, np.zeros(7 * n)], rcond=None)[0]
    dd = torc.delta(ch, orc.Params(), tprm, tp, tq, q0, lam, dense=True)
    db = torc.delta(ch, orc.Params(), tprm, tp, tq, q0, lam, dense=False)
    assert np.abs(dd.ravel() - x).max() < 1e-8 and np.abs(db - dd).max() < 1e-10
