/*
 * lm_coll_oracle.c -- fp64 CPU ORACLE of the capsule-capsule collision residual (test infrastructure,
 * see lm_coll_oracle.h).  Plain loops; the QP is solved by enumerating the active sets of its box.
 */
#include "lm_coll_oracle.h"

#include <math.h>
#include <string.h>

static double dot3(const double *x, const double *y) { return x[0] * y[0] + x[1] * y[1] + x[2] * y[2]; }

static double seg_cost(const double *a1, const double *d1, const double *a2, const double *d2, double t1, double t2) {
    double s = 0.0;
    for (int i = 0; i < 3; ++i) {
        const double e = (a1[i] + d1[i] * t1) - (a2[i] + d2[i] * t2);
        s += e * e;
    }
    return s;
}

static double clamp01(double x) { return x < 0.0 ? 0.0 : (x > 1.0 ? 1.0 : x); }

double orc_segment_distance(const double *a1, const double *b1, const double *a2, const double *b2,
                            double *t1, double *t2) {
    /* cost(t1, t2) = |r + d1 t1 - d2 t2|^2, r = a1 - a2: a convex quadratic on the unit box.
     * Candidates: the unconstrained stationary point (if inside), the minimiser along each of the four
     * edges (clamped to the edge), which also covers the four corners.  The smallest cost wins. */
    double d1[3], d2[3], r[3];
    for (int i = 0; i < 3; ++i) { d1[i] = b1[i] - a1[i]; d2[i] = b2[i] - a2[i]; r[i] = a1[i] - a2[i]; }
    const double A = dot3(d1, d1), B = dot3(d1, d2), E = dot3(d2, d2), C = dot3(d1, r), F = dot3(d2, r);
    double best = INFINITY, bt1 = 0.0, bt2 = 0.0;
    /* interior: [A -B; -B E] [t1; t2] = [-C; F] */
    const double det = A * E - B * B;
    if (det > 1e-14 * (A * E + 1e-300)) {
        const double s1 = (-C * E + B * F) / det, s2 = (A * F - B * C) / det;
        if (s1 >= 0.0 && s1 <= 1.0 && s2 >= 0.0 && s2 <= 1.0) {
            best = seg_cost(a1, d1, a2, d2, s1, s2); bt1 = s1; bt2 = s2;
        }
    }
    /* edges t1 = 0 and t1 = 1: minimise over t2; edges t2 = 0 and t2 = 1: minimise over t1 */
    for (int e = 0; e < 4; ++e) {
        double s1, s2;
        if (e < 2) {
            s1 = (double)e;
            s2 = E > 0.0 ? clamp01((F + B * s1) / E) : 0.0;
        } else {
            s2 = (double)(e - 2);
            s1 = A > 0.0 ? clamp01((B * s2 - C) / A) : 0.0;
        }
        const double cst = seg_cost(a1, d1, a2, d2, s1, s2);
        if (cst < best) { best = cst; bt1 = s1; bt2 = s2; }
    }
    if (t1) *t1 = bt1;
    if (t2) *t2 = bt2;
    return sqrt(best);
}

static double box_cost(const double *a, const double *d, const double *pmin, const double *pmax, double t, double *p) {
    double s = 0.0;
    for (int i = 0; i < 3; ++i) {
        const double x = a[i] + d[i] * t;
        const double c = x < pmin[i] ? pmin[i] : (x > pmax[i] ? pmax[i] : x);
        if (p) p[i] = c;
        s += (x - c) * (x - c);
    }
    return s;
}

double orc_segment_box_distance(const double *a, const double *b, const double *pmin, const double *pmax,
                                double *t_out, double *p_out) {
    double d[3], bp[8];
    int nb = 0;
    bp[nb++] = 0.0;
    for (int i = 0; i < 3; ++i) {
        d[i] = b[i] - a[i];
        if (d[i] != 0.0) {
            const double t1 = (pmin[i] - a[i]) / d[i], t2 = (pmax[i] - a[i]) / d[i];
            if (t1 > 0.0 && t1 < 1.0) bp[nb++] = t1;
            if (t2 > 0.0 && t2 < 1.0) bp[nb++] = t2;
        }
    }
    bp[nb++] = 1.0;
    for (int i = 1; i < nb; ++i) /* insertion sort of the breakpoints */
        for (int j = i; j > 0 && bp[j] < bp[j - 1]; --j) { const double tmp = bp[j]; bp[j] = bp[j - 1]; bp[j - 1] = tmp; }
    double best = INFINITY, bt = 0.0;
    for (int k = 0; k + 1 < nb; ++k) {
        const double lo = bp[k], hi = bp[k + 1], mid = 0.5 * (lo + hi);
        /* on [lo, hi] every coordinate stays on one side of each face: cost = sum over the outside axes of
         * (a_i + d_i t - bound_i)^2, a quadratic in t */
        double num = 0.0, den = 0.0;
        for (int i = 0; i < 3; ++i) {
            const double x = a[i] + d[i] * mid;
            double bound;
            if (x < pmin[i]) bound = pmin[i]; else if (x > pmax[i]) bound = pmax[i]; else continue;
            num += d[i] * (a[i] - bound);
            den += d[i] * d[i];
        }
        double ts = den > 0.0 ? -num / den : lo;
        if (ts < lo) ts = lo;
        if (ts > hi) ts = hi;
        const double cand[3] = {ts, lo, hi};
        for (int c = 0; c < 3; ++c) {
            const double v = box_cost(a, d, pmin, pmax, cand[c], NULL);
            if (v < best) { best = v; bt = cand[c]; }
        }
    }
    if (nb == 2 && best == INFINITY) { best = box_cost(a, d, pmin, pmax, 0.0, NULL); bt = 0.0; }
    box_cost(a, d, pmin, pmax, bt, p_out);
    if (t_out) *t_out = bt;
    return sqrt(best);
}

/* frame of link L: identity for L = -1 */
static void link_frame(int d, const double *Rj, const double *oj, int L, double *R, double *o) {
    (void)d;
    if (L < 0) {
        for (int i = 0; i < 9; ++i) R[i] = (i % 4 == 0) ? 1.0 : 0.0;
        o[0] = o[1] = o[2] = 0.0;
    } else {
        memcpy(R, Rj + 9 * L, 9 * sizeof(double));
        memcpy(o, oj + 3 * L, 3 * sizeof(double));
    }
}

void orc_capsule_world(const orc_chain *c, const orc_capsules *m, const double *q, double *wa, double *wb) {
    double Rj[9 * ORC_MAX_DOF], oj[3 * ORC_MAX_DOF];
    orc_fk_frames(c, q, Rj, oj);
    for (int k = 0; k < m->ncaps; ++k) {
        double R[9], o[3];
        link_frame(c->dof, Rj, oj, m->link[k], R, o);
        for (int i = 0; i < 3; ++i) {
            wa[3 * k + i] = o[i] + R[3 * i] * m->a[k][0] + R[3 * i + 1] * m->a[k][1] + R[3 * i + 2] * m->a[k][2];
            wb[3 * k + i] = o[i] + R[3 * i] * m->b[k][0] + R[3 * i + 1] * m->b[k][1] + R[3 * i + 2] * m->b[k][2];
        }
    }
}

int orc_coll_rows(const orc_capsules *m) {
    return (m->w_coll != 0.0 ? m->npairs : 0) + (m->w_env != 0.0 ? m->nenv : 0);
}

/* world point -> frame of obstacle o:  x_box = Ro^T (x - to) */
static void to_box(const orc_capsules *m, int o, const double *x, double *y) {
    for (int i = 0; i < 3; ++i) {
        y[i] = 0.0;
        for (int k = 0; k < 3; ++k) y[i] += m->Ro[o][3 * k + i] * (x[k] - m->to[o][k]);
    }
}

void orc_coll_residual(const orc_chain *c, const orc_capsules *m, const double *q, double *dist, double *r) {
    double wa[3 * ORC_MAX_CAPS], wb[3 * ORC_MAX_CAPS];
    orc_capsule_world(c, m, q, wa, wb);
    const int ns = m->w_coll != 0.0 ? m->npairs : 0;
    for (int p = 0; p < (m->w_env != 0.0 ? m->nenv : 0); ++p) { /* robot-environment rows */
        const int k = m->env_pair[p][0], o = m->env_pair[p][1];
        double ab[3], bb[3];
        to_box(m, o, wa + 3 * k, ab);
        to_box(m, o, wb + 3 * k, bb);
        const double dd = orc_segment_box_distance(ab, bb, m->pmin[o], m->pmax[o], NULL, NULL) - m->c[k];
        if (dist) dist[ns + p] = dd;
        if (r) r[ns + p] = m->w_env * (dd < m->d_safe_env ? m->d_safe_env - dd : 0.0);
    }
    if (ns == 0) return;
    for (int p = 0; p < m->npairs; ++p) {
        const int k1 = m->pair[p][0], k2 = m->pair[p][1];
        const double dd = orc_segment_distance(wa + 3 * k1, wb + 3 * k1, wa + 3 * k2, wb + 3 * k2, NULL, NULL)
                          - m->c[k1] - m->c[k2];                          /* C3 */
        if (dist) dist[p] = dd;
        if (r) r[p] = m->w_coll * (dd < m->d_safe ? m->d_safe - dd : 0.0); /* C4 */
    }
}

/* column j of the Jacobian of a point p rigidly attached to link L: z_j x (p - o_j) (revolute) or z_j
 * (prismatic) for j <= L, zero for the joints beyond the link */
static void point_jacobian_col(const orc_chain *c, const double *z, const double *o, int L, int j, const double *p, double *col) {
    col[0] = col[1] = col[2] = 0.0;
    if (j > L) return;
    const double *zj = z + 3 * j, *oj = o + 3 * j;
    if (c->joint_type[j] == 0) {
        const double e[3] = {p[0] - oj[0], p[1] - oj[1], p[2] - oj[2]};
        col[0] = zj[1] * e[2] - zj[2] * e[1];
        col[1] = zj[2] * e[0] - zj[0] * e[2];
        col[2] = zj[0] * e[1] - zj[1] * e[0];
    } else {
        col[0] = zj[0]; col[1] = zj[1]; col[2] = zj[2];
    }
}

void orc_coll_jacobian(const orc_chain *c, const orc_capsules *m, const double *q, double *J) {
    const int d = c->dof;
    double wa[3 * ORC_MAX_CAPS], wb[3 * ORC_MAX_CAPS], pe[3], Re[9], z[3 * ORC_MAX_DOF], o[3 * ORC_MAX_DOF];
    orc_capsule_world(c, m, q, wa, wb);
    orc_fk(c, q, pe, Re, z, o);
    memset(J, 0, sizeof(double) * (size_t)(orc_coll_rows(m) * d));
    const int ns = m->w_coll != 0.0 ? m->npairs : 0;
    for (int p = 0; p < (m->w_env != 0.0 ? m->nenv : 0); ++p) { /* environment rows: the obstacle does not move */
        const int k = m->env_pair[p][0], ob = m->env_pair[p][1];
        double ab[3], bb[3], t, pb[3];
        to_box(m, ob, wa + 3 * k, ab);
        to_box(m, ob, wb + 3 * k, bb);
        const double len = orc_segment_box_distance(ab, bb, m->pmin[ob], m->pmax[ob], &t, pb);
        const double dd = len - m->c[k];
        if (!(dd < m->d_safe_env) || !(len > 0.0)) continue;
        double ps[3], nb[3], n[3];
        for (int i = 0; i < 3; ++i) {
            ps[i] = wa[3 * k + i] + (wb[3 * k + i] - wa[3 * k + i]) * t;      /* closest point on the capsule axis, world */
            nb[i] = ((ab[i] + (bb[i] - ab[i]) * t) - pb[i]) / len;             /* direction box point -> axis point, box frame */
        }
        for (int i = 0; i < 3; ++i) n[i] = m->Ro[ob][3 * i] * nb[0] + m->Ro[ob][3 * i + 1] * nb[1] + m->Ro[ob][3 * i + 2] * nb[2];
        for (int j = 0; j < d; ++j) {
            double c1[3];
            point_jacobian_col(c, z, o, m->link[k], j, ps, c1);
            J[(ns + p) * d + j] = -m->w_env * (n[0] * c1[0] + n[1] * c1[1] + n[2] * c1[2]);
        }
    }
    for (int p = 0; p < ns; ++p) {
        const int k1 = m->pair[p][0], k2 = m->pair[p][1];
        double t1, t2;
        const double len = orc_segment_distance(wa + 3 * k1, wb + 3 * k1, wa + 3 * k2, wb + 3 * k2, &t1, &t2);
        const double dd = len - m->c[k1] - m->c[k2];
        if (!(dd < m->d_safe) || !(len > 0.0)) continue; /* hinge inactive (or the axes touch: no direction) */
        double p1[3], p2[3], n[3];
        for (int i = 0; i < 3; ++i) {
            p1[i] = wa[3 * k1 + i] + (wb[3 * k1 + i] - wa[3 * k1 + i]) * t1;
            p2[i] = wa[3 * k2 + i] + (wb[3 * k2 + i] - wa[3 * k2 + i]) * t2;
            n[i] = (p1[i] - p2[i]) / len;
        }
        for (int j = 0; j < d; ++j) { /* C5: d dist / d q_j = n . (J_p1 - J_p2)[:, j];  r = w (d_safe - dist) */
            double c1[3], c2[3];
            point_jacobian_col(c, z, o, m->link[k1], j, p1, c1);
            point_jacobian_col(c, z, o, m->link[k2], j, p2, c2);
            J[p * d + j] = -m->w_coll * (n[0] * (c1[0] - c2[0]) + n[1] * (c1[1] - c2[1]) + n[2] * (c1[2] - c2[2]));
        }
    }
}
