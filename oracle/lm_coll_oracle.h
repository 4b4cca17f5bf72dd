/*
 * lm_coll_oracle.h -- fp64 CPU ORACLE of the robot-robot collision residual of CppFlow
 * (arxiv 2309.09102 sec. III-C).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as lm_oracle.h).
 *
 * "each robot is represented as a set of capsules with endpoints (a, b) and radius c ... the minimum
 *  distance between a capsule pair (a1,b1,c1) and (a2,b2,c2) [is] the minimum cost, less c1 + c2, of
 *  [the] convex quadratic program  min_{t1,t2} |(a1 + (b1 - a1) t1) - (a2 + (b2 - a2) t2)|^2,
 *  0 <= t1, t2 <= 1".
 * The oracle solves that QP by its definition: every active set of the box (interior, 4 edges,
 * 4 corners) is tried, infeasible stationary points are discarded, the smallest cost wins.
 *
 * Readings (the paper gives none of them):
 *   C1 a capsule is rigidly attached to a link frame T_L (L = -1: the base / world frame);
 *   C2 the caller lists the capsule pairs to check (PAPER.md:L49 prunes impossible pairs);
 *   C3 dist = sqrt(min QP cost) - c1 - c2;
 *   C4 one residual row per pair and waypoint, a hinge: r = w_coll * max(0, d_safe - dist)
 *      (Fig. 6 lists "self-coll-dist(q_i)" rows but no functional form; a hinge is zero when clear);
 *   C5 d dist / d q = n^T (J_p1 - J_p2), n = (p1 - p2) / |p1 - p2|, with the closest points held
 *      fixed on their links (what forward-mode differentiation through the QP solution gives:
 *      the t* terms vanish by optimality / complementarity); pinned by finite differences;
 *   C6 the rows belong to the trajectory-level step (r_diff of Fig. 6), not to the pose phase.
 * PARITY UNPINNED BY THE PAPER: capsule models (its are fitted to meshes that are not available),
 * w_coll, d_safe, the hinge.
 */
#ifndef LM_COLL_ORACLE_H
#define LM_COLL_ORACLE_H

#include "lm_oracle.h"

#define ORC_MAX_CAPS 16
#define ORC_MAX_PAIRS 32
#define ORC_MAX_OBS 8

typedef struct {
    int32_t ncaps;
    int32_t link[ORC_MAX_CAPS];  /* -1 = base frame, j = frame moved by joint j (0-based) */
    double a[ORC_MAX_CAPS][3], b[ORC_MAX_CAPS][3]; /* endpoints in the link frame */
    double c[ORC_MAX_CAPS];      /* radius */
    int32_t npairs;
    int32_t pair[ORC_MAX_PAIRS][2];
    double w_coll, d_safe;       /* C4 */
    /* robot-environment rows: cuboid obstacles "with arbitrary spatial positioning", each given
     * by its frame in the world (rotation Ro row-major = box axes as columns, origin to) and extents pmin, pmax
     * in that frame; env_pair lists (capsule, obstacle) pairs; one hinge row per pair and waypoint:
     * r = w_env * max(0, d_safe_env - dist), dist = min over t in [0,1], pmin <= p <= pmax of |p - (a + (b-a) t)| - c
     * (the paper's QP "in a frame axis-aligned to the cuboid"); d dist / d q = n^T J_p(capsule point) (C5). */
    int32_t nobs;
    double Ro[ORC_MAX_OBS][9], to[ORC_MAX_OBS][3], pmin[ORC_MAX_OBS][3], pmax[ORC_MAX_OBS][3];
    int32_t nenv;
    int32_t env_pair[ORC_MAX_PAIRS][2];
    double w_env, d_safe_env;
} orc_capsules;

/* minimum of |(a1 + (b1-a1) t1) - (a2 + (b2-a2) t2)| over the unit box; t1, t2: a minimiser */
double orc_segment_distance(const double *a1, const double *b1, const double *a2, const double *b2,
                            double *t1, double *t2);

/* minimum of |p - (a + (b-a) t)| over t in [0,1] and p in the box [pmin, pmax] (all in the box frame): the QP of
 * PAPER.md:L176-178.  For fixed t the best p is the clamp of the segment point, so the cost is a convex
 * piecewise quadratic in t: its pieces are delimited by the t at which a coordinate of the segment point crosses
 * a face plane; every piece is minimised exactly and the smallest value wins.  t, p: a minimiser. */
double orc_segment_box_distance(const double *a, const double *b, const double *pmin, const double *pmax,
                                double *t, double *p);

/* world-frame endpoints of every capsule at configuration q: wa[ncaps][3], wb[ncaps][3] */
void orc_capsule_world(const orc_chain *c, const orc_capsules *m, const double *q, double *wa, double *wb);

/* rows per waypoint: npairs self-collision rows followed by nenv environment rows (those with zero weight excluded) */
int orc_coll_rows(const orc_capsules *m);

/* dist[rows] (C3) and hinge residuals r[rows] (C4) at q (either nullable) */
void orc_coll_residual(const orc_chain *c, const orc_capsules *m, const double *q, double *dist, double *r);

/* J[rows][dof] = d r / d q (C5); rows of inactive pairs are zero */
void orc_coll_jacobian(const orc_chain *c, const orc_capsules *m, const double *q, double *J);

#endif
