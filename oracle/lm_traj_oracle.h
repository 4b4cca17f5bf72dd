/*
 * lm_traj_oracle.h -- fp64 CPU ORACLE for the trajectory-level LM step of CppFlow
 * (arxiv 2309.09102 sec. III-C): the stacked residual  r = [w_pose r_pose ; w_diff r_diff]
 * of ONE trajectory xi = [q_1..q_n], with  r_diff = [q_2 - q_1 ; ... ; q_n - q_{n-1}]
 * (Fig. 6 "differencing loss"), its Jacobian (kinematic Jacobian blocks on
 * the pose rows; -I / +I blocks on the differencing rows) and the
 * Levenberg-Marquardt update (J^T J + lambda I) delta = -J^T r (DESIGN R4).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as lm_oracle.h): only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it; it
 * shares nothing with the CUDA path.
 *
 * Two solvers for the same normal equations:
 *   orc_traj_delta_dense   the definition written out: the full (6n + d(n-1)) x (n d) Jacobian,
 *                          J^T J by triple loop, dense LU with partial pivoting (the paper's
 *                          literal solver).  O((n d)^3): small n only.
 *   orc_traj_delta_banded  Gaussian elimination of the SAME matrix restricted to its band: the
 *                          pose rows couple only the d joints of one waypoint and a differencing
 *                          row couples joint a of waypoints i and i+1, so (J^T J + lambda I)[u][v]
 *                          = 0 for |u - v| > d; symmetric positive definite => Cholesky in band
 *                          storage, no pivoting.  tests/test_oracle_traj.py pins it to the dense
 *                          one and both to numpy's least-squares solution of the augmented system.
 * The batched driver uses the banded solver (a flag selects the dense one for the pins).
 *
 * Readings (T1-T6): per-TRAJECTORY lambda and accept/reject on the total
 * cost F = |r|^2 (the differencing rows couple the waypoints, so the step is one problem per
 * trajectory); the trial point is clamped; strict decrease accepts.
 * PARITY UNPINNED BY THE PAPER: w_pose, w_diff, the lambda constants (the paper gives none).
 */
#ifndef LM_TRAJ_ORACLE_H
#define LM_TRAJ_ORACLE_H

#include "lm_coll_oracle.h"
#include "lm_oracle.h"

typedef struct {
    double w_pose, w_diff;                                  /* DESIGN T1 */
    double lambda0, nu_up, nu_down, lambda_min, lambda_max; /* DESIGN T3 (= R5, per trajectory) */
    const orc_capsules *caps; /* nullable: self-collision rows (lm_coll_oracle.h, Fig. 6 "self-coll-dist(q_i)"),
                                 np = orc_coll_rows(caps) hinge rows per waypoint (self-collision pairs, then capsule-obstacle
                                 pairs) appended after the differencing rows: row 6n + d(n-1) + np * i + p */
} orc_traj_params;

/* rows of the stacked residual / Jacobian of one n-waypoint trajectory (without / with the collision rows) */
int64_t orc_traj_rows(int32_t dof, int64_t n);
int64_t orc_traj_rows_all(const orc_traj_params *tp_, int32_t dof, int64_t n);

/* r[6n + d(n-1)]: rows 6i..6i+5 = w_pose * pose residual of waypoint i (orc_residual, weights
 * prm->w_pos / w_rot); rows 6n + d k + a = w_diff * (q[k+1][a] - q[k][a]).   q: [n][d], tp: [n][3],
 * tquat: [n][4]. */
void orc_traj_residual(const orc_chain *c, const orc_params *prm, const orc_traj_params *tp_,
                       int64_t n, const double *tp, const double *tquat, const double *q, double *r);

/* J[rows][n d] row-major, the Jacobian of orc_traj_residual wrt xi as the paper states it:
 * pose rows = kinematic Jacobian of waypoint i in columns d i .. d i + d - 1 (used
 * as is: DESIGN R3), differencing row (k, a) = -w_diff at column d k + a, +w_diff at d (k+1) + a. */
void orc_traj_jacobian(const orc_chain *c, const orc_params *prm, const orc_traj_params *tp_,
                       int64_t n, const double *q, double *J);

/* delta[n d] = -(J^T J + lambda I)^-1 J^T r.  Return 0, or -1 (singular / not positive definite). */
int orc_traj_delta_dense(const orc_chain *c, const orc_params *prm, const orc_traj_params *tp_,
                         int64_t n, const double *tp, const double *tquat, const double *q,
                         double lambda, double *delta);
int orc_traj_delta_banded(const orc_chain *c, const orc_params *prm, const orc_traj_params *tp_,
                          int64_t n, const double *tp, const double *tquat, const double *q,
                          double lambda, double *delta);

/* Batched driver: B independent trajectories of n waypoints (trajectory-major: q[B][n][d],
 * tp[B][n][3], tquat[B][n][4]).  Per trajectory: state q, lambda, iters, mask, status; advances
 * until iters == max_total_iters or `at_most` iterations were done in this call (< 0: no cap).
 * Outputs (nullable): F_total = w_pose^2 F_pose + w_diff^2 F_diff, F_pose = sum_i |r_pose,i|^2,
 * F_diff = sum_k |q_{k+1} - q_k|^2 at the current q (the collision rows add their squares to F_total only).  Trace of the LAST iteration executed in
 * this call (nullable): trial_q[B][n][d], F_before[B], F_trial[B], accepted[B] (-1 = none).
 * use_dense != 0 selects orc_traj_delta_dense.  Returns the number of trajectory-iterations executed. */
int64_t orc_traj_lm_advance(const orc_chain *c, const orc_params *prm, const orc_traj_params *tp_,
                            int64_t B, int64_t n, const double *tp, const double *tquat, double *q,
                            double *lambda, int32_t *iters, uint64_t *mask, uint32_t *status,
                            int32_t max_total_iters, int32_t at_most, double *F_total, double *F_pose,
                            double *F_diff, double *trial_q, double *F_before, double *F_trial,
                            int32_t *accepted, int32_t use_dense, int32_t nthreads);

#endif
