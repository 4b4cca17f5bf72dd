/*
 * lm_oracle.h -- fp64 CPU ORACLE for the batched Levenberg-Marquardt pose refinement of
 * CppFlow (arxiv 2309.09102).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call anything in oracle/.
 * It shares no code, header, table or constant generator with the CUDA path
 * (paper_2309_09102_b200/csrc, include/lm.h) and neither includes the other.
 *
 * It is plain, slow and written to be checked against the paper by eye: 4x4 homogeneous
 * matrices multiplied with triple loops, a dense LU with partial pivoting (the paper's literal
 * choice of solver), one waypoint at a time.  Citations are PAPER.md line numbers;
 * "DESIGN R<n>" refers to the numbered readings of the paper's silences in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_pins.py): FK closed forms, Log map vs scipy, finite-difference
 * Jacobian, ridge-regression identity for the solve, lambda->inf / lambda->0 limits, exact
 * convergence on a locked 6-DoF chain.
 * PARITY UNPINNED BY THE PAPER: the lambda-rule constants (nu, lambda_min, lambda_max), unit
 * weights and the strict '<' tie-break -- the paper gives none (DESIGN R5); both sides
 * implement the same table.
 */
#ifndef LM_ORACLE_H
#define LM_ORACLE_H

#include <stdint.h>

#define ORC_MAX_DOF 8

/* Serial chain in modified-DH (Craig) form, DESIGN R1.  Row j (0-based) holds
 * a_{j-1}, alpha_{j-1}, d_j, theta_j of   A_j = Rot_x(alpha) Trans_x(a) Rot_z(theta) Trans_z(d).
 * Revolute: theta = theta[j] + q_j.  Prismatic: d = d[j] + q_j. */
typedef struct {
    int32_t dof;
    int32_t joint_type[ORC_MAX_DOF]; /* 0 revolute, 1 prismatic */
    double a[ORC_MAX_DOF], alpha[ORC_MAX_DOF], d[ORC_MAX_DOF], theta[ORC_MAX_DOF];
    double q_lo[ORC_MAX_DOF], q_hi[ORC_MAX_DOF]; /* joint limits */
    double tool_p[3];                            /* fixed flange transform after joint d */
    double tool_q[4];                            /* unit quaternion w,x,y,z */
} orc_chain;

typedef struct {
    double lambda0, nu_up, nu_down, lambda_min, lambda_max; /* DESIGN R5 */
    double tol;                                             /* DESIGN R7/R8: freeze when sqrt(F) < tol */
    double w_pos, w_rot;                                    /* DESIGN R2b */
    int32_t rot_mode; /* 0 (default): r_rot = Log(R R_t^T)^vee, DESIGN R2.  1: the paper's literal wording (PAPER.md:L47,
                         L115-117): element-wise difference of roll, pitch, yaw (variant) */
} orc_params;

/* status bits (same meaning as include/lm.h, restated, not shared) */
#define ORC_ST_FROZEN 1u
#define ORC_ST_MAXITER 2u
#define ORC_ST_SINGULAR 4u
#define ORC_ST_NONFINITE 8u
#define ORC_ST_CLAMPED 16u

/* ---- single-configuration pieces (all row-major) ---- */

/* FK(q): R^d -> SE(3).  p[3], R[9]; z[j], o[j] = joint axis / frame origin of
 * joint j in the world frame (nullable). */
void orc_fk(const orc_chain *c, const double *q, double *p, double *R, double *z, double *o);

/* link frames T_1..T_d: Rj[d][9] row-major rotations, oj[d][3] origins (world frame) */
void orc_fk_frames(const orc_chain *c, const double *q, double *Rj, double *oj);

/* unit-normalise then convert quaternion (w,x,y,z) to a rotation matrix, DESIGN R11 */
void orc_quat_to_R(const double *quat, double *R);

/* w = Log(E)^vee for E in SO(3), DESIGN R2; |w| is the geodesic distance of PAPER.md:L45 */
void orc_log_so3(const double *E, double *w);

/* r = [w_pos (p - p_t) ; w_rot Log(R R_t^T)^vee], PAPER.md:L47, L115-117 as read by DESIGN R2 */
void orc_residual(const double *p, const double *R, const double *tp, const double *tquat,
                  double w_pos, double w_rot, double *r);

/* roll, pitch, yaw of R = Rot_z(yaw) Rot_y(pitch) Rot_x(roll) (fixed-axis x-y-z; pitch in [-pi/2, pi/2]) */
void orc_rpy(const double *R, double *rpy);

/* the paper's literal pose residual: r = [w_pos (p - p_t) ; w_rot wrap(rpy(R) - rpy(R_t))],
 * every angle difference wrapped to (-pi, pi] */
void orc_residual_rpy(const double *p, const double *R, const double *tp, const double *tquat,
                      double w_pos, double w_rot, double *r);

/* rows 3..5 of J (6 x dof row-major, geometric Jacobian) <- E(rpy(R))^-1 J_w, the exact derivative of (roll, pitch,
 * yaw) wrt q:  w = E d(rpy)/dt,  E = [Rz Ry e_x | Rz e_y | e_z] */
void orc_jacobian_to_rpy(int dof, const double *R, double *J);

/* geometric Jacobian 6 x dof (row-major, leading dimension dof), DESIGN R3 */
void orc_jacobian(const orc_chain *c, const double *q, double *J);

/* solve A x = b (n x n, row-major) by LU with partial pivoting; returns 0, or -1 if singular */
int orc_lu_solve(int n, const double *A, const double *b, double *x);

/* LM step  delta = -(J^T J + lambda I)^-1 J^T r, PAPER.md:L121 as read by DESIGN R4.
 * J is 6 x n row-major.  Returns 0 or -1 (singular). */
int orc_lm_delta(int n, const double *J, const double *r, double lambda, double *delta);

/* ---- batched driver ----
 * W independent waypoints (the pose Jacobian is block diagonal).
 * Arrays are waypoint-major: q[W][dof], tp[W][3], tquat[W][4].
 * Advances every waypoint until it is frozen, or iters[w] == max_total_iters, or it has done
 * `at_most` iterations in this call (at_most < 0: no per-call cap).
 * State in/out: q, lambda, iters, mask, status.  Outputs (nullable): res_norm, pos_err, rot_err.
 * Trace of the LAST iteration executed in this call (nullable): trial_q[W][dof], F_before[W],
 * F_trial[W], accepted[W] (-1 if no iteration was executed).
 * nthreads <= 0: all cores (OpenMP).  Returns the number of iterations executed in this call. */
int64_t orc_lm_advance(const orc_chain *c, const orc_params *prm, int64_t W, const double *tp,
                       const double *tquat, double *q, double *lambda, int32_t *iters,
                       uint64_t *mask, uint32_t *status, int32_t max_total_iters, int32_t at_most,
                       double *res_norm, double *pos_err, double *rot_err, double *trial_q,
                       double *F_before, double *F_trial, int32_t *accepted, int32_t nthreads);

int orc_num_threads(void);

#endif
