/*
 * lm_oracle.c -- fp64 CPU ORACLE (test infrastructure, see lm_oracle.h).
 * Plain loops, one waypoint at a time, no blocking / fusion / reordering beyond what the
 * algorithm states.  Shares nothing with the CUDA path.
 */
#include "lm_oracle.h"

#include <math.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ 4x4 helpers */

static void mat4_identity(double T[4][4]) {
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) T[i][j] = (i == j) ? 1.0 : 0.0;
}

static void mat4_mul(const double A[4][4], const double B[4][4], double C[4][4]) {
    double tmp[4][4];
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) {
            double s = 0.0;
            for (int k = 0; k < 4; ++k) s += A[i][k] * B[k][j];
            tmp[i][j] = s;
        }
    memcpy(C, tmp, sizeof(tmp));
}

static void rot_x(double ang, double T[4][4]) {
    mat4_identity(T);
    T[1][1] = cos(ang); T[1][2] = -sin(ang);
    T[2][1] = sin(ang); T[2][2] = cos(ang);
}

static void rot_z(double ang, double T[4][4]) {
    mat4_identity(T);
    T[0][0] = cos(ang); T[0][1] = -sin(ang);
    T[1][0] = sin(ang); T[1][1] = cos(ang);
}

static void trans(double x, double y, double z, double T[4][4]) {
    mat4_identity(T);
    T[0][3] = x; T[1][3] = y; T[2][3] = z;
}

/* ------------------------------------------------------------------ quaternion / SO(3) */

void orc_quat_to_R(const double *quat, double *R) {
    /* DESIGN R11: re-normalise the stored quaternion, then the textbook conversion */
    double n = sqrt(quat[0] * quat[0] + quat[1] * quat[1] + quat[2] * quat[2] + quat[3] * quat[3]);
    double w = quat[0] / n, x = quat[1] / n, y = quat[2] / n, z = quat[3] / n;
    R[0] = 1.0 - 2.0 * (y * y + z * z); R[1] = 2.0 * (x * y - w * z);       R[2] = 2.0 * (x * z + w * y);
    R[3] = 2.0 * (x * y + w * z);       R[4] = 1.0 - 2.0 * (x * x + z * z); R[5] = 2.0 * (y * z - w * x);
    R[6] = 2.0 * (x * z - w * y);       R[7] = 2.0 * (y * z + w * x);       R[8] = 1.0 - 2.0 * (x * x + y * y);
}

void orc_log_so3(const double *E, double *w) {
    /* DESIGN R2.  v = vee of the antisymmetric part = sin(theta) * axis, c = cos(theta). */
    double v[3] = {0.5 * (E[7] - E[5]), 0.5 * (E[2] - E[6]), 0.5 * (E[3] - E[1])};
    double s = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    double c = 0.5 * (E[0] + E[4] + E[8] - 1.0);
    double theta = atan2(s, c);
    if (s < 1e-4 && c > 0.0) {
        /* small angle: theta/s = 1 + s^2/6 + O(s^4) */
        double k = 1.0 + s * s / 6.0;
        for (int i = 0; i < 3; ++i) w[i] = k * v[i];
        return;
    }
    if (s < 1e-4) {
        /* theta within 1e-4 of pi: v carries no direction.  Take the axis from the symmetric
         * part, E + E^T = 2 c I + 2 (1 - c) a a^T, largest component first, and give it the
         * sign of v (either sign is the same rotation at theta = pi exactly). */
        double a[3];
        int m = 0;
        for (int i = 0; i < 3; ++i) {
            double t = (E[4 * i] - c) / (1.0 - c);
            a[i] = t > 0.0 ? sqrt(t) : 0.0;
        }
        for (int i = 1; i < 3; ++i) if (a[i] > a[m]) m = i;
        for (int i = 0; i < 3; ++i)
            if (i != m && (E[3 * m + i] + E[3 * i + m]) < 0.0) a[i] = -a[i];
        if (a[0] * v[0] + a[1] * v[1] + a[2] * v[2] < 0.0)
            for (int i = 0; i < 3; ++i) a[i] = -a[i];
        for (int i = 0; i < 3; ++i) w[i] = theta * a[i];
        return;
    }
    for (int i = 0; i < 3; ++i) w[i] = v[i] * (theta / s);
}

/* ------------------------------------------------------------------ FK */

void orc_fk(const orc_chain *c, const double *q, double *p, double *R, double *z, double *o) {
    double T[4][4], M[4][4];
    mat4_identity(T); /* base frame = world frame, DESIGN R1 */
    for (int j = 0; j < c->dof; ++j) {
        double theta = c->theta[j], dd = c->d[j];
        if (c->joint_type[j] == 0) theta += q[j]; else dd += q[j];
        /* A_j = Rot_x(alpha_{j-1}) Trans_x(a_{j-1}) Rot_z(theta_j) Trans_z(d_j) */
        rot_x(c->alpha[j], M);   mat4_mul(T, M, T);
        trans(c->a[j], 0, 0, M); mat4_mul(T, M, T);
        rot_z(theta, M);         mat4_mul(T, M, T);
        trans(0, 0, dd, M);      mat4_mul(T, M, T);
        if (z) for (int i = 0; i < 3; ++i) z[3 * j + i] = T[i][2];
        if (o) for (int i = 0; i < 3; ++i) o[3 * j + i] = T[i][3];
    }
    /* fixed tool (flange) transform */
    double Rt[9];
    orc_quat_to_R(c->tool_q, Rt);
    mat4_identity(M);
    for (int i = 0; i < 3; ++i) {
        for (int k = 0; k < 3; ++k) M[i][k] = Rt[3 * i + k];
        M[i][3] = c->tool_p[i];
    }
    mat4_mul(T, M, T);
    for (int i = 0; i < 3; ++i) {
        p[i] = T[i][3];
        for (int k = 0; k < 3; ++k) R[3 * i + k] = T[i][k];
    }
}


/* Frames of every link: Rj[j] (row-major 3x3) and oj[j] = rotation and origin of the frame attached to the
 * link that joint j moves (T_1 .. T_d of DESIGN R1, before the tool transform).  Used by the collision
 * oracle (capsules are attached to link frames). */
void orc_fk_frames(const orc_chain *c, const double *q, double *Rj, double *oj) {
    double T[4][4], M[4][4];
    mat4_identity(T);
    for (int j = 0; j < c->dof; ++j) {
        double theta = c->theta[j], dd = c->d[j];
        if (c->joint_type[j] == 0) theta += q[j]; else dd += q[j];
        rot_x(c->alpha[j], M);   mat4_mul(T, M, T);
        trans(c->a[j], 0, 0, M); mat4_mul(T, M, T);
        rot_z(theta, M);         mat4_mul(T, M, T);
        trans(0, 0, dd, M);      mat4_mul(T, M, T);
        for (int i = 0; i < 3; ++i) {
            for (int k = 0; k < 3; ++k) Rj[9 * j + 3 * i + k] = T[i][k];
            oj[3 * j + i] = T[i][3];
        }
    }
}

/* ------------------------------------------------------------------ residual */

void orc_residual(const double *p, const double *R, const double *tp, const double *tquat,
                  double w_pos, double w_rot, double *r) {
    double Rt[9], E[9], w[3];
    orc_quat_to_R(tquat, Rt);
    /* E = R_ee R_t^T */
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += R[3 * i + k] * Rt[3 * j + k];
            E[3 * i + j] = s;
        }
    orc_log_so3(E, w);
    for (int i = 0; i < 3; ++i) {
        r[i] = w_pos * (p[i] - tp[i]);
        r[3 + i] = w_rot * w[i];
    }
}

/* ------------------------------------------------------------------ variant: roll-pitch-yaw residual */

void orc_rpy(const double *R, double *rpy) {
    /* R = Rz(yaw) Ry(pitch) Rx(roll):  R31 = -sin(pitch), R32 = cos(pitch) sin(roll), R33 = cos(pitch) cos(roll),
     * R11 = cos(yaw) cos(pitch), R21 = sin(yaw) cos(pitch) */
    rpy[0] = atan2(R[7], R[8]);
    rpy[1] = atan2(-R[6], sqrt(R[0] * R[0] + R[3] * R[3]));
    rpy[2] = atan2(R[3], R[0]);
}

static double wrap_pi(double x) {
    const double two_pi = 6.283185307179586476925287;
    x -= two_pi * floor((x + 0.5 * two_pi) / two_pi);
    return x;
}

void orc_residual_rpy(const double *p, const double *R, const double *tp, const double *tquat,
                      double w_pos, double w_rot, double *r) {
    double Rt[9], a[3], b[3];
    orc_quat_to_R(tquat, Rt);
    orc_rpy(R, a);
    orc_rpy(Rt, b);
    for (int i = 0; i < 3; ++i) {
        r[i] = w_pos * (p[i] - tp[i]);
        r[3 + i] = w_rot * wrap_pi(a[i] - b[i]);
    }
}

void orc_jacobian_to_rpy(int n, const double *R, double *J) {
    double rpy[3];
    orc_rpy(R, rpy);
    const double cp = cos(rpy[1]), sp = sin(rpy[1]), cy = cos(rpy[2]), sy = sin(rpy[2]);
    /* E = [[cy cp, -sy, 0], [sy cp, cy, 0], [-sp, 0, 1]];  E^-1 = 1/cp [[cy, sy, 0], [-sy cp, cy cp, 0], [cy sp, sy sp, cp]] */
    const double Ei[9] = {cy / cp, sy / cp, 0.0, -sy, cy, 0.0, cy * sp / cp, sy * sp / cp, 1.0};
    for (int j = 0; j < n; ++j) {
        const double w[3] = {J[3 * n + j], J[4 * n + j], J[5 * n + j]};
        for (int i = 0; i < 3; ++i) J[(3 + i) * n + j] = Ei[3 * i] * w[0] + Ei[3 * i + 1] * w[1] + Ei[3 * i + 2] * w[2];
    }
}

/* ------------------------------------------------------------------ Jacobian */

static void jacobian_from_axes(const orc_chain *c, const double *p, const double *z, const double *o,
                               double *J) {
    int n = c->dof;
    for (int j = 0; j < n; ++j) {
        const double *zj = z + 3 * j, *oj = o + 3 * j;
        if (c->joint_type[j] == 0) {
            double e[3] = {p[0] - oj[0], p[1] - oj[1], p[2] - oj[2]};
            J[0 * n + j] = zj[1] * e[2] - zj[2] * e[1];
            J[1 * n + j] = zj[2] * e[0] - zj[0] * e[2];
            J[2 * n + j] = zj[0] * e[1] - zj[1] * e[0];
            J[3 * n + j] = zj[0]; J[4 * n + j] = zj[1]; J[5 * n + j] = zj[2];
        } else {
            J[0 * n + j] = zj[0]; J[1 * n + j] = zj[1]; J[2 * n + j] = zj[2];
            J[3 * n + j] = 0.0;   J[4 * n + j] = 0.0;   J[5 * n + j] = 0.0;
        }
    }
}

void orc_jacobian(const orc_chain *c, const double *q, double *J) {
    double p[3], R[9], z[3 * ORC_MAX_DOF], o[3 * ORC_MAX_DOF];
    orc_fk(c, q, p, R, z, o);
    jacobian_from_axes(c, p, z, o, J);
}

/* ------------------------------------------------------------------ linear solve */

int orc_lu_solve(int n, const double *A, const double *b, double *x) {
    /* Gaussian elimination with partial pivoting on a copy ("batched LU") */
    double M[ORC_MAX_DOF][ORC_MAX_DOF + 1];
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) M[i][j] = A[i * n + j];
        M[i][n] = b[i];
    }
    for (int k = 0; k < n; ++k) {
        int piv = k;
        for (int i = k + 1; i < n; ++i)
            if (fabs(M[i][k]) > fabs(M[piv][k])) piv = i;
        if (!(fabs(M[piv][k]) > 0.0)) return -1; /* zero or NaN pivot */
        if (piv != k)
            for (int j = 0; j <= n; ++j) { double t = M[k][j]; M[k][j] = M[piv][j]; M[piv][j] = t; }
        for (int i = k + 1; i < n; ++i) {
            double f = M[i][k] / M[k][k];
            for (int j = k; j <= n; ++j) M[i][j] -= f * M[k][j];
        }
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = M[i][n];
        for (int j = i + 1; j < n; ++j) s -= M[i][j] * x[j];
        x[i] = s / M[i][i];
    }
    return 0;
}

int orc_lm_delta(int n, const double *J, const double *r, double lambda, double *delta) {
    /* (J^T J + lambda I) delta = -J^T r, DESIGN R4 */
    double A[ORC_MAX_DOF * ORC_MAX_DOF], g[ORC_MAX_DOF];
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j < n; ++j) {
            double s = 0.0;
            for (int k = 0; k < 6; ++k) s += J[k * n + i] * J[k * n + j];
            A[i * n + j] = s + (i == j ? lambda : 0.0);
        }
        double s = 0.0;
        for (int k = 0; k < 6; ++k) s += J[k * n + i] * r[k];
        g[i] = -s;
    }
    return orc_lu_solve(n, A, g, delta);
}

/* ------------------------------------------------------------------ LM, one waypoint */

typedef struct {
    double q[ORC_MAX_DOF];
    double p[3], R[9], z[3 * ORC_MAX_DOF], o[3 * ORC_MAX_DOF]; /* FK at q, retained */
    double r[6], F;
} wp_eval;

static void wp_evaluate(const orc_chain *c, const orc_params *prm, const double *tp,
                        const double *tquat, wp_eval *e) {
    orc_fk(c, e->q, e->p, e->R, e->z, e->o);
    if (prm->rot_mode == 1) orc_residual_rpy(e->p, e->R, tp, tquat, prm->w_pos, prm->w_rot, e->r);
    else orc_residual(e->p, e->R, tp, tquat, prm->w_pos, prm->w_rot, e->r);
    e->F = 0.0;
    for (int k = 0; k < 6; ++k) e->F += e->r[k] * e->r[k];
}

static int all_finite(const double *x, int n) {
    for (int i = 0; i < n; ++i) if (!isfinite(x[i])) return 0;
    return 1;
}

int64_t orc_lm_advance(const orc_chain *c, const orc_params *prm, int64_t W, const double *tp,
                       const double *tquat, double *q, double *lambda, int32_t *iters,
                       uint64_t *mask, uint32_t *status, int32_t max_total_iters, int32_t at_most,
                       double *res_norm, double *pos_err, double *rot_err, double *trial_q,
                       double *F_before, double *F_trial, int32_t *accepted, int32_t nthreads) {
    const int n = c->dof;
    int64_t total = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads) reduction(+ : total)
#endif
    for (int64_t w = 0; w < W; ++w) {
        wp_eval cur, tri;
        double lam = lambda[w];
        int32_t k = iters[w];
        uint64_t m = mask[w];
        uint32_t st = status[w] & ~(ORC_ST_FROZEN | ORC_ST_MAXITER);
        int32_t done = 0, last_acc = -1;
        for (int j = 0; j < n; ++j) cur.q[j] = q[w * n + j];
        wp_evaluate(c, prm, tp + 3 * w, tquat + 4 * w, &cur);

        /* DESIGN R7/R9: loop while not frozen (sqrt(F) >= tol) and iterations remain */
        while (k < max_total_iters && (at_most < 0 || done < at_most) && !(sqrt(cur.F) < prm->tol)) {
            double J[6 * ORC_MAX_DOF], Jw[6 * ORC_MAX_DOF], delta[ORC_MAX_DOF];
            jacobian_from_axes(c, cur.p, cur.z, cur.o, J);          /* DESIGN R3 */
            if (prm->rot_mode == 1) orc_jacobian_to_rpy(n, cur.R, J); /* variant: d(rpy)/dq = E^-1 J_w */
            for (int row = 0; row < 6; ++row)                         /* DESIGN R2b */
                for (int j = 0; j < n; ++j) Jw[row * n + j] = (row < 3 ? prm->w_pos : prm->w_rot) * J[row * n + j];
            int ok = (orc_lm_delta(n, Jw, cur.r, lam, delta) == 0) && all_finite(delta, n);
            if (!ok) st |= ORC_ST_SINGULAR;
            int clamped = 0;
            for (int j = 0; j < n; ++j) {                             /* DESIGN R6 */
                double t = cur.q[j] + (ok ? delta[j] : 0.0);
                if (t < c->q_lo[j]) { t = c->q_lo[j]; clamped = 1; }
                if (t > c->q_hi[j]) { t = c->q_hi[j]; clamped = 1; }
                tri.q[j] = t;
            }
            wp_evaluate(c, prm, tp + 3 * w, tquat + 4 * w, &tri);
            if (!isfinite(tri.F)) st |= ORC_ST_NONFINITE;
            if (F_before) F_before[w] = cur.F;
            if (F_trial) F_trial[w] = tri.F;
            if (trial_q) for (int j = 0; j < n; ++j) trial_q[w * n + j] = tri.q[j];
            /* DESIGN R5: strict decrease accepts, ties reject; Marquardt update, clipped */
            if (ok && isfinite(tri.F) && tri.F < cur.F) {
                cur = tri;
                if (k < 64) m |= (uint64_t)1 << k;
                lam = fmax(lam / prm->nu_down, prm->lambda_min);
                if (clamped) st |= ORC_ST_CLAMPED;
                last_acc = 1;
            } else {
                lam = fmin(lam * prm->nu_up, prm->lambda_max);
                last_acc = 0;
            }
            ++k; ++done;
        }
        if (sqrt(cur.F) < prm->tol) st |= ORC_ST_FROZEN;
        else if (k >= max_total_iters) st |= ORC_ST_MAXITER;

        for (int j = 0; j < n; ++j) q[w * n + j] = cur.q[j];
        lambda[w] = lam; iters[w] = k; mask[w] = m; status[w] = st;
        if (res_norm) res_norm[w] = sqrt(cur.F);
        /* reported errors are unweighted: PAPER.md:L45 position norm and geodesic angle */
        if (pos_err) pos_err[w] = sqrt(cur.r[0] * cur.r[0] + cur.r[1] * cur.r[1] + cur.r[2] * cur.r[2]) / prm->w_pos;
        if (rot_err) rot_err[w] = sqrt(cur.r[3] * cur.r[3] + cur.r[4] * cur.r[4] + cur.r[5] * cur.r[5]) / prm->w_rot;
        if (accepted) accepted[w] = last_acc;
        total += done;
    }
    return total;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
