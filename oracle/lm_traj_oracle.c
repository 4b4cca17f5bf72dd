/*
 * lm_traj_oracle.c -- fp64 CPU ORACLE of the trajectory-level LM step (test infrastructure, see
 * lm_traj_oracle.h).  Plain loops; the dense path is the definition written out, the banded path
 * is Gaussian elimination of the same matrix that skips its structural zeros.
 */
#include "lm_traj_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int64_t orc_traj_rows(int32_t dof, int64_t n) { return 6 * n + (int64_t)dof * (n - 1); }

static int coll_rows(const orc_traj_params *t) { return t->caps ? orc_coll_rows(t->caps) : 0; }

int64_t orc_traj_rows_all(const orc_traj_params *t, int32_t dof, int64_t n) {
    return orc_traj_rows(dof, n) + (int64_t)coll_rows(t) * n;
}

/* ------------------------------------------------------------------ residual, PAPER.md:L117 (Fig. 6) */

void orc_traj_residual(const orc_chain *c, const orc_params *prm, const orc_traj_params *t,
                       int64_t n, const double *tp, const double *tquat, const double *q, double *r) {
    const int d = c->dof;
    for (int64_t i = 0; i < n; ++i) { /* r_pose: one 6-vector per waypoint */
        double p[3], R[9], ri[6];
        orc_fk(c, q + i * d, p, R, NULL, NULL);
        orc_residual(p, R, tp + 3 * i, tquat + 4 * i, prm->w_pos, prm->w_rot, ri);
        for (int k = 0; k < 6; ++k) r[6 * i + k] = t->w_pose * ri[k];
    }
    for (int64_t k = 0; k + 1 < n; ++k) /* r_diff: q_{k+1} - q_k */
        for (int a = 0; a < d; ++a)
            r[6 * n + d * k + a] = t->w_diff * (q[(k + 1) * d + a] - q[k * d + a]);
    const int np = coll_rows(t);
    for (int64_t i = 0; i < n && np > 0; ++i) /* self-collision hinge rows, PAPER.md:L117 (Fig. 6) */
        orc_coll_residual(c, t->caps, q + i * d, NULL, r + orc_traj_rows(d, n) + np * i);
}

/* ------------------------------------------------------------------ Jacobian */

void orc_traj_jacobian(const orc_chain *c, const orc_params *prm, const orc_traj_params *t,
                       int64_t n, const double *q, double *J) {
    const int d = c->dof;
    const int64_t rows = orc_traj_rows_all(t, d, n), cols = n * d;
    memset(J, 0, sizeof(double) * (size_t)(rows * cols));
    for (int64_t i = 0; i < n; ++i) {
        double Ji[6 * ORC_MAX_DOF];
        orc_jacobian(c, q + i * d, Ji); /* kinematic Jacobian of waypoint i */
        for (int k = 0; k < 6; ++k)
            for (int a = 0; a < d; ++a)
                J[(6 * i + k) * cols + d * i + a] = t->w_pose * (k < 3 ? prm->w_pos : prm->w_rot) * Ji[k * d + a];
    }
    for (int64_t k = 0; k + 1 < n; ++k)
        for (int a = 0; a < d; ++a) {
            /* "identity for q_{i+1}, negated identity for q_i" */
            J[(6 * n + d * k + a) * cols + d * k + a] = -t->w_diff;
            J[(6 * n + d * k + a) * cols + d * (k + 1) + a] = t->w_diff;
        }
    const int np = coll_rows(t);
    for (int64_t i = 0; i < n && np > 0; ++i) { /* collision rows of waypoint i depend on q_i only */
        double Jc[2 * ORC_MAX_PAIRS * ORC_MAX_DOF];
        orc_coll_jacobian(c, t->caps, q + i * d, Jc);
        for (int p = 0; p < np; ++p)
            for (int a = 0; a < d; ++a) J[(orc_traj_rows(d, n) + np * i + p) * cols + d * i + a] = Jc[p * d + a];
    }
}

/* ------------------------------------------------------------------ dense solve (the definition) */

/* A x = b, N x N row-major, Gaussian elimination with partial pivoting on copies */
static int lu_solve_big(int64_t N, const double *A, const double *b, double *x) {
    double *M = (double *)malloc(sizeof(double) * (size_t)(N * (N + 1)));
    if (!M) return -1;
    for (int64_t i = 0; i < N; ++i) {
        for (int64_t j = 0; j < N; ++j) M[i * (N + 1) + j] = A[i * N + j];
        M[i * (N + 1) + N] = b[i];
    }
    int rc = 0;
    for (int64_t k = 0; k < N && rc == 0; ++k) {
        int64_t piv = k;
        for (int64_t i = k + 1; i < N; ++i)
            if (fabs(M[i * (N + 1) + k]) > fabs(M[piv * (N + 1) + k])) piv = i;
        if (!(fabs(M[piv * (N + 1) + k]) > 0.0)) { rc = -1; break; }
        if (piv != k)
            for (int64_t j = 0; j <= N; ++j) {
                double tmp = M[k * (N + 1) + j]; M[k * (N + 1) + j] = M[piv * (N + 1) + j]; M[piv * (N + 1) + j] = tmp;
            }
        for (int64_t i = k + 1; i < N; ++i) {
            double f = M[i * (N + 1) + k] / M[k * (N + 1) + k];
            if (f != 0.0)
                for (int64_t j = k; j <= N; ++j) M[i * (N + 1) + j] -= f * M[k * (N + 1) + j];
        }
    }
    if (rc == 0)
        for (int64_t i = N - 1; i >= 0; --i) {
            double s = M[i * (N + 1) + N];
            for (int64_t j = i + 1; j < N; ++j) s -= M[i * (N + 1) + j] * x[j];
            x[i] = s / M[i * (N + 1) + i];
        }
    free(M);
    return rc;
}

int orc_traj_delta_dense(const orc_chain *c, const orc_params *prm, const orc_traj_params *t,
                         int64_t n, const double *tp, const double *tquat, const double *q,
                         double lambda, double *delta) {
    const int d = c->dof;
    const int64_t rows = orc_traj_rows_all(t, d, n), N = n * d;
    double *J = (double *)malloc(sizeof(double) * (size_t)(rows * N));
    double *r = (double *)malloc(sizeof(double) * (size_t)rows);
    double *A = (double *)malloc(sizeof(double) * (size_t)(N * N));
    double *g = (double *)malloc(sizeof(double) * (size_t)N);
    if (!J || !r || !A || !g) { free(J); free(r); free(A); free(g); return -1; }
    orc_traj_jacobian(c, prm, t, n, q, J);
    orc_traj_residual(c, prm, t, n, tp, tquat, q, r);
    /* (J^T J + lambda I) delta = -J^T r, DESIGN R4 */
    for (int64_t u = 0; u < N; ++u) {
        for (int64_t v = 0; v < N; ++v) {
            double s = 0.0;
            for (int64_t k = 0; k < rows; ++k) s += J[k * N + u] * J[k * N + v];
            A[u * N + v] = s + (u == v ? lambda : 0.0);
        }
        double s = 0.0;
        for (int64_t k = 0; k < rows; ++k) s += J[k * N + u] * r[k];
        g[u] = -s;
    }
    int rc = lu_solve_big(N, A, g, delta);
    free(J); free(r); free(A); free(g);
    return rc;
}

/* ------------------------------------------------------------------ banded solve (same matrix) */

/* Lower band storage: ab[u * (kd + 1) + k] = A[u + k][u], k = 0..kd (column u, k-th subdiagonal). */
static int band_cholesky_solve(int64_t N, int kd, double *ab, double *x /* in: rhs, out: solution */) {
    const int ld = kd + 1;
    for (int64_t j = 0; j < N; ++j) {
        double ajj = ab[j * ld];
        if (!(ajj > 0.0)) return -1;
        ajj = sqrt(ajj);
        ab[j * ld] = ajj;
        const int kn = (int)((N - 1 - j) < kd ? (N - 1 - j) : kd);
        for (int k = 1; k <= kn; ++k) ab[j * ld + k] /= ajj;
        for (int cc = 1; cc <= kn; ++cc)      /* A[j+r][j+cc] -= L[j+r][j] L[j+cc][j],  r >= cc */
            for (int rr = cc; rr <= kn; ++rr) ab[(j + cc) * ld + (rr - cc)] -= ab[j * ld + rr] * ab[j * ld + cc];
    }
    for (int64_t j = 0; j < N; ++j) { /* L y = b */
        x[j] /= ab[j * ld];
        const int kn = (int)((N - 1 - j) < kd ? (N - 1 - j) : kd);
        for (int k = 1; k <= kn; ++k) x[j + k] -= ab[j * ld + k] * x[j];
    }
    for (int64_t j = N - 1; j >= 0; --j) { /* L^T x = y */
        const int kn = (int)((N - 1 - j) < kd ? (N - 1 - j) : kd);
        double s = x[j];
        for (int k = 1; k <= kn; ++k) s -= ab[j * ld + k] * x[j + k];
        x[j] = s / ab[j * ld];
    }
    return 0;
}

int orc_traj_delta_banded(const orc_chain *c, const orc_params *prm, const orc_traj_params *t,
                          int64_t n, const double *tp, const double *tquat, const double *q,
                          double lambda, double *delta) {
    const int d = c->dof, kd = d, ld = kd + 1;
    const int64_t N = n * d;
    double *ab = (double *)calloc((size_t)(N * ld), sizeof(double));
    if (!ab) return -1;
    const double wd2 = t->w_diff * t->w_diff;
    for (int64_t i = 0; i < n; ++i) {
        /* pose rows of waypoint i: J_i^T J_i on the diagonal block, J_i^T r_i in the gradient */
        double p[3], R[9], ri[6], Ji[6 * ORC_MAX_DOF];
        orc_fk(c, q + i * d, p, R, NULL, NULL);
        orc_residual(p, R, tp + 3 * i, tquat + 4 * i, prm->w_pos, prm->w_rot, ri);
        orc_jacobian(c, q + i * d, Ji);
        for (int k = 0; k < 6; ++k) {
            const double w = t->w_pose * (k < 3 ? prm->w_pos : prm->w_rot);
            ri[k] *= t->w_pose;
            for (int a = 0; a < d; ++a) Ji[k * d + a] *= w;
        }
        for (int a = 0; a < d; ++a) {
            for (int b = 0; b <= a; ++b) { /* entry (d i + a, d i + b), a >= b: column d i + b, subdiagonal a - b */
                double s = 0.0;
                for (int k = 0; k < 6; ++k) s += Ji[k * d + a] * Ji[k * d + b];
                ab[(d * i + b) * ld + (a - b)] += s;
            }
            double s = 0.0;
            for (int k = 0; k < 6; ++k) s += Ji[k * d + a] * ri[k];
            delta[d * i + a] = -s;
            ab[(d * i + a) * ld] += lambda;
        }
        const int np = coll_rows(t);
        if (np > 0) { /* collision rows of waypoint i: J_c^T J_c on the diagonal block, J_c^T r_c in the gradient */
            double Jc[2 * ORC_MAX_PAIRS * ORC_MAX_DOF], rc[2 * ORC_MAX_PAIRS];
            orc_coll_jacobian(c, t->caps, q + i * d, Jc);
            orc_coll_residual(c, t->caps, q + i * d, NULL, rc);
            for (int p = 0; p < np; ++p)
                for (int a = 0; a < d; ++a) {
                    for (int b = 0; b <= a; ++b) ab[(d * i + b) * ld + (a - b)] += Jc[p * d + a] * Jc[p * d + b];
                    delta[d * i + a] -= Jc[p * d + a] * rc[p];
                }
        }
    }
    for (int64_t k = 0; k + 1 < n; ++k) /* differencing row (k, a): -w at column (k, a), +w at (k+1, a) */
        for (int a = 0; a < d; ++a) {
            const double rk = t->w_diff * (q[(k + 1) * d + a] - q[k * d + a]);
            ab[(d * k + a) * ld] += wd2;
            ab[(d * (k + 1) + a) * ld] += wd2;
            ab[(d * k + a) * ld + d] += -wd2; /* entry (d (k+1) + a, d k + a) */
            delta[d * k + a] -= -t->w_diff * rk;
            delta[d * (k + 1) + a] -= t->w_diff * rk;
        }
    int rc = band_cholesky_solve(N, kd, ab, delta);
    free(ab);
    return rc;
}

/* ------------------------------------------------------------------ cost and LM driver */

static void traj_cost(const orc_chain *c, const orc_params *prm, const orc_traj_params *t, int64_t n,
                      const double *tp, const double *tquat, const double *q, double *Fp, double *Fd, double *F) {
    const int d = c->dof;
    double fp = 0.0, fd = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double p[3], R[9], ri[6];
        orc_fk(c, q + i * d, p, R, NULL, NULL);
        orc_residual(p, R, tp + 3 * i, tquat + 4 * i, prm->w_pos, prm->w_rot, ri);
        for (int k = 0; k < 6; ++k) fp += ri[k] * ri[k];
    }
    for (int64_t k = 0; k + 1 < n; ++k)
        for (int a = 0; a < d; ++a) {
            const double e = q[(k + 1) * d + a] - q[k * d + a];
            fd += e * e;
        }
    double fc = 0.0;
    const int np = coll_rows(t);
    for (int64_t i = 0; i < n && np > 0; ++i) {
        double rc[2 * ORC_MAX_PAIRS];
        orc_coll_residual(c, t->caps, q + i * d, NULL, rc);
        for (int p = 0; p < np; ++p) fc += rc[p] * rc[p];
    }
    *Fp = fp; *Fd = fd;
    *F = t->w_pose * t->w_pose * fp + t->w_diff * t->w_diff * fd + fc;
}

int64_t orc_traj_lm_advance(const orc_chain *c, const orc_params *prm, const orc_traj_params *t,
                            int64_t B, int64_t n, const double *tp, const double *tquat, double *q,
                            double *lambda, int32_t *iters, uint64_t *mask, uint32_t *status,
                            int32_t max_total_iters, int32_t at_most, double *F_total, double *F_pose,
                            double *F_diff, double *trial_q, double *F_before, double *F_trial,
                            int32_t *accepted, int32_t use_dense, int32_t nthreads) {
    const int d = c->dof;
    const int64_t N = n * d;
    int64_t total = 0;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads) reduction(+ : total)
#endif
    for (int64_t b = 0; b < B; ++b) {
        const double *tpb = tp + 3 * n * b, *tqb = tquat + 4 * n * b;
        double *qb = q + N * b;
        double *delta = (double *)malloc(sizeof(double) * (size_t)N);
        double *qt = (double *)malloc(sizeof(double) * (size_t)N);
        double lam = lambda[b];
        int32_t k = iters[b], done = 0, last_acc = -1;
        uint64_t m = mask[b];
        uint32_t st = status[b] & ~(ORC_ST_MAXITER);
        double Fp, Fd, F;
        traj_cost(c, prm, t, n, tpb, tqb, qb, &Fp, &Fd, &F);
        while (k < max_total_iters && (at_most < 0 || done < at_most)) {
            int ok = ((use_dense ? orc_traj_delta_dense : orc_traj_delta_banded)(c, prm, t, n, tpb, tqb, qb, lam, delta) == 0);
            for (int64_t u = 0; u < N && ok; ++u) if (!isfinite(delta[u])) ok = 0;
            if (!ok) st |= ORC_ST_SINGULAR;
            int clamped = 0;
            for (int64_t i = 0; i < n; ++i)
                for (int a = 0; a < d; ++a) { /* the trial point is clamped */
                    double v = qb[i * d + a] + (ok ? delta[i * d + a] : 0.0);
                    if (v < c->q_lo[a]) { v = c->q_lo[a]; clamped = 1; }
                    if (v > c->q_hi[a]) { v = c->q_hi[a]; clamped = 1; }
                    qt[i * d + a] = v;
                }
            double Fpt, Fdt, Ft;
            traj_cost(c, prm, t, n, tpb, tqb, qt, &Fpt, &Fdt, &Ft);
            if (!isfinite(Ft)) st |= ORC_ST_NONFINITE;
            if (F_before) F_before[b] = F;
            if (F_trial) F_trial[b] = Ft;
            if (trial_q) memcpy(trial_q + N * b, qt, sizeof(double) * (size_t)N);
            if (ok && isfinite(Ft) && Ft < F) { /* strict decrease accepts (DESIGN R5 / T3) */
                memcpy(qb, qt, sizeof(double) * (size_t)N);
                F = Ft; Fp = Fpt; Fd = Fdt;
                if (k < 64) m |= (uint64_t)1 << k;
                lam = fmax(lam / t->nu_down, t->lambda_min);
                if (clamped) st |= ORC_ST_CLAMPED;
                last_acc = 1;
            } else {
                lam = fmin(lam * t->nu_up, t->lambda_max);
                last_acc = 0;
            }
            ++k; ++done;
        }
        if (k >= max_total_iters) st |= ORC_ST_MAXITER;
        lambda[b] = lam; iters[b] = k; mask[b] = m; status[b] = st;
        if (F_total) F_total[b] = F;
        if (F_pose) F_pose[b] = Fp;
        if (F_diff) F_diff[b] = Fd;
        if (accepted) accepted[b] = last_acc;
        total += done;
        free(delta); free(qt);
    }
    return total;
}
