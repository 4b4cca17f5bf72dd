// lm_traj.cuh -- kernels of the trajectory-level LM step (sm_100a): the stacked residual
//   r = [w_pose r_pose ; w_diff (q_{k+1} - q_k)_k]            (Fig. 6)
// whose Jacobian has the kinematic Jacobian J_i on the pose rows of waypoint i and
// -I / +I on the differencing rows, so that per trajectory
//   J^T J + lambda I = block-tridiag( T_i , -w_d^2 I ),   T_i = w_p^2 J_i^T J_i + (c_i w_d^2 + lambda) I,
//   c_i = 1 at the two ends, 2 inside (0 for n = 1).
// The block structure is kept (include/lm.h): block Gaussian elimination
// along the waypoint index (block Thomas),
//   S_1 = T_1,  S_i = T_i - w_d^4 S_{i-1}^-1,  h_i = g_i + w_d^2 S_{i-1}^-1 h_{i-1},
//   x_n = S_n^-1 h_n,  x_i = S_i^-1 h_i + w_d^2 S_i^-1 x_{i+1},          delta = -x,
// one THREAD per trajectory (the recurrence is sequential in i, the trajectories are the parallel
// dimension), d x d symmetric blocks in registers, S_i^-1 by the symmetric sweep operator.
// Everything per-waypoint (FK, Jacobian, J^T J, J^T r, trial cost) runs one thread per waypoint.
//
// Layout: "e-order" structure-of-arrays, e = i * B + b (trajectory index fastest), so that both
// the per-waypoint kernels (consecutive lanes = consecutive e) and the per-trajectory kernel
// (consecutive lanes = consecutive b at the same i) touch consecutive 4-byte words.
// Determinism: fixed summation orders, no float atomics; explicit round-to-nearest intrinsics.
#pragma once
#include "lm_device.cuh"
#include "lm_kernels.cuh"

namespace lmk {

struct TArgs {
    KChain ch;
    float w_pos, w_rot;            // pose residual weights (lm_params)
    float wp2, wd2, wd4;           // w_pose^2, w_diff^2, w_diff^4
    float nu_up, inv_nu_down, lambda_min, lambda_max;
    int64_t B, nB;                 // trajectories, n * B
    int32_t n;
    int32_t shared_targets;
    int32_t max_total;             // iteration cap per trajectory (mask width)
    int32_t mode;                  // solve kernel: 0 = factor + solve for g, 1 = re-solve for rho (refinement)
    const float *tp, *tq;          // targets, e-order [3][nBt], [4][nBt] (nBt = n when shared)
    float *q;                      // [2][D][nB]   current / candidate joint values
    float *A;                      // [2][NA][nB]  w_p^2 J^T J, packed lower triangle
    float *gp;                     // [2][D][nB]   w_p^2 J^T r
    float *cst;                    // [2][2][nB]   |r_pose,i|^2 and |q_{i+1} - q_i|^2 (0 for the last waypoint)
    float *V;                      // [NA][nB]     -(S_i)^-1
    float *z;                      // [D][nB]
    float *delta;                  // [D][nB]
    float *rho;                    // [D][nB]
    float *lam, *F, *Fp, *Fd;      // [B]
    uint32_t *its;                 // [B] iters | status << 8
    unsigned long long *mask;      // [B]
    int32_t *sel;                  // [B] which of the two buffers holds the current point
    int32_t *ok;                   // [B] this iteration's solve succeeded
    float *trace_q, *trace_F;      // nullable: trial point [D][W] in w-order (w = b n + i), (F, F+) [2][B]
    // pack / unpack (w-order <-> e-order)
    const float *src_q;            // [D][W] w-order
    const float *src_tp, *src_tq;  // [3][Wt], [4][Wt] w-order
    float *dst_q;                  // [D][W] w-order
};

template <int D> struct Tri { static constexpr int NA = D * (D + 1) / 2; };
__host__ __device__ constexpr int tri(int r, int c) { return r >= c ? r * (r + 1) / 2 + c : c * (c + 1) / 2 + r; }

// ---- w-order -> e-order (targets once per attach, q at the start of every lm_traj_run)
template <int D>
__global__ void __launch_bounds__(256) tl_pack_kernel(const __grid_constant__ TArgs A, int what) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.nB) return;
    const int64_t i = e / A.B, b = e - i * A.B;
    const int64_t w = b * A.n + i, W = A.nB;
    if (what == 0) { // joint values into the buffer the trajectory currently selects
        float *dst = A.q + (int64_t)A.sel[b] * D * A.nB;
#pragma unroll
        for (int j = 0; j < D; ++j) dst[(int64_t)j * A.nB + e] = A.src_q[(int64_t)j * W + w];
    } else if (!A.shared_targets) {
#pragma unroll
        for (int c = 0; c < 3; ++c) const_cast<float *>(A.tp)[(int64_t)c * A.nB + e] = A.src_tp[(int64_t)c * W + w];
#pragma unroll
        for (int c = 0; c < 4; ++c) const_cast<float *>(A.tq)[(int64_t)c * A.nB + e] = A.src_tq[(int64_t)c * W + w];
    }
}

template <int D>
__global__ void __launch_bounds__(256) tl_unpack_kernel(const __grid_constant__ TArgs A) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.nB) return;
    const int64_t i = e / A.B, b = e - i * A.B;
    const int64_t w = b * A.n + i, W = A.nB;
    const float *src = A.q + (int64_t)A.sel[b] * D * A.nB;
#pragma unroll
    for (int j = 0; j < D; ++j) A.dst_q[(int64_t)j * W + w] = src[(int64_t)j * A.nB + e];
}

// load the target of (i, b) and convert the quaternion (DESIGN R11)
__device__ __forceinline__ void tl_load_target(const TArgs &A, int64_t e, int64_t i, float (&pt)[3], float (&Rt)[3][3]) {
    const int64_t Wt = A.shared_targets ? (int64_t)A.n : A.nB;
    const int64_t wt = A.shared_targets ? i : e;
#pragma unroll
    for (int c = 0; c < 3; ++c) pt[c] = __ldg(A.tp + (int64_t)c * Wt + wt);
    quat_to_cols(__ldg(A.tq + wt), __ldg(A.tq + Wt + wt), __ldg(A.tq + 2 * Wt + wt), __ldg(A.tq + 3 * Wt + wt), Rt);
}

// w_p^2 J^T J (packed lower), w_p^2 J^T r, |r|^2 of one waypoint -> buffer `dstsel`
template <int D>
__device__ __forceinline__ void tl_store_normal(const TArgs &A, const Pose<D> &P, int dstsel, int64_t e, float fd) {
    constexpr int NA = Tri<D>::NA;
    float *Ad = A.A + (int64_t)dstsel * NA * A.nB + e;
    float *gd = A.gp + (int64_t)dstsel * D * A.nB + e;
#pragma unroll
    for (int r = 0; r < D; ++r) {
#pragma unroll
        for (int c = 0; c <= r; ++c) Ad[(int64_t)tri(r, c) * A.nB] = mul(A.wp2, coldot<D>(P, r, c));
        gd[(int64_t)r * A.nB] = mul(A.wp2, colvec<D>(P, r, P.r));
    }
    float *cd = A.cst + (int64_t)dstsel * 2 * A.nB + e;
    cd[0] = P.F;
    cd[A.nB] = fd;
}

// ---- assemble at the current point (entry of lm_traj_run): thread per waypoint
template <int D, bool FAST, bool WEIGHTED, typename SpecT>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) tl_assemble_kernel(const __grid_constant__ TArgs A) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.nB) return;
    const int64_t i = e / A.B, b = e - i * A.B;
    const int s = A.sel[b];
    const float *qs = A.q + (int64_t)s * D * A.nB;
    float q[D], fd = 0.f;
#pragma unroll
    for (int j = 0; j < D; ++j) q[j] = qs[(int64_t)j * A.nB + e];
    if (i + 1 < A.n) {
#pragma unroll
        for (int j = 0; j < D; ++j) {
            const float t = sub(qs[(int64_t)j * A.nB + e + A.B], q[j]);
            fd = fma_(t, t, fd);
        }
    }
    float pt[3], Rt[3][3];
    tl_load_target(A, e, i, pt, Rt);
    Pose<D> P;
    eval_pose<D, FAST, WEIGHTED, SpecT>(A.ch, q, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr);
    tl_store_normal<D>(A, P, s, e, fd);
}

// Kahan-compensated sum step (explicit intrinsics: the compiler cannot simplify the compensation away)
__device__ __forceinline__ void kahan_add(float &s, float &c, float x) {
    const float y = sub(x, c);
    const float t = add(s, y);
    c = sub(sub(t, s), y);
    s = t;
}

// total cost of buffer `s` of trajectory b, fixed order i = 0..n-1
__device__ __forceinline__ void tl_sum_cost(const TArgs &A, int s, int64_t b, float &Fp, float &Fd, float &F) {
    const float *cp = A.cst + (int64_t)s * 2 * A.nB + b;
    float sp = 0.f, cpp = 0.f, sd = 0.f, cd = 0.f;
    for (int i = 0; i < A.n; ++i) {
        kahan_add(sp, cpp, cp[(int64_t)i * A.B]);
        kahan_add(sd, cd, cp[A.nB + (int64_t)i * A.B]);
    }
    Fp = sp; Fd = sd;
    F = fma_(A.wd2, sd, mul(A.wp2, sp));
}

#ifdef LM_TRAJ_PLAIN_KERNELS // non-template kernels: defined in exactly one translation unit (lm_traj_api.cu)
// ---- cost of the current point (entry of lm_traj_run): thread per trajectory
__global__ void __launch_bounds__(128) tl_init_cost_kernel(const __grid_constant__ TArgs A) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= A.B) return;
    float Fp, Fd, F;
    tl_sum_cost(A, A.sel[b], b, Fp, Fd, F);
    A.Fp[b] = Fp; A.Fd[b] = Fd; A.F[b] = F;
}
#endif

// In-place symmetric sweep of the packed lower triangle S (SPD): returns W = -S^-1.
// Sweep k: p = 1/S_kk; S_ij -= S_ik S_jk p (i, j != k); S_ik *= p; S_kk = -p.  The diagonal entries
// not yet swept are the Schur complements (> 0 for an SPD matrix): ok = all pivots > 0.
template <int D>
__device__ __forceinline__ bool sweep_neg_inverse(float (&S)[Tri<D>::NA]) {
    bool ok = true;
#pragma unroll
    for (int k = 0; k < D; ++k) {
        const float piv = S[tri(k, k)];
        ok = ok && (piv > 0.f);
        const float p = __fdividef(1.0f, piv);
        float t[D];
#pragma unroll
        for (int i = 0; i < D; ++i) t[i] = S[tri(i, k)];
#pragma unroll
        for (int i = 0; i < D; ++i) {
            if (i == k) continue;
            const float tp = mul(t[i], p);
#pragma unroll
            for (int j = 0; j <= i; ++j) {
                if (j == k) continue;
                S[tri(i, j)] = fma_(-tp, t[j], S[tri(i, j)]);
            }
            S[tri(i, k)] = tp;
        }
        S[tri(k, k)] = -p;
    }
    return ok;
}

// y = M x for a packed symmetric M
template <int D>
__device__ __forceinline__ void symv(const float (&M)[Tri<D>::NA], const float (&x)[D], float (&y)[D]) {
#pragma unroll
    for (int r = 0; r < D; ++r) {
        float s = mul(M[tri(r, 0)], x[0]);
#pragma unroll
        for (int c = 1; c < D; ++c) s = fma_(M[tri(r, c)], x[c], s);
        y[r] = s;
    }
}

// ---- block-tridiagonal solve: thread per trajectory
//   mode 0: factor (stores W_i = -S_i^-1) and solve for g = gp + w_d^2 D^T D q;  delta  = -x
//   mode 1: re-solve with the stored W_i for rho (iterative refinement);          delta +=  x
template <int D>
__global__ void __launch_bounds__(128) tl_solve_kernel(const __grid_constant__ TArgs A) {
    constexpr int NA = Tri<D>::NA;
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= A.B) return;
    const uint32_t pk = A.its[b];
    if ((pk & 0xffu) >= (uint32_t)A.max_total) return;
    if (A.mode == 1 && !A.ok[b]) return;
    const int s = A.sel[b];
    const int n = A.n;
    const int64_t nB = A.nB, B = A.B;
    const float lam = A.lam[b];
    const float *Ab = A.A + (int64_t)s * NA * nB + b;
    const float *gb = A.gp + (int64_t)s * D * nB + b;
    const float *qb = A.q + (int64_t)s * D * nB + b;
    float *Vb = A.V + b, *zb = A.z + b, *db = A.delta + b;
    const float *rb = A.rho + b;

    float W[NA], zp[D];
#pragma unroll
    for (int t = 0; t < NA; ++t) W[t] = 0.f;
#pragma unroll
    for (int j = 0; j < D; ++j) zp[j] = 0.f;
    bool ok = true;

    // ---- forward elimination
    float qm[D], qc[D], qn[D];
    if (A.mode == 0) {
#pragma unroll
        for (int j = 0; j < D; ++j) { qm[j] = 0.f; qc[j] = qb[(int64_t)j * nB]; }
    }
    for (int i = 0; i < n; ++i) {
        const int64_t off = (int64_t)i * B;
        float rhs[D];
        if (A.mode == 0) {
            const float ci = (n == 1) ? 0.f : ((i == 0 || i == n - 1) ? 1.f : 2.f);
            const bool has_next = i + 1 < n;
#pragma unroll
            for (int j = 0; j < D; ++j) qn[j] = has_next ? qb[(int64_t)j * nB + off + B] : 0.f;
            float S[NA];
#pragma unroll
            for (int t = 0; t < NA; ++t) S[t] = Ab[(int64_t)t * nB + off];
            const float dg = fma_(ci, A.wd2, lam);
#pragma unroll
            for (int r = 0; r < D; ++r) {
                S[tri(r, r)] = add(S[tri(r, r)], dg);
                // g_i = gp_i + w_d^2 (c_i q_i - q_{i-1} - q_{i+1})
                const float dd = sub(sub(mul(ci, qc[r]), qm[r]), qn[r]);
                rhs[r] = fma_(A.wd2, dd, gb[(int64_t)r * nB + off]);
            }
            // S_i = T_i - w_d^4 S_{i-1}^-1 = T_i + w_d^4 W_{i-1}
#pragma unroll
            for (int t = 0; t < NA; ++t) S[t] = fma_(A.wd4, W[t], S[t]);
            ok = sweep_neg_inverse<D>(S) && ok;
#pragma unroll
            for (int t = 0; t < NA; ++t) { W[t] = S[t]; Vb[(int64_t)t * nB + off] = S[t]; }
#pragma unroll
            for (int j = 0; j < D; ++j) { qm[j] = qc[j]; qc[j] = qn[j]; }
        } else {
#pragma unroll
            for (int t = 0; t < NA; ++t) W[t] = Vb[(int64_t)t * nB + off];
#pragma unroll
            for (int r = 0; r < D; ++r) rhs[r] = rb[(int64_t)r * nB + off];
        }
        // h_i = rhs_i + w_d^2 z_{i-1};  z_i = S_i^-1 h_i = -(W_i h_i)
        float h[D], y[D];
#pragma unroll
        for (int r = 0; r < D; ++r) h[r] = fma_(A.wd2, zp[r], rhs[r]);
        symv<D>(W, h, y);
#pragma unroll
        for (int r = 0; r < D; ++r) { zp[r] = -y[r]; zb[(int64_t)r * nB + off] = zp[r]; }
    }

    // ---- back substitution: x_n = z_n, x_i = z_i + w_d^2 S_i^-1 x_{i+1} = z_i - w_d^2 W_i x_{i+1}
    float x[D];
#pragma unroll
    for (int j = 0; j < D; ++j) x[j] = 0.f;
    float asum = 0.f;
    for (int i = n - 1; i >= 0; --i) {
        const int64_t off = (int64_t)i * B;
        if (i == n - 1) {
#pragma unroll
            for (int r = 0; r < D; ++r) x[r] = zp[r]; // W, zp still hold waypoint n-1
        } else {
            float y[D];
#pragma unroll
            for (int t = 0; t < NA; ++t) W[t] = Vb[(int64_t)t * nB + off];
            symv<D>(W, x, y);
#pragma unroll
            for (int r = 0; r < D; ++r) x[r] = fma_(-A.wd2, y[r], zb[(int64_t)r * nB + off]);
        }
#pragma unroll
        for (int r = 0; r < D; ++r) {
            const float dv = (A.mode == 0) ? -x[r] : add(db[(int64_t)r * nB + off], x[r]);
            db[(int64_t)r * nB + off] = dv;
            asum = fmaxf(asum, fabsf(dv));
        }
    }
    ok = ok && (asum < 1e30f); // NaN compares false
    if (A.mode == 0) A.ok[b] = ok ? 1 : 0;
    else if (!ok) A.ok[b] = 0;
}

// ---- refinement residual (DESIGN R4 carried over to the stacked system): thread per waypoint
//   rho_i = -[ w_p^2 J_i^T (r_i + J_i delta_i) + w_d^2 (D^T D (q + delta))_i + lambda delta_i ]
template <int D, bool FAST, bool WEIGHTED, typename SpecT>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) tl_rho_kernel(const __grid_constant__ TArgs A) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.nB) return;
    const int64_t i = e / A.B, b = e - i * A.B;
    if ((A.its[b] & 0xffu) >= (uint32_t)A.max_total || !A.ok[b]) return;
    const int s = A.sel[b];
    const int64_t nB = A.nB;
    const float *qs = A.q + (int64_t)s * D * nB;
    const float lam = A.lam[b];
    const int n = A.n;
    const float ci = (n == 1) ? 0.f : ((i == 0 || i == n - 1) ? 1.f : 2.f);
    float q[D], dl[D], dd[D];
#pragma unroll
    for (int j = 0; j < D; ++j) {
        q[j] = qs[(int64_t)j * nB + e];
        dl[j] = A.delta[(int64_t)j * nB + e];
        const float yc = add(q[j], dl[j]);
        const float ym = (i > 0) ? add(qs[(int64_t)j * nB + e - A.B], A.delta[(int64_t)j * nB + e - A.B]) : 0.f;
        const float yn = (i + 1 < n) ? add(qs[(int64_t)j * nB + e + A.B], A.delta[(int64_t)j * nB + e + A.B]) : 0.f;
        dd[j] = sub(sub(mul(ci, yc), ym), yn);
    }
    float pt[3], Rt[3][3];
    tl_load_target(A, e, i, pt, Rt);
    Pose<D> P;
    eval_pose<D, FAST, WEIGHTED, SpecT>(A.ch, q, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr);
    float t[6];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        float sv = P.r[k], sw = P.r[3 + k];
#pragma unroll
        for (int j = 0; j < D; ++j) {
            sv = fma_(P.Jv[j][k], dl[j], sv);
            sw = fma_(P.Jw[j][k], dl[j], sw);
        }
        t[k] = sv; t[3 + k] = sw;
    }
#pragma unroll
    for (int j = 0; j < D; ++j) {
        const float acc = fma_(lam, dl[j], fma_(A.wd2, dd[j], mul(A.wp2, colvec<D>(P, j, t))));
        A.rho[(int64_t)j * nB + e] = -acc;
    }
}

// ---- trial point: q+ = clamp(q + delta), its cost terms and its normal equations
//      into the candidate buffer (1 - sel): thread per waypoint
template <int D, bool FAST, bool WEIGHTED, typename SpecT>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) tl_trial_kernel(const __grid_constant__ TArgs A) {
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= A.nB) return;
    const int64_t i = e / A.B, b = e - i * A.B;
    const uint32_t pk = A.its[b];
    if ((pk & 0xffu) >= (uint32_t)A.max_total) return;
    const int s = A.sel[b];
    const bool ok = A.ok[b] != 0;
    const int64_t nB = A.nB;
    const float *qs = A.q + (int64_t)s * D * nB;
    float *qd = A.q + (int64_t)(1 - s) * D * nB;
    float qt[D], fd = 0.f;
    bool clamped = false;
#pragma unroll
    for (int j = 0; j < D; ++j) {
        const float t = ok ? add(qs[(int64_t)j * nB + e], A.delta[(int64_t)j * nB + e]) : qs[(int64_t)j * nB + e];
        qt[j] = fminf(fmaxf(t, A.ch.lo[j]), A.ch.hi[j]);
        clamped = clamped || (qt[j] != t);
        qd[(int64_t)j * nB + e] = qt[j];
    }
    if (i + 1 < A.n) {
#pragma unroll
        for (int j = 0; j < D; ++j) {
            const float t = ok ? add(qs[(int64_t)j * nB + e + A.B], A.delta[(int64_t)j * nB + e + A.B]) : qs[(int64_t)j * nB + e + A.B];
            const float tn = fminf(fmaxf(t, A.ch.lo[j]), A.ch.hi[j]);
            const float df = sub(tn, qt[j]);
            fd = fma_(df, df, fd);
        }
    }
    if (clamped) atomicOr(A.its + b, 32u << 8); // "a trial point was clamped" (integer atomic: order-free)
    float pt[3], Rt[3][3];
    tl_load_target(A, e, i, pt, Rt);
    Pose<D> P;
    eval_pose<D, FAST, WEIGHTED, SpecT>(A.ch, qt, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr);
    tl_store_normal<D>(A, P, 1 - s, e, fd);
    if (A.trace_q != nullptr) {
        const int64_t w = b * A.n + i;
#pragma unroll
        for (int j = 0; j < D; ++j) A.trace_q[(int64_t)j * nB + w] = qt[j];
    }
}

#ifdef LM_TRAJ_PLAIN_KERNELS
// ---- accept / reject and the lambda update, per trajectory (DESIGN T3 = R5 on the total cost)
__global__ void __launch_bounds__(128) tl_decide_kernel(const __grid_constant__ TArgs A) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= A.B) return;
    uint32_t pk = A.its[b];
    uint32_t k = pk & 0xffu, st = pk >> 8;
    if (k >= (uint32_t)A.max_total) return;
    const int s = A.sel[b];
    const bool ok = A.ok[b] != 0;
    float Fp, Fd, Ft;
    tl_sum_cost(A, 1 - s, b, Fp, Fd, Ft);
    const float F = A.F[b];
    if (A.trace_F != nullptr) { A.trace_F[b] = F; A.trace_F[A.B + b] = Ft; }
    const bool finite = fabsf(Ft) < 3.0e38f;
    const bool accept = ok && finite && (Ft < F);
    if (!ok) st |= 4u;
    if (!finite) st |= 8u;
    const bool trial_clamped = (st & 32u) != 0;
    st &= ~32u;
    float lam = A.lam[b];
    if (accept) {
        if (trial_clamped) st |= 16u;
        lam = fmaxf(mul(lam, A.inv_nu_down), A.lambda_min);
        A.mask[b] |= 1ull << k;
        A.sel[b] = 1 - s;
        A.F[b] = Ft; A.Fp[b] = Fp; A.Fd[b] = Fd;
    } else {
        lam = fminf(mul(lam, A.nu_up), A.lambda_max);
    }
    A.lam[b] = lam;
    ++k;
    st &= ~2u;
    if (k >= (uint32_t)A.max_total) st |= 2u;
    A.its[b] = k | (st << 8);
}

__global__ void __launch_bounds__(256) tl_reset_kernel(const __grid_constant__ TArgs A, const float *lam_in, float lambda0) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= A.B) return;
    A.lam[b] = lam_in ? lam_in[b] : lambda0;
    A.its[b] = 0u;
    A.mask[b] = 0ull;
    A.sel[b] = 0;
    A.ok[b] = 0;
}
#endif

} // namespace lmk
