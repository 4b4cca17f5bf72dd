// lm_kernels.cuh -- the kernels of the batched LM hot path (sm_100a).
//
//   lm_iterate_kernel<D, FAST>  S0..S10: load -> [Jacobian -> normal equations -> Cholesky ->
//                               trial -> FK + residual -> accept / lambda -> freeze]* -> store.
//                               One thread per waypoint block, the whole iteration loop on the
//                               device, state in registers; lm_step and lm_run are the same
//                               kernel with different iteration limits.
//   lm_fk_kernel<D, FAST>       S1 only (targets for synthetic workloads, FK parity tests).
//   lm_traj_stats_kernel        per-trajectory converged flag / iteration count (integer only).
#pragma once
#include "lm_device.cuh"

namespace lmk {

struct KArgs {
    KChain ch;
    float lambda0, nu_up, inv_nu_down, lambda_min, lambda_max, tol2;
    float w_pos, w_rot, inv_w_pos, inv_w_rot;
    int32_t weighted, refine, variant; // variant: 0, LM_VAR_DUAL or LM_VAR_RPY
    int64_t W;              // waypoint blocks
    int32_t n;              // waypoints per trajectory
    int32_t shared_targets; // target index = w % n
    int32_t fresh;          // 1: state := (seeds, lambda0, 0 iters) instead of reading the state arrays
    int32_t max_total;      // stop when iters == max_total
    int32_t at_most;        // and after this many iterations in this launch
    const float *tp, *tq, *seeds;
    float *q, *lam, *res, *perr, *rerr; // state / outputs, SoA [.][W]
    uint32_t *its;                      // iters | status << 8
    unsigned long long *mask;
    float *trace_q, *trace_F;           // nullable debug trace
};

__device__ __forceinline__ void quat_to_cols(float w, float x, float y, float z, float (&Rt)[3][3]) {
    // DESIGN R11: re-normalise, then the textbook conversion; Rt[k] = k-th COLUMN of R_t
    const float n2 = fma_(z, z, fma_(y, y, fma_(x, x, mul(w, w))));
    const float inv = rsqrtf(n2);
    w = mul(w, inv); x = mul(x, inv); y = mul(y, inv); z = mul(z, inv);
    const float xx = mul(x, x), yy = mul(y, y), zz = mul(z, z);
    const float xy = mul(x, y), xz = mul(x, z), yz = mul(y, z);
    const float wx = mul(w, x), wy = mul(w, y), wz = mul(w, z);
    Rt[0][0] = fma_(-2.f, add(yy, zz), 1.f); Rt[1][0] = mul(2.f, sub(xy, wz));        Rt[2][0] = mul(2.f, add(xz, wy));
    Rt[0][1] = mul(2.f, add(xy, wz));        Rt[1][1] = fma_(-2.f, add(xx, zz), 1.f); Rt[2][1] = mul(2.f, sub(yz, wx));
    Rt[0][2] = mul(2.f, sub(xz, wy));        Rt[1][2] = mul(2.f, add(yz, wx));        Rt[2][2] = fma_(-2.f, add(xx, yy), 1.f);
}

// LM_PACKED_DELTA: which kernels take S4 + S5 through the packed FFMA2 form (lm_delta_p, same bits): 0 none, 1 the
// generic (run-time chain structure) kernels, 2 all.  Measured on C4 (profiles/r2_rf_model.md): generic 2.875 -> 2.807
// ms, Panda-specialised 2.064 -> 2.316 ms (the specialised scalar form skips the structural zeros of J; the packed
// form cannot, and register-file reads, not issue slots, are the limit), hence 1.
#ifndef LM_PACKED_DELTA
#define LM_PACKED_DELTA 1
#endif
#ifndef LM_MAX_THREADS
#define LM_MAX_THREADS 256
#endif
#ifndef LM_MIN_BLOCKS
#define LM_MIN_BLOCKS 1
#endif

// VAR: 0 = the d x d system with the rotation-vector residual (the hot path), LM_VAR_DUAL = the 6 x 6 dual form,
// LM_VAR_RPY = the roll-pitch-yaw residual (disclosed variants, DESIGN.md sections 12 and 14)
constexpr int LM_VAR_DUAL = 1, LM_VAR_RPY = 2;
// G: lanes per waypoint (1 = the product path; 2 / 4 = the lane-group form lm_delta_lg, LM_OPT_LANES_PER_WAYPOINT)
// HOT: the common configuration as compile-time constants -- exactly one refinement step (the default) and no debug
// trace -- launched whenever the context is in it (lm_launch.h); the same operations, 29 + 7 fewer instructions per
// iteration (the refinement loop's counter and branch, the trace test).
template <int D, bool FAST, bool WEIGHTED, typename SpecT, int VAR = 0, int G = 1, bool HOT = false>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) lm_iterate_kernel(const __grid_constant__ KArgs A) {
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t w = G == 1 ? tid : tid / G;
    const int gl = G == 1 ? 0 : (int)(threadIdx.x % G); // lane within the waypoint's group
    const bool live = w < A.W;
    const int64_t wc = live ? w : A.W - 1; // tail lanes shadow the last waypoint, never store
    const int64_t W = A.W;

    // ---- S0 load (SoA: consecutive lanes read consecutive 4-byte words => 128-byte lines)
    float q[D];
    float lam;
    uint32_t k, st;
    unsigned long long mask;
    if (A.fresh) {
#pragma unroll
        for (int j = 0; j < D; ++j) q[j] = __ldg(A.seeds + (int64_t)j * W + wc);
        lam = A.lambda0; k = 0; st = 0; mask = 0ull;
    } else {
#pragma unroll
        for (int j = 0; j < D; ++j) q[j] = A.q[(int64_t)j * W + wc];
        lam = A.lam[wc];
        const uint32_t pk = A.its[wc];
        k = pk & 0xffu;
        st = (pk >> 8) & ~(1u | 2u); // FROZEN / MAXITER are re-derived below
        mask = A.mask[wc];
    }
    float pt[3], Rt[3][3];
    {
        const int64_t Wt = A.shared_targets ? (int64_t)A.n : W;
        const int64_t wt = A.shared_targets ? (wc % A.n) : wc;
#pragma unroll
        for (int i = 0; i < 3; ++i) pt[i] = __ldg(A.tp + (int64_t)i * Wt + wt);
        quat_to_cols(__ldg(A.tq + wt), __ldg(A.tq + Wt + wt), __ldg(A.tq + 2 * Wt + wt), __ldg(A.tq + 3 * Wt + wt), Rt);
    }
    constexpr bool DUAL = VAR == LM_VAR_DUAL, RPY = VAR == LM_VAR_RPY;
    float trpy[3] = {0.f, 0.f, 0.f}; // roll, pitch, yaw of the target (Rt[k] = k-th column of R_t)
    if (RPY) {
        trpy[0] = atan2_full(Rt[1][2], Rt[2][2]);
        trpy[1] = atan2_full(-Rt[0][2], sqrtf(fma_(Rt[0][1], Rt[0][1], mul(Rt[0][0], Rt[0][0]))));
        trpy[2] = atan2_full(Rt[0][1], Rt[0][0]);
    }
    Pose<D> cur;
    eval_pose<D, FAST, WEIGHTED, SpecT, true, NoFrameSink, RPY>(A.ch, q, pt, Rt, A.w_pos, A.w_rot, cur, nullptr, nullptr, nullptr,
                                                                NoFrameSink(), trpy);

    // ---- S3..S9: the LM loop, entirely on the device.  A lane is `active` while it is not
    // frozen and has iterations left; the warp leaves the loop when no lane is active.
    uint32_t done = 0;
    while (true) {
        const bool active = (k < (uint32_t)A.max_total) && (done < (uint32_t)A.at_most) && !(cur.F < A.tol2);
        if (!__any_sync(0xffffffffu, active)) break;

        float delta[D];
        constexpr bool PACKED = LM_PACKED_DELTA == 2 || (LM_PACKED_DELTA == 1 && SpecT::spec.generic);
        bool ok;
        if constexpr (DUAL) ok = lm_delta_dual<D, WEIGHTED, SpecT>(cur, lam, delta);                // S4, S5 (variant)
        else if constexpr (G > 1) ok = lm_delta_lg<D, G>(cur, lam, A.refine, gl, delta);
        else if constexpr (PACKED) ok = lm_delta_p<D, WEIGHTED, SpecT, RPY>(cur, lam, A.refine, delta);
        else ok = lm_delta<D, WEIGHTED, SpecT, RPY, HOT ? 1 : -1>(cur, lam, A.refine, delta);        // S4, S5
        float qt[D];
        bool clamped = false;
#pragma unroll
        for (int j = 0; j < D; ++j) {                               // S6 (DESIGN R6)
            const float t = add(q[j], delta[j]);
            qt[j] = fminf(fmaxf(t, A.ch.lo[j]), A.ch.hi[j]);
            clamped = clamped || (qt[j] != t);
        }
        Pose<D> tri; // S7: FK + residual at the trial point; its Jacobian (S3) is formed only if the step is accepted
        float ptri[3];
        eval_pose<D, FAST, WEIGHTED, SpecT, false, NoFrameSink, RPY>(A.ch, qt, pt, Rt, A.w_pos, A.w_rot, tri, nullptr, nullptr, ptri,
                                                                     NoFrameSink(), trpy);

        if (!HOT && A.trace_q != nullptr && active && live && gl == 0) {
#pragma unroll
            for (int j = 0; j < D; ++j) A.trace_q[(int64_t)j * W + w] = qt[j];
            A.trace_F[w] = cur.F;
            A.trace_F[W + w] = tri.F;
        }

        // S8 (DESIGN R5): strict decrease accepts; NaN / inf trial cost compares false => reject
        const bool accept = active && ok && (tri.F < cur.F);
        if (active) {
            if (!ok) st |= 4u;
            if (!(fabsf(tri.F) < 3.0e38f)) st |= 8u;
            if (accept && clamped) st |= 16u;
            const float lam_acc = fmaxf(mul(lam, A.inv_nu_down), A.lambda_min);
            const float lam_rej = fminf(mul(lam, A.nu_up), A.lambda_max);
            lam = accept ? lam_acc : lam_rej;
            if (accept) mask |= 1ull << k;
            ++k;
            ++done;
        }
        if (accept) {
#pragma unroll
            for (int j = 0; j < D; ++j) q[j] = qt[j];
            finish_jacobian<D, WEIGHTED, SpecT, RPY>(A.ch, tri, ptri, A.w_pos, A.w_rot, cur); // S3 straight into the current state
#pragma unroll
            for (int i = 0; i < 6; ++i) cur.r[i] = tri.r[i];
            cur.F = tri.F;
        }
    }

    // ---- S10 store
    if (!live || gl != 0) return;
    const bool frozen = cur.F < A.tol2;
    if (frozen) st |= 1u;
    else if (k >= (uint32_t)A.max_total) st |= 2u;
#pragma unroll
    for (int j = 0; j < D; ++j) A.q[(int64_t)j * W + w] = q[j];
    A.lam[w] = lam;
    A.its[w] = k | (st << 8);
    A.mask[w] = mask;
    A.res[w] = sqrtf(cur.F);
    A.perr[w] = mul(sqrtf(fma_(cur.r[2], cur.r[2], fma_(cur.r[1], cur.r[1], mul(cur.r[0], cur.r[0])))), A.inv_w_pos);
    A.rerr[w] = mul(sqrtf(fma_(cur.r[5], cur.r[5], fma_(cur.r[4], cur.r[4], mul(cur.r[3], cur.r[3])))), A.inv_w_rot);
}

struct KFkArgs {
    KChain ch;
    int64_t count;
    const float *q;
    float *pos, *rot;
};

template <int D, bool FAST, typename SpecT>
__global__ void __launch_bounds__(256) lm_fk_kernel(const __grid_constant__ KFkArgs A) {
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= A.count) return;
    float q[D];
#pragma unroll
    for (int j = 0; j < D; ++j) q[j] = __ldg(A.q + (int64_t)j * A.count + w);
    const float pt[3] = {0.f, 0.f, 0.f};
    const float Rt[3][3] = {{1.f, 0.f, 0.f}, {0.f, 1.f, 0.f}, {0.f, 0.f, 1.f}};
    Pose<D> P;
    float p[3], R[3][3];
    eval_pose<D, FAST, false, SpecT>(A.ch, q, pt, Rt, 1.f, 1.f, P, p, R);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        A.pos[(int64_t)i * A.count + w] = p[i];
#pragma unroll
        for (int c = 0; c < 3; ++c) A.rot[(int64_t)(3 * i + c) * A.count + w] = R[i][c];
    }
}

template <int D>
struct GenericSpec { static constexpr ChainSpec spec = generic_spec(D); };

} // namespace lmk
