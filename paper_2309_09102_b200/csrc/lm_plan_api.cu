// lm_plan_api.cu -- C ABI of the non-stationary schedule with anytime bookkeeping (include/lm.h,
// lm_plan_*): pose-only phases (lm_iterate_kernel) alternate with single
// trajectory-level LM iterations (lm_traj.cuh); a per-trajectory kernel checks validity
// (PAPER.md:L45, L53), measures the trajectory and keeps the latest valid
// one.  The host only enqueues launches.
#include "lm_ctx.h"

#include <cmath>
#include <cstring>

using namespace lmk;

namespace {

constexpr int PLAN_THREADS = 128;

struct PLayout {
    size_t q_valid, clear, cur, len_valid, gate, first, records, valid, total, all;
};

PLayout make_playout(int d, int64_t B, int64_t n) {
    const size_t W = (size_t)B * (size_t)n;
    PLayout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    L.q_valid = take(4 * W * d);
    L.clear = take(4 * W);
    L.cur = take(4 * 6 * (size_t)B);
    L.len_valid = take(4 * (size_t)B);
    L.gate = take(4 * (size_t)B);
    L.first = take(4 * (size_t)B);
    L.records = take(4 * (size_t)B);
    L.valid = take((size_t)B);
    L.total = take(16);
    L.all = off;
    return L;
}

struct PArgs {
    int32_t dof, n;
    int64_t B, W;
    uint32_t prismatic_mask;
    float pos_tol, rot_tol, mjac_rev, mjac_pris, min_clearance;
    int32_t cycle, use_clear;
    const float *clear;        // [W] smallest capsule clearance per waypoint (use_clear)
    const float *q;            // [d][W] w-order, current joint values
    const float *perr, *rerr;  // [W] of the pose kernel's last launch
    float *q_valid, *cur, *len_valid;
    int32_t *gate, *first, *records;
    uint8_t *valid;
};

// One block per trajectory.  max is order-free; the length is summed in a fixed order (each thread
// its strided waypoints in order, then a fixed tree): it depends on n only.
__global__ void __launch_bounds__(PLAN_THREADS) plan_check_kernel(const PArgs A) {
    __shared__ float red[6][PLAN_THREADS];
    __shared__ int s_valid;
    const int64_t b = blockIdx.x;
    const int t = threadIdx.x;
    const int64_t w0 = b * A.n;
    float mpos = 0.f, mrot = 0.f, mrev = 0.f, mpris = 0.f, len = 0.f, mclr = 3.0e38f;
    for (int i = t; i < A.n; i += PLAN_THREADS) {
        if (A.use_clear) mclr = fminf(mclr, A.clear[w0 + i]);
        mpos = fmaxf(mpos, A.perr[w0 + i]);
        mrot = fmaxf(mrot, A.rerr[w0 + i]);
        if (i + 1 < A.n) {
            for (int j = 0; j < A.dof; ++j) {
                const float *qj = A.q + (int64_t)j * A.W + w0 + i;
                const float dq = fabsf(__fsub_rn(qj[1], qj[0]));
                len = __fadd_rn(len, dq);
                if ((A.prismatic_mask >> j) & 1u) mpris = fmaxf(mpris, dq);
                else mrev = fmaxf(mrev, dq);
            }
        }
    }
    red[0][t] = mpos; red[1][t] = mrot; red[2][t] = mrev; red[3][t] = mpris; red[4][t] = len; red[5][t] = mclr;
    __syncthreads();
    for (int s = PLAN_THREADS / 2; s > 0; s >>= 1) {
        if (t < s) {
            red[0][t] = fmaxf(red[0][t], red[0][t + s]);
            red[1][t] = fmaxf(red[1][t], red[1][t + s]);
            red[2][t] = fmaxf(red[2][t], red[2][t + s]);
            red[3][t] = fmaxf(red[3][t], red[3][t + s]);
            red[4][t] = __fadd_rn(red[4][t], red[4][t + s]);
            red[5][t] = fminf(red[5][t], red[5][t + s]);
        }
        __syncthreads();
    }
    if (t == 0) {
        mpos = red[0][0]; mrot = red[1][0]; mrev = red[2][0]; mpris = red[3][0]; len = red[4][0]; mclr = red[5][0];
        A.cur[b] = mpos; A.cur[A.B + b] = mrot; A.cur[2 * A.B + b] = mrev; A.cur[3 * A.B + b] = mpris; A.cur[4 * A.B + b] = len; A.cur[5 * A.B + b] = A.use_clear ? mclr : nanf("");
        const bool pose_ok = (mpos < A.pos_tol) && (mrot < A.rot_tol) && (len == len);
        const bool ok = pose_ok && (mrev <= A.mjac_rev) && (mpris <= A.mjac_pris) && (!A.use_clear || mclr >= A.min_clearance);
        A.gate[b] = pose_ok ? 1 : 0;
        if (ok) {
            if (!A.valid[b]) A.first[b] = A.cycle;
            A.valid[b] = 1;
            A.records[b] += 1;
            A.len_valid[b] = len;
        }
        s_valid = ok ? 1 : 0;
    }
    __syncthreads();
    if (!s_valid) return;
    for (int j = 0; j < A.dof; ++j)
        for (int i = t; i < A.n; i += PLAN_THREADS) A.q_valid[(int64_t)j * A.W + w0 + i] = A.q[(int64_t)j * A.W + w0 + i];
}

__global__ void plan_clear_kernel(PArgs A, float nanv) {
    const int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (x < A.W * A.dof) A.q_valid[x] = nanv;
    if (x < A.B) {
        A.gate[x] = 0; A.first[x] = -1; A.records[x] = 0; A.valid[x] = 0; A.len_valid[x] = nanv;
        for (int k = 0; k < 6; ++k) A.cur[k * A.B + x] = nanv;
    }
}

__global__ void plan_count_kernel(const uint8_t *valid, int64_t B, unsigned long long *total) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < B && valid[b]) atomicAdd(total, 1ull); // integer: order-free
}

PArgs plan_args(lm_ctx *c, int cycle) {
    const PlanState &p = c->plan;
    PArgs a{};
    a.dof = c->dof; a.n = (int32_t)c->n; a.B = c->B; a.W = c->W;
    a.prismatic_mask = c->args.ch.prismatic_mask;
    a.pos_tol = p.prm.pos_tol; a.rot_tol = p.prm.rot_tol; a.mjac_rev = p.prm.mjac_rev; a.mjac_pris = p.prm.mjac_pris;
    a.cycle = cycle;
    a.min_clearance = p.prm.min_clearance;
    a.use_clear = (c->traj.args.caps.npairs + c->traj.args.caps.nenv) > 0 ? 1 : 0;
    a.clear = p.clear;
    a.q = c->args.q; a.perr = c->args.perr; a.rerr = c->args.rerr;
    a.q_valid = p.q_valid; a.cur = p.cur; a.len_valid = p.len_valid;
    a.gate = p.gate; a.first = p.first; a.records = p.records; a.valid = p.valid;
    return a;
}

} // namespace

extern "C" {

size_t lm_plan_workspace_bytes(int32_t dof, int64_t B, int64_t n) {
    if (dof < 1 || dof > LM_MAX_DOF || B <= 0 || n <= 0) return 0;
    return make_playout(dof, B, n).all;
}

int lm_plan_default_params(lm_plan_params *out) {
    if (!out) return LM_EINVAL;
    const double deg = 3.14159265358979323846 / 180.0;
    out->pos_tol = 1e-4f;
    out->rot_tol = (float)(0.1 * deg);
    out->mjac_rev = (float)(7.0 * deg);
    out->mjac_pris = 0.02f;
    out->pose_iters = 10;
    out->min_clearance = 0.f;
    return LM_OK;
}

int lm_plan_attach(lm_ctx *c, const lm_plan_params *p, void *workspace, size_t bytes) {
    if (!c || !p || !workspace || !c->traj.attached) return LM_EINVAL;
    if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return LM_EINVAL;
    if (!(p->pos_tol > 0.f) || !(p->rot_tol > 0.f) || !(p->mjac_rev > 0.f) || !(p->mjac_pris > 0.f) ||
        p->pose_iters < 1 || p->pose_iters > LM_MAX_ITERS)
        return LM_EINVAL;
    const PLayout L = make_playout(c->dof, c->B, c->n);
    if (bytes < L.all) return LM_ENOMEM;
    PlanState &s = c->plan;
    s = PlanState{};
    s.prm = *p;
    s.ws = static_cast<char *>(workspace);
    s.q_valid = reinterpret_cast<float *>(s.ws + L.q_valid);
    s.cur = reinterpret_cast<float *>(s.ws + L.cur);
    s.clear = reinterpret_cast<float *>(s.ws + L.clear);
    s.len_valid = reinterpret_cast<float *>(s.ws + L.len_valid);
    s.gate = reinterpret_cast<int32_t *>(s.ws + L.gate);
    s.first = reinterpret_cast<int32_t *>(s.ws + L.first);
    s.records = reinterpret_cast<int32_t *>(s.ws + L.records);
    s.valid = reinterpret_cast<uint8_t *>(s.ws + L.valid);
    s.total = reinterpret_cast<unsigned long long *>(s.ws + L.total);
    s.attached = true;
    return LM_OK;
}

int lm_plan_run(lm_ctx *c, int32_t cycles) {
    if (!c || !c->plan.attached || !c->traj.attached || cycles < 0 || cycles > LM_MAX_ITERS) return LM_EINVAL;
    int rc = materialize_state(c);
    if (rc != LM_OK) return rc;
    rc = lm_traj_reset(c, nullptr);
    if (rc != LM_OK) return rc;
    {
        const PArgs a = plan_args(c, 0);
        const int64_t items = (c->W * c->dof > c->B) ? c->W * c->dof : c->B;
        launch_counter().fetch_add(1);
        plan_clear_kernel<<<(unsigned)((items + 255) / 256), 256, 0, c->stream>>>(a, nanf(""));
        LM_CUDA(cudaGetLastError());
    }
    for (int cyc = 0; cyc <= cycles; ++cyc) {
        // pose-only phase from fresh per-waypoint LM state (reading P1)
        rc = reset_waypoint_lm_state(c);
        if (rc != LM_OK) return rc;
        rc = run_pose_phase(c, c->plan.prm.pose_iters);
        if (rc != LM_OK) return rc;
        // validity, measurements, latest valid solution (P3); with capsules set, the smallest clearance per waypoint first
        if ((c->traj.args.caps.npairs + c->traj.args.caps.nenv) > 0) {
            rc = launch_clearance(c, c->plan.clear);
            if (rc != LM_OK) return rc;
        }
        launch_counter().fetch_add(1);
        plan_check_kernel<<<(unsigned)c->B, PLAN_THREADS, 0, c->stream>>>(plan_args(c, cyc));
        LM_CUDA(cudaGetLastError());
        if (cyc == cycles) break;
        // one trajectory-level iteration for the pose-valid trajectories (P2)
        c->traj.args.gate = c->plan.gate;
        rc = lm_traj_run(c, 1);
        c->traj.args.gate = nullptr;
        if (rc != LM_OK) return rc;
    }
    return LM_OK;
}

int lm_plan_fetch(lm_ctx *c, float *q_valid_out, lm_plan_stats *s) {
    if (!c || !c->plan.attached) return LM_EINVAL;
    const PlanState &p = c->plan;
    const size_t B = (size_t)c->B;
    auto out = [&](void *dst, const void *src, size_t bytes) -> cudaError_t {
        return dst ? cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDefault, c->stream) : cudaSuccess;
    };
    LM_CUDA(out(q_valid_out, p.q_valid, 4 * (size_t)c->W * c->dof));
    unsigned long long h = 0;
    if (s) {
        LM_CUDA(out(s->valid, p.valid, B));
        LM_CUDA(out(s->first_valid_cycle, p.first, 4 * B));
        LM_CUDA(out(s->records, p.records, 4 * B));
        LM_CUDA(out(s->length, p.len_valid, 4 * B));
        LM_CUDA(out(s->max_pos_err, p.cur, 4 * B));
        LM_CUDA(out(s->max_rot_err, p.cur + B, 4 * B));
        LM_CUDA(out(s->mjac_rev, p.cur + 2 * B, 4 * B));
        LM_CUDA(out(s->mjac_pris, p.cur + 3 * B, 4 * B));
        LM_CUDA(out(s->cur_length, p.cur + 4 * B, 4 * B));
        LM_CUDA(out(s->min_clearance, p.cur + 5 * B, 4 * B));
        LM_CUDA(cudaMemsetAsync(p.total, 0, 16, c->stream));
        launch_counter().fetch_add(1);
        plan_count_kernel<<<(unsigned)((B + 255) / 256), 256, 0, c->stream>>>(p.valid, c->B, p.total);
        LM_CUDA(cudaGetLastError());
        LM_CUDA(cudaMemcpyAsync(&h, p.total, 8, cudaMemcpyDeviceToHost, c->stream));
    }
    LM_CUDA(cudaStreamSynchronize(c->stream));
    if (s) s->valid_trajectories = (int64_t)h;
    return LM_OK;
}

} // extern "C"
