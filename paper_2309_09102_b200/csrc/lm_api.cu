// lm_api.cu -- C ABI of include/lm.h: validation, workspace carving, launches.  No torch types,
// no CPU compute path: every step of the hot path runs in the kernels of lm_kernels.cuh.
#include "lm_ctx.h"
#include "lm_launch.h"

#include <climits>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

using namespace lmk;

namespace {

thread_local char g_cuda_err[256] = "no CUDA error recorded";
std::atomic<long long> g_launches{0};

Layout make_layout(int dof, int64_t B, int64_t n, int shared, int memory) {
    const size_t W = (size_t)B * (size_t)n, Wt = shared ? (size_t)n : W;
    Layout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    L.q = take(4 * W * dof);
    L.lam = take(4 * W);
    L.res = take(4 * W);
    L.perr = take(4 * W);
    L.rerr = take(4 * W);
    L.its = take(4 * W);
    L.mask = take(8 * W);
    L.ui = take(4 * W); // unpacked iters / status for host destinations of lm_fetch
    L.us = take(4 * W);
    L.conv = take((size_t)B);
    L.titers = take(4 * (size_t)B);
    L.totals = take(16);
    if (memory == LM_MEM_HOST) {
        L.s_seeds = take(4 * W * dof);
        L.s_tp = take(4 * Wt * 3);
        L.s_tq = take(4 * Wt * 4);
    }
    L.total = off;
    return L;
}

float round_inward(double x, bool lower) { // fp32 value inside [lo, hi] of the fp64 limits
    float f = (float)x;
    if (lower && (double)f < x) f = nextafterf(f, INFINITY);
    if (!lower && (double)f > x) f = nextafterf(f, -INFINITY);
    return f;
}

// Structure of a run-time chain in the canonical form of lm_specs.cuh (prismatic joints carry
// the d0 / t0 bits: neither offset is used on that path).
ChainSpec chain_signature(int d, const KChain &k) {
    ChainSpec s{false, d, 0, 0, 0, 0, 0, 0, 0, k.tool_has_rot != 0, 0};
    for (int j = 0; j < d; ++j) {
        const uint32_t b = 1u << j;
        const bool pris = (k.prismatic_mask & b) != 0;
        if (pris) s.pris |= b;
        if (k.ca[j] == 1.f && k.sa[j] == 0.f) s.al0 |= b;
        if (k.ca[j] == 0.f && k.sa[j] == 1.f) s.alp |= b;
        if (k.ca[j] == 0.f && k.sa[j] == -1.f) s.aln |= b;
        if (k.a[j] == 0.f) s.a0 |= b;
        if (k.d[j] == 0.f || pris) s.d0 |= b;
        if (k.toff[j] == 0.f || pris) s.t0 |= b;
    }
    for (int i = 0; i < 3; ++i)
        if (k.tool_p[i] == 0.f) s.tp0 |= 1u << i;
    return s;
}

int match_spec(const ChainSpec &s) {
    for (int id = 1; id < SPEC_COUNT; ++id) {
        const ChainSpec *r = registered_spec(id);
        if (r && r->dof == s.dof && r->pris == s.pris && r->al0 == s.al0 && r->alp == s.alp && r->aln == s.aln &&
            r->a0 == s.a0 && r->d0 == s.d0 && r->t0 == s.t0 && r->tool_rot == s.tool_rot && r->tp0 == s.tp0)
            return id;
    }
    return SPEC_GENERIC;
}

} // namespace

namespace lmk {
int cuda_fail(cudaError_t e) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    return LM_ECUDA;
}
std::atomic<long long> &launch_counter() { return g_launches; }
} // namespace lmk

extern "C" {

size_t lm_workspace_bytes(int32_t dof, int64_t B, int64_t n, int32_t shared_targets, int32_t memory) {
    if (dof < 1 || dof > LM_MAX_DOF || B <= 0 || n <= 0) return 0;
    return make_layout(dof, B, n, shared_targets, memory).total;
}

int lm_default_params(lm_params *out) {
    if (!out) return LM_EINVAL;
    out->lambda0 = 1e-3f;
    out->nu_up = 10.f;
    out->nu_down = 10.f;
    out->lambda_min = 1e-4f;
    out->lambda_max = 1e7f;
    out->tol = 0.f;
    out->w_pos = 1.f;
    out->w_rot = 1.f;
    out->refine_steps = 1;
    out->fast_sincos = 0;
    out->solver = LM_SOLVER_PRIMAL;
    out->rot_residual = LM_ROT_LOG;
    return LM_OK;
}

int lm_init(lm_ctx **out, const lm_chain *chain, const lm_problem *pb, const lm_params *prm, void *cuda_stream) {
    if (!out) return LM_EINVAL;
    *out = nullptr;
    if (!chain || !pb || !prm) return LM_EINVAL;
    const int d = chain->dof;
    if (d < 1 || d > LM_MAX_DOF) return LM_EINVAL;
    if (!chain->joint_type || !chain->dh || !chain->q_lo || !chain->q_hi) return LM_EINVAL;
    if (pb->B <= 0 || pb->n <= 0 || pb->n > INT32_MAX) return LM_EINVAL;
    if (!pb->target_pos || !pb->target_quat || !pb->seeds || !pb->workspace) return LM_EINVAL;
    if (pb->memory != LM_MEM_DEVICE && pb->memory != LM_MEM_HOST) return LM_EINVAL;
    if ((reinterpret_cast<uintptr_t>(pb->workspace) & 255u) != 0) return LM_EINVAL;
    if (pb->memory == LM_MEM_DEVICE && !(aligned16(pb->target_pos) && aligned16(pb->target_quat) && aligned16(pb->seeds)))
        return LM_EINVAL;
    if (!(prm->lambda0 > 0.f) || !(prm->nu_up > 1.f) || !(prm->nu_down > 1.f) || !(prm->lambda_min > 0.f) ||
        !(prm->lambda_max >= prm->lambda_min) || !(prm->tol >= 0.f) || !(prm->w_pos > 0.f) || !(prm->w_rot > 0.f) ||
        prm->refine_steps < 0 || prm->refine_steps > 2 || (prm->solver != LM_SOLVER_PRIMAL && prm->solver != LM_SOLVER_DUAL) ||
        (prm->rot_residual != LM_ROT_LOG && prm->rot_residual != LM_ROT_RPY) ||
        (prm->solver == LM_SOLVER_DUAL && prm->rot_residual == LM_ROT_RPY))
        return LM_EINVAL;
    for (int j = 0; j < d; ++j) {
        if (!(chain->q_lo[j] <= chain->q_hi[j])) return LM_EINVAL;
        if (chain->joint_type[j] > 1) return LM_EINVAL;
    }
    const double *tq = chain->tool + 3;
    const double tn = std::sqrt(tq[0] * tq[0] + tq[1] * tq[1] + tq[2] * tq[2] + tq[3] * tq[3]);
    if (!(tn > 0.0)) return LM_EINVAL;

    const Layout lay = make_layout(d, pb->B, pb->n, pb->shared_targets, pb->memory);
    if (pb->workspace_bytes < lay.total) return LM_ENOMEM;

    lm_ctx *c = new (std::nothrow) lm_ctx();
    if (!c) return LM_ENOMEM;
    c->dof = d; c->B = pb->B; c->n = pb->n; c->W = pb->B * pb->n; c->shared = pb->shared_targets ? 1 : 0;
    c->lay = lay; c->ws = static_cast<char *>(pb->workspace);
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->fresh = true; c->stale = false; c->block = 128; c->fast = prm->fast_sincos != 0;

    KArgs &a = c->args;
    std::memset(&a, 0, sizeof(a));
    KChain &k = a.ch;
    for (int j = 0; j < d; ++j) {
        const double aj = chain->dh[4 * j + 0], al = chain->dh[4 * j + 1], dj = chain->dh[4 * j + 2], th = chain->dh[4 * j + 3];
        // exact 0 / +-1 for the quarter-turn twists every standard DH table uses
        double ca = std::cos(al), sa = std::sin(al);
        if (std::fabs(ca) < 1e-15) ca = 0.0;
        if (std::fabs(sa) < 1e-15) sa = 0.0;
        k.ca[j] = (float)ca; k.sa[j] = (float)sa; k.a[j] = (float)aj; k.d[j] = (float)dj;
        k.toff[j] = (float)th; k.cth[j] = (float)std::cos(th); k.sth[j] = (float)std::sin(th);
        k.lo[j] = round_inward(chain->q_lo[j], true);
        k.hi[j] = round_inward(chain->q_hi[j], false);
        if (k.lo[j] > k.hi[j]) k.lo[j] = k.hi[j] = (float)chain->q_lo[j];
        if (chain->joint_type[j]) k.prismatic_mask |= 1u << j;
    }
    {
        const double w = tq[0] / tn, x = tq[1] / tn, y = tq[2] / tn, z = tq[3] / tn;
        const double R[9] = {1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y),
                             2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x),
                             2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)};
        bool ident = true;
        for (int i = 0; i < 9; ++i) {
            k.tool_R[i] = (float)R[i];
            if (std::fabs(R[i] - ((i % 4 == 0) ? 1.0 : 0.0)) > 0.0) ident = false;
        }
        k.tool_has_rot = ident ? 0u : 1u;
        for (int i = 0; i < 3; ++i) k.tool_p[i] = (float)chain->tool[i];
    }
    c->sig = chain_signature(d, k);
    c->spec_id = match_spec(c->sig);
    c->jit_fn = nullptr;
    c->jit_hot = false;
    c->use_generic = false;
    c->lanes = 1;
    a.lambda0 = prm->lambda0; a.nu_up = prm->nu_up; a.inv_nu_down = (float)(1.0 / (double)prm->nu_down);
    a.lambda_min = prm->lambda_min; a.lambda_max = prm->lambda_max; a.tol2 = prm->tol * prm->tol;
    a.w_pos = prm->w_pos; a.w_rot = prm->w_rot;
    a.inv_w_pos = (float)(1.0 / (double)prm->w_pos); a.inv_w_rot = (float)(1.0 / (double)prm->w_rot);
    a.weighted = (prm->w_pos != 1.f || prm->w_rot != 1.f) ? 1 : 0;
    a.refine = prm->refine_steps;
    a.variant = prm->solver == LM_SOLVER_DUAL ? LM_VAR_DUAL : (prm->rot_residual == LM_ROT_RPY ? LM_VAR_RPY : 0);
    a.W = c->W; a.n = (int32_t)c->n; a.shared_targets = c->shared;
    a.q = reinterpret_cast<float *>(c->ws + lay.q);
    a.lam = reinterpret_cast<float *>(c->ws + lay.lam);
    a.res = reinterpret_cast<float *>(c->ws + lay.res);
    a.perr = reinterpret_cast<float *>(c->ws + lay.perr);
    a.rerr = reinterpret_cast<float *>(c->ws + lay.rerr);
    a.its = reinterpret_cast<uint32_t *>(c->ws + lay.its);
    a.mask = reinterpret_cast<unsigned long long *>(c->ws + lay.mask);

    if (pb->memory == LM_MEM_HOST) {
        const size_t W = (size_t)c->W, Wt = c->shared ? (size_t)c->n : W;
        float *s = reinterpret_cast<float *>(c->ws + lay.s_seeds);
        float *tp = reinterpret_cast<float *>(c->ws + lay.s_tp);
        float *tqd = reinterpret_cast<float *>(c->ws + lay.s_tq);
        cudaError_t e = cudaMemcpyAsync(s, pb->seeds, 4 * W * d, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(tp, pb->target_pos, 4 * Wt * 3, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(tqd, pb->target_quat, 4 * Wt * 4, cudaMemcpyHostToDevice, c->stream);
        if (e != cudaSuccess) { delete c; return cuda_fail(e); }
        a.seeds = s; a.tp = tp; a.tq = tqd;
    } else {
        a.seeds = pb->seeds; a.tp = pb->target_pos; a.tq = pb->target_quat;
    }
    *out = c;
    return LM_OK;
}

} // extern "C"

namespace {

cudaError_t launch_iterate(lm_ctx *c, const KArgs &a) {
    g_launches.fetch_add(1);
    const bool weighted = a.weighted != 0;
    if (c->lanes > 1) { // lane-group form: validated by lm_set_option, re-checked here because the parameters can change after it
        if (c->spec_id == SPEC_GENERIC || c->use_generic || c->fast || weighted || a.variant != 0) return cudaErrorInvalidValue;
        const unsigned grid_lg = (unsigned)((c->W * c->lanes + c->block - 1) / c->block);
        return launch_iterate_lanegroup(c->spec_id, c->lanes, grid_lg, c->block, c->stream, a);
    }
    const unsigned grid = (unsigned)((c->W + c->block - 1) / c->block);
    if (c->jit_fn && !c->use_generic && (!c->jit_hot || (a.refine == 1 && a.trace_q == nullptr))) // lm_specialize
        return jit_launch(c->jit_fn, grid, c->block, c->stream, a);
    if (c->spec_id != SPEC_GENERIC && !c->use_generic)
        return launch_iterate_spec(c->spec_id, c->fast, weighted, grid, c->block, c->stream, a);
    return c->dof <= 4 ? launch_iterate_generic_lo(c->dof, c->fast, weighted, grid, c->block, c->stream, a)
                       : launch_iterate_generic_hi(c->dof, c->fast, weighted, grid, c->block, c->stream, a);
}

int iterate(lm_ctx *c, int max_total, int at_most) {
    KArgs a = c->args;
    a.fresh = c->fresh ? 1 : 0;
    a.max_total = max_total;
    a.at_most = at_most;
    cudaError_t e = launch_iterate(c, a);
    if (e != cudaSuccess) return cuda_fail(e);
    c->fresh = false;
    c->stale = false; // every launch re-evaluates |r|, the errors and the frozen flag at the state it loads
    return LM_OK;
}

} // namespace

namespace lmk {
int materialize_state(lm_ctx *c) { return c->fresh ? iterate(c, 0, 0) : LM_OK; }
int refresh_waypoint_outputs(lm_ctx *c) { return iterate(c, LM_MAX_ITERS, 0); }
int run_pose_phase(lm_ctx *c, int max_iters) { return iterate(c, max_iters, INT_MAX); }
} // namespace lmk

namespace {

// copy `bytes` from a device workspace array to a device-or-host destination (UVA decides)
cudaError_t copy_out(void *dst, const void *src, size_t bytes, cudaStream_t s) {
    if (!dst) return cudaSuccess;
    return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDefault, s);
}

// One warp per trajectory: converged = AND of frozen bits, iters = MAX, total = SUM (integers only,
// so the atomics below cannot disturb bit-stability).
__global__ void lm_traj_stats_kernel(const uint32_t *__restrict__ its, int64_t B, int32_t n,
                                     uint8_t *__restrict__ conv, int32_t *__restrict__ titers,
                                     unsigned long long *__restrict__ totals) {
    const int64_t b = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (b >= B) return;
    uint32_t all = 1u, mx = 0u;
    unsigned long long sum = 0ull;
    for (int i = lane; i < n; i += 32) {
        const uint32_t pk = its[b * n + i];
        all &= (pk >> 8) & 1u;
        mx = max(mx, pk & 0xffu);
        sum += pk & 0xffu;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        all &= __shfl_xor_sync(0xffffffffu, all, o);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
    }
    if (lane == 0) {
        conv[b] = (uint8_t)all;
        titers[b] = (int32_t)mx;
        atomicAdd(totals, sum);
        if (all) atomicAdd(totals + 1, 1ull);
    }
}

// FP32 FMA-pipe ceiling of this device, measured: 16 independent FFMA chains per thread, nothing
// else in the loop.  Used by bench.py as the measured counterpart of the derived ALU peak.
__global__ void __launch_bounds__(256) lm_fma_peak_kernel(float *out, int iters, float a, float b) {
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = __fmaf_rn(x[i], a, b);
    }
    float sum = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) sum += x[i];
    if (sum == 12345.678f) out[0] = sum; // never true: keeps the chains alive
}

__global__ void lm_unpack_kernel(const uint32_t *__restrict__ its, int64_t W, int32_t *__restrict__ iters,
                                 uint32_t *__restrict__ status) {
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= W) return;
    const uint32_t pk = its[w];
    if (iters) iters[w] = (int32_t)(pk & 0xffu);
    if (status) status[w] = pk >> 8;
}

__global__ void lm_fill_state_kernel(float *__restrict__ lam, uint32_t *__restrict__ its,
                                     unsigned long long *__restrict__ mask, int64_t W, float lambda0, int set_lam) {
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= W) return;
    if (set_lam) lam[w] = lambda0;
    its[w] = 0u;
    mask[w] = 0ull;
}

} // namespace

extern "C" {

int lm_step(lm_ctx *c) {
    if (!c) return LM_EINVAL;
    return iterate(c, LM_MAX_ITERS, 1);
}

int lm_run(lm_ctx *c, int32_t max_iters) {
    if (!c || max_iters < 0 || max_iters > LM_MAX_ITERS) return LM_EINVAL;
    return iterate(c, max_iters, INT_MAX);
}

int lm_reset(lm_ctx *c) {
    if (!c) return LM_EINVAL;
    c->fresh = true;
    return LM_OK;
}

int lm_set_trace(lm_ctx *c, float *trial_q, float *trial_F) {
    if (!c || ((trial_q == nullptr) != (trial_F == nullptr))) return LM_EINVAL;
    c->args.trace_q = trial_q;
    c->args.trace_F = trial_F;
    return LM_OK;
}

int lm_set_option(lm_ctx *c, int32_t option, int32_t value) {
    if (!c) return LM_EINVAL;
    switch (option) {
    case LM_OPT_BLOCK_THREADS:
        if (value == 0) value = 128;
        if (value < 32 || value > 256 || (value % 32) != 0) return LM_EINVAL;
        c->block = value;
        return LM_OK;
    case LM_OPT_GENERIC_KERNEL:
        if (value != 0 && c->lanes > 1) return LM_EINVAL;
        c->use_generic = value != 0;
        return LM_OK;
    case LM_OPT_TRAJ_COST_LANES:
        if (value < 0 || value > 2 || !c->traj.attached) return LM_EINVAL;
        c->traj.cost_lanes = value;
        return LM_OK;
    case LM_OPT_TRAJ_FUSED:
        if (value < 0 || value > 2 || !c->traj.attached) return LM_EINVAL;
        c->traj.fused_mode = value;
        return LM_OK;
    case LM_OPT_LANES_PER_WAYPOINT:
        if (value != 1 && value != 2 && value != 4) return LM_EINVAL;
        if (value > 1 && (c->spec_id == SPEC_GENERIC || c->use_generic || c->fast || c->args.weighted || c->args.variant != 0))
            return LM_EINVAL;
        c->lanes = value;
        return LM_OK;
    default:
        return LM_EINVAL;
    }
}

const char *lm_kernel_name(lm_ctx *c) {
    if (!c) return "";
    if (c->jit_fn && !c->use_generic && (!c->jit_hot || (c->args.refine == 1 && c->args.trace_q == nullptr))) return "jit";
    return (c->spec_id != SPEC_GENERIC && !c->use_generic) ? spec_name(c->spec_id) : "generic";
}

int lm_specialize(lm_ctx *c) {
    if (!c) return LM_EINVAL;
    if (c->spec_id != SPEC_GENERIC || c->jit_fn) return LM_OK; // an ahead-of-time kernel (or an earlier call) already serves this chain
    void *fn = nullptr;
    const bool hot = !c->fast && c->args.variant == 0 && c->args.refine == 1;
    const int rc = jit_get_kernel(c->sig, c->fast, c->args.weighted != 0, c->args.variant, hot, &fn);
    if (rc == LM_EINVAL) snprintf(g_cuda_err, sizeof(g_cuda_err), "lm_specialize: %s", jit_last_log());
    if (rc != LM_OK) return rc == LM_EINVAL ? LM_ECUDA : rc; // the reason is in lm_strerror(LM_ECUDA)
    c->jit_fn = fn;
    c->jit_hot = hot;
    return LM_OK;
}

int lm_set_state(lm_ctx *c, const float *q, const float *lambda) {
    if (!c || !q) return LM_EINVAL;
    const size_t W = (size_t)c->W;
    LM_CUDA(cudaMemcpyAsync(c->args.q, q, 4 * W * c->dof, cudaMemcpyDefault, c->stream));
    if (lambda) LM_CUDA(cudaMemcpyAsync(c->args.lam, lambda, 4 * W, cudaMemcpyDefault, c->stream));
    const unsigned grid = (unsigned)((W + 255) / 256);
    g_launches.fetch_add(1);
    lm_fill_state_kernel<<<grid, 256, 0, c->stream>>>(c->args.lam, c->args.its, c->args.mask, c->W,
                                                      c->args.lambda0, lambda ? 0 : 1);
    LM_CUDA(cudaGetLastError());
    c->fresh = false;
    c->stale = true; // res_norm / pos_err / rot_err / status still describe the previous q: lm_fetch re-evaluates them
    return LM_OK;
}

} // extern "C"

namespace lmk {
int reset_waypoint_lm_state(lm_ctx *c) {
    const unsigned grid = (unsigned)((c->W + 255) / 256);
    g_launches.fetch_add(1);
    lm_fill_state_kernel<<<grid, 256, 0, c->stream>>>(c->args.lam, c->args.its, c->args.mask, c->W, c->args.lambda0, 1);
    LM_CUDA(cudaGetLastError());
    return LM_OK;
}
} // namespace lmk

extern "C" {

int lm_fk(lm_ctx *c, const float *q, int64_t count, float *pos, float *rot) {
    if (!c || !q || !pos || !rot || count <= 0) return LM_EINVAL;
    if (!(aligned16(q) && aligned16(pos) && aligned16(rot))) return LM_EINVAL;
    KFkArgs a;
    a.ch = c->args.ch; a.count = count; a.q = q; a.pos = pos; a.rot = rot;
    g_launches.fetch_add(1);
    const unsigned grid = (unsigned)((count + 127) / 128);
    cudaError_t e = (c->spec_id != SPEC_GENERIC && !c->use_generic)
                        ? launch_fk_spec(c->spec_id, c->fast, grid, 128, c->stream, a)
                        : launch_fk_generic(c->dof, c->fast, grid, 128, c->stream, a);
    if (e != cudaSuccess) return cuda_fail(e);
    return LM_OK;
}

int lm_fetch(lm_ctx *c, float *q_out, lm_stats *s) {
    if (!c) return LM_EINVAL;
    const size_t W = (size_t)c->W;
    const KArgs &a = c->args;
    if (c->fresh) { // nothing has run yet: materialise the initial state so that fetch is well defined
        int rc = iterate(c, 0, 0);
        if (rc != LM_OK) return rc;
    } else if (c->stale) { // lm_set_state and nothing since: a zero-iteration launch evaluates the outputs at the injected q
        int rc = iterate(c, LM_MAX_ITERS, 0);
        if (rc != LM_OK) return rc;
    }
    LM_CUDA(copy_out(q_out, a.q, 4 * W * c->dof, c->stream));
    if (s) {
        LM_CUDA(copy_out(s->res_norm, a.res, 4 * W, c->stream));
        LM_CUDA(copy_out(s->pos_err, a.perr, 4 * W, c->stream));
        LM_CUDA(copy_out(s->rot_err, a.rerr, 4 * W, c->stream));
        LM_CUDA(copy_out(s->lambda, a.lam, 4 * W, c->stream));
        LM_CUDA(copy_out(s->accept_mask, a.mask, 8 * W, c->stream));
        uint8_t *conv = reinterpret_cast<uint8_t *>(c->ws + c->lay.conv);
        int32_t *tit = reinterpret_cast<int32_t *>(c->ws + c->lay.titers);
        unsigned long long *tot = reinterpret_cast<unsigned long long *>(c->ws + c->lay.totals);
        LM_CUDA(cudaMemsetAsync(tot, 0, 16, c->stream));
        const int64_t threads = c->B * 32;
        g_launches.fetch_add(1);
        lm_traj_stats_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, c->stream>>>(a.its, c->B, (int32_t)c->n, conv, tit, tot);
        LM_CUDA(cudaGetLastError());
        LM_CUDA(copy_out(s->traj_converged, conv, (size_t)c->B, c->stream));
        LM_CUDA(copy_out(s->traj_iters, tit, 4 * (size_t)c->B, c->stream));
        if (s->iters || s->status) {
            // unpack iters | status << 8 into the caller's arrays; host destinations go through scratch
            cudaPointerAttributes pa;
            int32_t *di = s->iters;
            uint32_t *ds = s->status;
            bool host_i = false, host_s = false;
            if (di) { LM_CUDA(cudaPointerGetAttributes(&pa, di)); host_i = (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged); }
            if (ds) { LM_CUDA(cudaPointerGetAttributes(&pa, ds)); host_s = (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged); }
            int32_t *ki = di ? (host_i ? reinterpret_cast<int32_t *>(c->ws + c->lay.ui) : di) : nullptr;
            uint32_t *ks = ds ? (host_s ? reinterpret_cast<uint32_t *>(c->ws + c->lay.us) : ds) : nullptr;
            g_launches.fetch_add(1);
            lm_unpack_kernel<<<(unsigned)((W + 255) / 256), 256, 0, c->stream>>>(a.its, c->W, ki, ks);
            LM_CUDA(cudaGetLastError());
            if (host_i) LM_CUDA(cudaMemcpyAsync(di, ki, 4 * W, cudaMemcpyDeviceToHost, c->stream));
            if (host_s) LM_CUDA(cudaMemcpyAsync(ds, ks, 4 * W, cudaMemcpyDeviceToHost, c->stream));
        }
        unsigned long long h[2] = {0, 0};
        LM_CUDA(cudaMemcpyAsync(h, tot, 16, cudaMemcpyDeviceToHost, c->stream));
        LM_CUDA(cudaStreamSynchronize(c->stream));
        s->total_waypoint_iters = (int64_t)h[0];
        s->converged_trajectories = (int64_t)h[1];
        return LM_OK;
    }
    LM_CUDA(cudaStreamSynchronize(c->stream));
    return LM_OK;
}

namespace {
// trajectories [b0, b1) of chunk k when B trajectories are split into `chunks` nearly equal parts
inline void chunk_range(int64_t B, int chunks, int k, int64_t &b0, int64_t &b1) {
    b0 = B * k / chunks;
    b1 = B * (k + 1) / chunks;
}
} // namespace

size_t lm_solve_host_workspace_bytes(int32_t dof, int64_t B, int64_t n, int32_t chunks) {
    if (dof < 1 || dof > LM_MAX_DOF || B <= 0 || n <= 0 || chunks < 1 || chunks > B) return 0;
    size_t total = 0;
    for (int k = 0; k < chunks; ++k) {
        int64_t b0, b1;
        chunk_range(B, chunks, k, b0, b1);
        total += make_layout(dof, b1 - b0, n, 0, LM_MEM_HOST).total;
    }
    return total;
}

} // extern "C"

// The streams, events and pinned totals of the host-data pipeline (include/lm.h: lm_pipe_*).  Owned by the handle, bound
// to the device that was current at lm_pipe_create; one lm_pipe_solve at a time per handle.
struct lm_pipe {
    static constexpr int NS = 4;
    int dev = -1;
    int max_chunks = 0;
    cudaStream_t st[NS] = {nullptr, nullptr, nullptr, nullptr}; // host->device copies, device->host copies, 2 x kernels
    cudaEvent_t *ev_in = nullptr, *ev_done = nullptr;           // [max_chunks]
    cudaEvent_t ev_entry = nullptr, ev_exit[NS] = {nullptr, nullptr, nullptr, nullptr};
    unsigned long long *totals = nullptr;                       // pinned, [2 * max_chunks]
};

extern "C" {

void lm_pipe_destroy(lm_pipe *p) {
    if (!p) return;
    for (int i = 0; i < lm_pipe::NS; ++i) {
        if (p->st[i]) cudaStreamDestroy(p->st[i]);
        if (p->ev_exit[i]) cudaEventDestroy(p->ev_exit[i]);
    }
    for (int i = 0; i < p->max_chunks; ++i) {
        if (p->ev_in && p->ev_in[i]) cudaEventDestroy(p->ev_in[i]);
        if (p->ev_done && p->ev_done[i]) cudaEventDestroy(p->ev_done[i]);
    }
    if (p->ev_entry) cudaEventDestroy(p->ev_entry);
    if (p->totals) cudaFreeHost(p->totals);
    delete[] p->ev_in;
    delete[] p->ev_done;
    delete p;
}

int lm_pipe_create(lm_pipe **out, int32_t max_chunks) {
    if (!out || max_chunks < 1 || max_chunks > LM_PIPE_MAX_CHUNKS) return LM_EINVAL;
    *out = nullptr;
    lm_pipe *p = new (std::nothrow) lm_pipe();
    if (!p) return LM_ENOMEM;
    p->ev_in = new (std::nothrow) cudaEvent_t[max_chunks]();
    p->ev_done = new (std::nothrow) cudaEvent_t[max_chunks]();
    if (!p->ev_in || !p->ev_done) { lm_pipe_destroy(p); return LM_ENOMEM; }
    p->max_chunks = max_chunks;
    cudaError_t e = cudaGetDevice(&p->dev);
    for (int i = 0; i < lm_pipe::NS && e == cudaSuccess; ++i) {
        e = cudaStreamCreateWithFlags(&p->st[i], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_exit[i], cudaEventDisableTiming);
    }
    for (int i = 0; i < max_chunks && e == cudaSuccess; ++i) {
        e = cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_done[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_entry, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMallocHost(reinterpret_cast<void **>(&p->totals), 16 * (size_t)max_chunks);
    if (e != cudaSuccess) { lm_pipe_destroy(p); return cuda_fail(e); }
    *out = p;
    return LM_OK;
}

int lm_solve_host(const lm_chain *chain, const lm_problem *pb, const lm_params *prm, int32_t max_iters, int32_t chunks,
                  float *q_out, lm_stats *st) {
    if (chunks < 1 || chunks > LM_PIPE_MAX_CHUNKS) return LM_EINVAL;
    lm_pipe *p = nullptr;
    int rc = lm_pipe_create(&p, chunks);
    if (rc != LM_OK) return rc;
    rc = lm_pipe_solve(p, nullptr, chain, pb, prm, max_iters, chunks, q_out, st);
    lm_pipe_destroy(p);
    return rc;
}

int lm_pipe_solve(lm_pipe *pp, void *cuda_stream, const lm_chain *chain, const lm_problem *pb, const lm_params *prm, int32_t max_iters,
                  int32_t chunks, float *q_out, lm_stats *st) {
    if (!pp || !chain || !pb || !prm || max_iters < 0 || max_iters > LM_MAX_ITERS) return LM_EINVAL;
    if (pb->memory != LM_MEM_HOST || pb->shared_targets || pb->B <= 0 || pb->n <= 0 || chunks < 1 || chunks > pb->B) return LM_EINVAL;
    if (!pb->target_pos || !pb->target_quat || !pb->seeds || !pb->workspace) return LM_EINVAL;
    const int d = chain->dof;
    if (d < 1 || d > LM_MAX_DOF) return LM_EINVAL;
    if (chunks > pp->max_chunks) return LM_EINVAL;
    if (pb->workspace_bytes < lm_solve_host_workspace_bytes(d, pb->B, pb->n, chunks)) return LM_ENOMEM;
    const size_t W = (size_t)pb->B * (size_t)pb->n;
    lm_pipe &pipe = *pp;
    constexpr int NS = lm_pipe::NS;
    int rc = LM_OK;
    auto fail = [&](cudaError_t e) { rc = cuda_fail(e); };
    int dev = 0;
    LM_CUDA(cudaGetDevice(&dev));
    if (dev != pipe.dev) return LM_EINVAL; // the handle belongs to the device that was current when it was created
    // everything the caller has enqueued on its stream (e.g. the production of the host inputs by a device->host copy)
    // precedes the pipeline
    cudaStream_t caller = static_cast<cudaStream_t>(cuda_stream);
    LM_CUDA(cudaEventRecord(pipe.ev_entry, caller));
    for (int i = 0; i < NS; ++i) LM_CUDA(cudaStreamWaitEvent(pipe.st[i], pipe.ev_entry, 0));
    cudaStream_t s_in = pipe.st[0], s_out = pipe.st[1];
    cudaStream_t s_kk[2] = {pipe.st[2], pipe.st[3]}; // chunks alternate between two kernel streams: the tail of one
                                                     // chunk's last wave overlaps the head of the next chunk's kernel
    unsigned long long *totals = pipe.totals;
    lm_ctx **ctxs = new (std::nothrow) lm_ctx *[chunks]();
    if (!ctxs) return LM_ENOMEM;
    struct Chunk { int64_t b0, Bc; size_t w0, Wc; Layout lay; char *ws; };
    Chunk *ck = new (std::nothrow) Chunk[chunks];
    if (!ck) { delete[] ctxs; return LM_ENOMEM; }
    {
        char *ws = static_cast<char *>(pb->workspace);
        for (int k = 0; k < chunks; ++k) {
            int64_t b0, b1;
            chunk_range(pb->B, chunks, k, b0, b1);
            ck[k].b0 = b0; ck[k].Bc = b1 - b0;
            ck[k].w0 = (size_t)b0 * (size_t)pb->n; ck[k].Wc = (size_t)(b1 - b0) * (size_t)pb->n;
            ck[k].lay = make_layout(d, b1 - b0, pb->n, 0, LM_MEM_HOST);
            ck[k].ws = ws;
            ws += ck[k].lay.total;
        }
    }
    // stage 1 (copy stream): every chunk's inputs, in order; rows of the SoA arrays are W apart on the host,
    // Wc apart in the chunk's staging area
    for (int k = 0; k < chunks && rc == LM_OK; ++k) {
        const Chunk &c = ck[k];
        float *sd = reinterpret_cast<float *>(c.ws + c.lay.s_seeds), *tpd = reinterpret_cast<float *>(c.ws + c.lay.s_tp),
              *tqd = reinterpret_cast<float *>(c.ws + c.lay.s_tq);
        cudaError_t e = cudaMemcpy2DAsync(sd, 4 * c.Wc, pb->seeds + c.w0, 4 * W, 4 * c.Wc, d, cudaMemcpyHostToDevice, s_in);
        if (e == cudaSuccess) e = cudaMemcpy2DAsync(tpd, 4 * c.Wc, pb->target_pos + c.w0, 4 * W, 4 * c.Wc, 3, cudaMemcpyHostToDevice, s_in);
        if (e == cudaSuccess) e = cudaMemcpy2DAsync(tqd, 4 * c.Wc, pb->target_quat + c.w0, 4 * W, 4 * c.Wc, 4, cudaMemcpyHostToDevice, s_in);
        if (e == cudaSuccess) e = cudaEventRecord(pipe.ev_in[k], s_in);
        if (e != cudaSuccess) fail(e);
    }
    // stage 2 (kernel stream): the LM kernel of chunk k as soon as its inputs have arrived, then its statistics
    for (int k = 0; k < chunks && rc == LM_OK; ++k) {
        const Chunk &c = ck[k];
        cudaStream_t s_k = s_kk[k & 1];
        cudaError_t e = cudaStreamWaitEvent(s_k, pipe.ev_in[k], 0);
        if (e != cudaSuccess) { fail(e); break; }
        lm_problem pk = *pb;
        pk.B = c.Bc;
        pk.seeds = reinterpret_cast<float *>(c.ws + c.lay.s_seeds);
        pk.target_pos = reinterpret_cast<float *>(c.ws + c.lay.s_tp);
        pk.target_quat = reinterpret_cast<float *>(c.ws + c.lay.s_tq);
        pk.memory = LM_MEM_DEVICE;
        pk.workspace = c.ws; pk.workspace_bytes = c.lay.total;
        rc = lm_init(&ctxs[k], chain, &pk, prm, s_k);
        if (rc != LM_OK) break;
        rc = iterate(ctxs[k], max_iters, INT_MAX);
        if (rc != LM_OK) break;
        const KArgs &a = ctxs[k]->args;
        unsigned long long *tot = reinterpret_cast<unsigned long long *>(c.ws + c.lay.totals);
        e = cudaMemsetAsync(tot, 0, 16, s_k);
        if (e != cudaSuccess) { fail(e); break; }
        g_launches.fetch_add(1);
        lm_traj_stats_kernel<<<(unsigned)((c.Bc * 32 + 255) / 256), 256, 0, s_k>>>(
            a.its, c.Bc, (int32_t)pb->n, reinterpret_cast<uint8_t *>(c.ws + c.lay.conv), reinterpret_cast<int32_t *>(c.ws + c.lay.titers), tot);
        if (st && (st->iters || st->status)) {
            g_launches.fetch_add(1);
            lm_unpack_kernel<<<(unsigned)((c.Wc + 255) / 256), 256, 0, s_k>>>(
                a.its, (int64_t)c.Wc, st->iters ? reinterpret_cast<int32_t *>(c.ws + c.lay.ui) : nullptr,
                st->status ? reinterpret_cast<uint32_t *>(c.ws + c.lay.us) : nullptr);
        }
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventRecord(pipe.ev_done[k], s_k);
        if (e != cudaSuccess) fail(e);
    }
    // stage 3 (copy-back stream): the outputs of chunk k as soon as its kernels are done
    for (int k = 0; k < chunks && rc == LM_OK; ++k) {
        const Chunk &c = ck[k];
        const KArgs &a = ctxs[k]->args;
        cudaError_t e = cudaStreamWaitEvent(s_out, pipe.ev_done[k], 0);
        if (e != cudaSuccess) { fail(e); break; }
        auto out1 = [&](void *dst, const void *src, size_t elem, size_t off, size_t count) {
            if (dst && rc == LM_OK) {
                cudaError_t e2 = cudaMemcpyAsync(static_cast<char *>(dst) + elem * off, src, elem * count, cudaMemcpyDeviceToHost, s_out);
                if (e2 != cudaSuccess) fail(e2);
            }
        };
        if (q_out) {
            e = cudaMemcpy2DAsync(q_out + c.w0, 4 * W, a.q, 4 * c.Wc, 4 * c.Wc, d, cudaMemcpyDeviceToHost, s_out);
            if (e != cudaSuccess) { fail(e); break; }
        }
        if (st) {
            out1(st->res_norm, a.res, 4, c.w0, c.Wc);
            out1(st->pos_err, a.perr, 4, c.w0, c.Wc);
            out1(st->rot_err, a.rerr, 4, c.w0, c.Wc);
            out1(st->lambda, a.lam, 4, c.w0, c.Wc);
            out1(st->accept_mask, a.mask, 8, c.w0, c.Wc);
            out1(st->traj_converged, c.ws + c.lay.conv, 1, (size_t)c.b0, (size_t)c.Bc);
            out1(st->traj_iters, c.ws + c.lay.titers, 4, (size_t)c.b0, (size_t)c.Bc);
            out1(st->iters, c.ws + c.lay.ui, 4, c.w0, c.Wc);
            out1(st->status, c.ws + c.lay.us, 4, c.w0, c.Wc);
        }
        if (rc == LM_OK) {
            e = cudaMemcpyAsync(totals + 2 * k, c.ws + c.lay.totals, 16, cudaMemcpyDeviceToHost, s_out);
            if (e != cudaSuccess) fail(e);
        }
    }
    for (int i = 0; i < NS; ++i) { // later work on the caller's stream is ordered after the pipeline; the host waits for it
        cudaError_t e = cudaEventRecord(pipe.ev_exit[i], pipe.st[i]);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(caller, pipe.ev_exit[i], 0);
        if (e == cudaSuccess) e = cudaStreamSynchronize(pipe.st[i]);
        if (e != cudaSuccess && rc == LM_OK) fail(e);
    }
    if (st && rc == LM_OK) {
        st->total_waypoint_iters = 0;
        st->converged_trajectories = 0;
        for (int k = 0; k < chunks; ++k) {
            st->total_waypoint_iters += (int64_t)totals[2 * k];
            st->converged_trajectories += (int64_t)totals[2 * k + 1];
        }
    }
    delete[] ck;
    for (int k = 0; k < chunks; ++k) delete ctxs[k];
    delete[] ctxs;
    return rc;
}

int lm_fp32_peak(void *cuda_stream, double *tflops_out) {
    if (!tflops_out) return LM_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    LM_CUDA(cudaGetDevice(&dev));
    LM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *sink = nullptr; // the kernel's never-taken store needs an address
    LM_CUDA(cudaMalloc(&sink, 256));
    cudaEvent_t e0, e1;
    LM_CUDA(cudaEventCreate(&e0));
    LM_CUDA(cudaEventCreate(&e1));
    const int iters = 32768, blocks = sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(e0, st);
        g_launches.fetch_add(1);
        lm_fma_peak_kernel<<<blocks, threads, 0, st>>>(sink, iters, 0.999f, 1e-3f);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(sink); return cuda_fail(e); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double tf = 2.0 * 16.0 * iters * (double)blocks * threads / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *tflops_out = best;
    return LM_OK;
}

void lm_free(lm_ctx *c) { delete c; }

const char *lm_strerror(int code) {
    switch (code) {
    case LM_OK: return "ok";
    case LM_EINVAL: return "invalid argument";
    case LM_ENOMEM: return "workspace too small or out of host memory";
    case LM_ECUDA: return g_cuda_err;
    case LM_ECAPACITY: return "problem exceeds the fixed scratch of lm_search_static (LM_SEARCH_STATIC_BYTES); use lm_search with a caller-allocated workspace";
    default: return "unknown lm_status";
    }
}

int64_t lm_launch_count(void) { return g_launches.load(); }

} // extern "C"
