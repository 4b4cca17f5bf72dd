// lm_traj_api.cu -- C ABI of the trajectory-level LM step (include/lm.h, lm_traj_*): workspace
// carving and the launch sequence of one iteration.  Every arithmetic step runs in the kernels
// of lm_traj.cuh; the host only enqueues launches (no synchronisation before lm_traj_fetch).
#define LM_TRAJ_PLAIN_KERNELS
#include "lm_ctx.h"
#include "lm_traj_launch.h"

#include <cmath>
#include <cstring>

using namespace lmk;

namespace {

struct TLayout {
    size_t tp, tq, q, Ag, rho, rows, rcnt, cst, V, z, delta, lam, F, Fp, Fd, Fc, its, mask, sel, ok, totals, ui, us, total;
};

// tile order (lm_traj.cuh): Bt = ceil(B / 32) tiles, nS = Bt * n * 32 slots, C floats per slot and array
TLayout make_tlayout(int d, int64_t B, int64_t n) {
    const size_t Bt = ((size_t)B + 31) / 32, Bp = Bt * 32, nS = Bp * (size_t)n, NA = (size_t)d * (d + 1) / 2;
    TLayout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    L.tp = take(4 * 3 * nS);
    L.tq = take(4 * 4 * nS);
    L.q = take(4 * 2 * d * nS);
    L.Ag = take(4 * (NA + d) * nS);
    L.rho = take(4 * d * nS);
    L.rows = take(4 * 2 * (size_t)TL_RMAX * (d + 1) * nS);
    L.rcnt = take(4 * 2 * nS);
    L.cst = take(4 * 3 * nS);
    L.V = take(4 * NA * nS);
    L.z = take(4 * d * nS);
    L.delta = take(4 * d * nS);
    L.lam = take(4 * Bp);
    L.F = take(4 * Bp);
    L.Fp = take(4 * Bp);
    L.Fd = take(4 * Bp);
    L.Fc = take(4 * Bp);
    L.its = take(4 * Bp);
    L.mask = take(8 * Bp);
    L.sel = take(4 * Bp);
    L.ok = take(4 * Bp);
    L.totals = take(16);
    L.ui = take(4 * Bp);
    L.us = take(4 * Bp);
    L.total = off;
    return L;
}

cudaError_t launch_pose(lm_ctx *c, int which, const TArgs &a) {
    launch_counter().fetch_add(1);
    const unsigned block = 128;
    const unsigned grid = (unsigned)(((which == TK_CLEARANCE ? a.B * a.n : a.nS) + block - 1) / block);
    const bool weighted = c->args.weighted != 0;
    if (c->spec_id != SPEC_GENERIC && !c->use_generic)
        return launch_traj_pose_spec(which, c->spec_id, weighted, grid, block, c->stream, a);
    return c->dof <= 4 ? launch_traj_pose_generic_lo(which, c->dof, weighted, grid, block, c->stream, a)
                       : launch_traj_pose_generic_hi(which, c->dof, weighted, grid, block, c->stream, a);
}

cudaError_t launch_plain(lm_ctx *c, int which, const TArgs &a) {
    launch_counter().fetch_add(1);
    if (which == TK_SOLVE_FACTOR_HBM || which == TK_SOLVE_REFINE_HBM) return launch_traj_plain(which, c->dof, 0, 0, c->stream, a);
    const unsigned block = 256, grid = (unsigned)((a.nS + block - 1) / block);
    return launch_traj_plain(which, c->dof, grid, block, c->stream, a);
}

__global__ void tl_stats_kernel(const uint32_t *__restrict__ its, int64_t B, int32_t *__restrict__ iters,
                                uint32_t *__restrict__ status, unsigned long long *__restrict__ totals) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const uint32_t pk = its[b];
    if (iters) iters[b] = (int32_t)(pk & 0xffu);
    if (status) status[b] = (pk >> 8) & ~32u;
    atomicAdd(totals, (unsigned long long)(pk & 0xffu)); // integer: order-free
}

bool is_host_ptr(const void *p) {
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, p) != cudaSuccess) { cudaGetLastError(); return true; }
    return pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged;
}

} // namespace

namespace lmk {
int launch_clearance(lm_ctx *c, float *clear_out) { // smallest capsule clearance per waypoint at the context's current q
    TArgs a = c->traj.args;
    a.src_q = c->args.q;
    a.clear_out = clear_out;
    LM_CUDA(launch_pose(c, TK_CLEARANCE, a));
    return LM_OK;
}
} // namespace lmk

extern "C" {

size_t lm_traj_workspace_bytes(int32_t dof, int64_t B, int64_t n) {
    if (dof < 1 || dof > LM_MAX_DOF || B <= 0 || n <= 0) return 0;
    return make_tlayout(dof, B, n).total;
}

int lm_traj_default_params(lm_traj_params *out) {
    if (!out) return LM_EINVAL;
    out->w_pose = 1.f;
    out->w_diff = 1.f;
    out->lambda0 = 1e-3f;
    out->nu_up = 10.f;
    out->nu_down = 10.f;
    out->lambda_min = 1e-4f;
    out->lambda_max = 1e7f;
    out->refine_steps = 1;
    return LM_OK;
}

int lm_traj_attach(lm_ctx *c, const lm_traj_params *p, void *workspace, size_t bytes) {
    if (!c || !p || !workspace) return LM_EINVAL;
    if (c->args.variant == LM_VAR_RPY) return LM_EINVAL; // the trajectory-level step uses the rotation-vector residual
    if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return LM_EINVAL;
    if (!(p->w_pose >= 0.f) || !(p->w_diff >= 0.f) || !(p->lambda0 > 0.f) || !(p->nu_up > 1.f) || !(p->nu_down > 1.f) ||
        !(p->lambda_min > 0.f) || !(p->lambda_max >= p->lambda_min) || p->refine_steps < 0 || p->refine_steps > 2)
        return LM_EINVAL;
    const TLayout L = make_tlayout(c->dof, c->B, c->n);
    if (bytes < L.total) return LM_ENOMEM;
    TrajState &t = c->traj;
    t = TrajState{};
    t.ws = static_cast<char *>(workspace);
    t.bytes = bytes;
    t.lambda0 = p->lambda0;
    t.refine = p->refine_steps;
    t.off_totals = L.totals; t.off_ui = L.ui; t.off_us = L.us;
    TArgs &a = t.args;
    std::memset(&a, 0, sizeof(a));
    a.ch = c->args.ch;
    a.w_pos = c->args.w_pos; a.w_rot = c->args.w_rot;
    a.wp2 = p->w_pose * p->w_pose;
    a.wd2 = p->w_diff * p->w_diff;
    a.wd4 = a.wd2 * a.wd2;
    a.nu_up = p->nu_up; a.inv_nu_down = (float)(1.0 / (double)p->nu_down);
    a.lambda_min = p->lambda_min; a.lambda_max = p->lambda_max;
    a.B = c->B; a.n = (int32_t)c->n; a.Bt = (c->B + 31) / 32; a.nS = a.Bt * 32 * c->n;
    a.shared_targets = c->shared;
    a.max_total = LM_MAX_ITERS;
    auto f = [&](size_t off) { return reinterpret_cast<float *>(t.ws + off); };
    if (c->shared) { // one path for all trajectories: the plain arrays [.][n] are read by waypoint index
        a.tp = c->args.tp; a.tq = c->args.tq;
    } else {
        a.tp = a.tp_w = f(L.tp); a.tq = a.tq_w = f(L.tq);
    }
    a.q = f(L.q); a.Ag = f(L.Ag); a.rho = f(L.rho); a.rows = f(L.rows); a.cst = f(L.cst);
    a.rcnt = reinterpret_cast<int32_t *>(t.ws + L.rcnt); a.V = f(L.V); a.z = f(L.z);
    a.delta = f(L.delta); a.lam = f(L.lam); a.F = f(L.F); a.Fp = f(L.Fp); a.Fd = f(L.Fd); a.Fc = f(L.Fc);
    a.its = reinterpret_cast<uint32_t *>(t.ws + L.its);
    a.mask = reinterpret_cast<unsigned long long *>(t.ws + L.mask);
    a.sel = reinterpret_cast<int32_t *>(t.ws + L.sel);
    a.ok = reinterpret_cast<int32_t *>(t.ws + L.ok);
    a.src_tp = c->args.tp; a.src_tq = c->args.tq;
    t.attached = true;
    return lm_traj_reset(c, nullptr);
}

int lm_traj_reset(lm_ctx *c, const float *lambda) {
    if (!c || !c->traj.attached) return LM_EINVAL;
    TrajState &t = c->traj;
    const float *lam_dev = lambda;
    if (lambda && is_host_ptr(lambda)) { // stage through the z array (rewritten by every solve before it is read)
        LM_CUDA(cudaMemcpyAsync(t.args.z, lambda, 4 * (size_t)c->B, cudaMemcpyHostToDevice, c->stream));
        lam_dev = t.args.z;
    }
    launch_counter().fetch_add(1);
    tl_reset_kernel<<<(unsigned)((t.args.Bt * 32 + 255) / 256), 256, 0, c->stream>>>(t.args, lam_dev, t.lambda0);
    LM_CUDA(cudaGetLastError());
    return LM_OK;
}

int lm_traj_set_capsules(lm_ctx *c, const lm_capsules *m) {
    if (!c || !c->traj.attached) return LM_EINVAL;
    KCaps &k = c->traj.args.caps;
    std::memset(&k, 0, sizeof(k));
    if (!m || m->ncaps == 0) return LM_OK; // no capsules: no collision rows of either kind
    if (m->ncaps < 1 || m->ncaps > LM_MAX_CAPSULES || m->npairs < 0 || m->npairs > LM_MAX_CAPSULE_PAIRS) return LM_EINVAL;
    if (!m->link || !m->a || !m->b || !m->radius || (m->npairs > 0 && !m->pairs) || !(m->w_coll >= 0.f) || !(m->d_safe >= 0.f))
        return LM_EINVAL;
    for (int i = 0; i < m->ncaps; ++i) {
        if (m->link[i] < -1 || m->link[i] >= c->dof || !(m->radius[i] >= 0.f)) return LM_EINVAL;
        k.link[i] = (int8_t)m->link[i];
        k.on_link[m->link[i] + 1] |= (uint16_t)(1u << i);
        k.c[i] = m->radius[i];
        double l2 = 0.0;
        for (int x = 0; x < 3; ++x) {
            k.a[i][x] = m->a[3 * i + x]; k.b[i][x] = m->b[3 * i + x];
            l2 += ((double)k.b[i][x] - k.a[i][x]) * ((double)k.b[i][x] - k.a[i][x]);
        }
        k.hl[i] = (float)(0.5 * std::sqrt(l2) * (1.0 + 1e-6)); // rounded up: the bounding sphere must contain the axis
    }
    for (int p = 0; p < m->npairs; ++p) {
        const int32_t k1 = m->pairs[2 * p], k2 = m->pairs[2 * p + 1];
        if (k1 < 0 || k1 >= m->ncaps || k2 < 0 || k2 >= m->ncaps || k1 == k2) return LM_EINVAL;
        k.pair[p][0] = (uint8_t)k1; k.pair[p][1] = (uint8_t)k2;
    }
    k.ncaps = m->ncaps; k.npairs = (m->w_coll > 0.f) ? m->npairs : 0; k.w_coll = m->w_coll; k.d_safe = m->d_safe;
    return LM_OK;
}

int lm_traj_set_obstacles(lm_ctx *c, const lm_obstacles *o) {
    if (!c || !c->traj.attached) return LM_EINVAL;
    KCaps &k = c->traj.args.caps;
    k.nobs = 0; k.nenv = 0; k.w_env = 0.f; k.d_safe_env = 0.f;
    if (!o || o->npairs == 0 || o->w_env == 0.f) return LM_OK;
    if (k.ncaps == 0) return LM_EINVAL; // lm_traj_set_capsules first
    if (o->nobs < 1 || o->nobs > LM_MAX_OBSTACLES || o->npairs < 0 || o->npairs > LM_MAX_CAPSULE_PAIRS) return LM_EINVAL;
    if (!o->pose || !o->pmin || !o->pmax || !o->pairs || !(o->w_env > 0.f) || !(o->d_safe >= 0.f)) return LM_EINVAL;
    for (int i = 0; i < o->nobs; ++i) {
        const float *ps = o->pose + 7 * i;
        const double n = std::sqrt((double)ps[3] * ps[3] + (double)ps[4] * ps[4] + (double)ps[5] * ps[5] + (double)ps[6] * ps[6]);
        if (!(n > 0.0)) return LM_EINVAL;
        const double w = ps[3] / n, x = ps[4] / n, y = ps[5] / n, z = ps[6] / n;
        const double R[9] = {1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y),
                             2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x),
                             2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)};
        for (int e = 0; e < 9; ++e) k.Ro[i][e] = (float)R[e];
        for (int e = 0; e < 3; ++e) {
            k.to[i][e] = ps[e];
            k.pmin[i][e] = o->pmin[3 * i + e];
            k.pmax[i][e] = o->pmax[3 * i + e];
            if (!(k.pmin[i][e] <= k.pmax[i][e])) return LM_EINVAL;
        }
        double r2 = 0.0;
        for (int e = 0; e < 3; ++e) { // bounding sphere: centre = to + R (pmin + pmax) / 2, radius = |pmax - pmin| / 2
            const double mid[3] = {0.5 * ((double)k.pmin[i][0] + k.pmax[i][0]), 0.5 * ((double)k.pmin[i][1] + k.pmax[i][1]),
                                   0.5 * ((double)k.pmin[i][2] + k.pmax[i][2])};
            k.oc[i][e] = (float)(ps[e] + R[3 * e] * mid[0] + R[3 * e + 1] * mid[1] + R[3 * e + 2] * mid[2]);
            const double h = 0.5 * ((double)k.pmax[i][e] - k.pmin[i][e]);
            r2 += h * h;
        }
        k.orad[i] = (float)(std::sqrt(r2) * (1.0 + 1e-6));
    }
    for (int p = 0; p < o->npairs; ++p) {
        const int32_t kc = o->pairs[2 * p], ob = o->pairs[2 * p + 1];
        if (kc < 0 || kc >= k.ncaps || ob < 0 || ob >= o->nobs) return LM_EINVAL;
        k.env_pair[p][0] = (uint8_t)kc; k.env_pair[p][1] = (uint8_t)ob;
    }
    k.nobs = o->nobs; k.nenv = o->npairs; k.w_env = o->w_env; k.d_safe_env = o->d_safe;
    return LM_OK;
}

int lm_traj_set_trace(lm_ctx *c, float *trial_q, float *trial_F) {
    if (!c || !c->traj.attached || ((trial_q == nullptr) != (trial_F == nullptr))) return LM_EINVAL;
    c->traj.args.trace_q = trial_q;
    c->traj.args.trace_F = trial_F;
    return LM_OK;
}

int lm_traj_run(lm_ctx *c, int32_t iters) {
    if (!c || !c->traj.attached || iters < 0 || iters > LM_MAX_ITERS) return LM_EINVAL;
    TrajState &t = c->traj;
    int rc = materialize_state(c);
    if (rc != LM_OK) return rc;
    TArgs a = t.args;
    a.src_q = c->args.q;
    a.dst_q = c->args.q;
    if (!t.targets_packed && !c->shared) {
        LM_CUDA(launch_plain(c, TK_PACK_TARGETS, a));
        t.targets_packed = true;
    }
    // collision cost: lanes along the path unless the trajectories of a tile are known to be alike (LM_OPT_TRAJ_COST_LANES);
    // set before the entry cost pass, which obeys it too
    a.cost_by_waypoints = t.cost_lanes == 2 || (t.cost_lanes == 0 && !c->shared) ? 1 : 0;
    // current point -> tile order, and its cost
    LM_CUDA(launch_plain(c, TK_PACK_Q, a));
    LM_CUDA(launch_pose(c, TK_COST_INIT, a));
    launch_counter().fetch_add(1);
    tl_init_cost_kernel<<<(unsigned)a.Bt, TL_SUM_WARPS * 32, 0, c->stream>>>(a);
    LM_CUDA(cudaGetLastError());
    // Fused path: the solve kernel's producer warps assemble the normal equations / the refinement residual in shared
    // memory (3 + refine launches per iteration).  Unfused path: per-waypoint kernels write them to HBM and the solve kernel
    // fetches them (4 + 2 refine launches) -- with collision rows (their divergent pair loops need every SM, not the few
    // producer warps of one block per tile) and when there are too few tiles to keep the producers of a block ahead of
    // its chains.  Same functions, same bits either way (tests/test_gpu_traj.py).
    const bool coll = a.caps.npairs + a.caps.nenv > 0;
    // (with the stored rows the producers could take them too; measured: 0.62 vs 0.55 ms at 4096 x 300 with 9 pairs, the
    // recompute fallback spills in the solve kernel)
    const bool fused = !coll && (t.fused_mode == 1 || (t.fused_mode == 0 && a.Bt >= TL_FUSED_MIN_TILES));
    for (int it = 0; it < iters; ++it) { // nothing on the host in between
        if (fused) {
            LM_CUDA(launch_pose(c, TK_SOLVE_FACTOR, a));                                    // assemble + factor + solve: delta
            for (int r = 0; r < t.refine; ++r) LM_CUDA(launch_pose(c, TK_SOLVE_REFINE, a)); // rho + re-solve: delta += e
        } else {
            LM_CUDA(launch_pose(c, TK_ASSEMBLE, a));
            LM_CUDA(launch_plain(c, TK_SOLVE_FACTOR_HBM, a));
            for (int r = 0; r < t.refine; ++r) {
                LM_CUDA(launch_pose(c, TK_RHO, a));
                LM_CUDA(launch_plain(c, TK_SOLVE_REFINE_HBM, a));
            }
        }
        LM_CUDA(launch_pose(c, TK_COST, a));                                      // trial point and its cost
        launch_counter().fetch_add(1);
        tl_decide_kernel<<<(unsigned)a.Bt, TL_SUM_WARPS * 32, 0, c->stream>>>(a); // accept / reject, lambda
        LM_CUDA(cudaGetLastError());
    }
    LM_CUDA(launch_plain(c, TK_UNPACK, a));
    // refresh the per-waypoint outputs of lm_fetch (|r|, pos / rot error, frozen flag) at the new joint values
    return refresh_waypoint_outputs(c);
}

int lm_traj_fetch(lm_ctx *c, lm_traj_stats *s) {
    if (!c || !c->traj.attached || !s) return LM_EINVAL;
    TrajState &t = c->traj;
    const TArgs &a = t.args;
    const size_t B = (size_t)c->B;
    auto out = [&](void *dst, const void *src, size_t bytes) -> cudaError_t {
        return dst ? cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDefault, c->stream) : cudaSuccess;
    };
    LM_CUDA(out(s->cost, a.F, 4 * B));
    LM_CUDA(out(s->cost_pose, a.Fp, 4 * B));
    LM_CUDA(out(s->cost_diff, a.Fd, 4 * B));
    LM_CUDA(out(s->cost_coll, a.Fc, 4 * B));
    LM_CUDA(out(s->lambda, a.lam, 4 * B));
    LM_CUDA(out(s->accept_mask, a.mask, 8 * B));
    unsigned long long *tot = reinterpret_cast<unsigned long long *>(t.ws + t.off_totals);
    int32_t *ui = reinterpret_cast<int32_t *>(t.ws + t.off_ui);
    uint32_t *us = reinterpret_cast<uint32_t *>(t.ws + t.off_us);
    LM_CUDA(cudaMemsetAsync(tot, 0, 16, c->stream));
    launch_counter().fetch_add(1);
    tl_stats_kernel<<<(unsigned)((B + 255) / 256), 256, 0, c->stream>>>(a.its, c->B, ui, us, tot);
    LM_CUDA(cudaGetLastError());
    LM_CUDA(out(s->iters, ui, 4 * B));
    LM_CUDA(out(s->status, us, 4 * B));
    unsigned long long h[2] = {0, 0};
    LM_CUDA(cudaMemcpyAsync(h, tot, 16, cudaMemcpyDeviceToHost, c->stream));
    LM_CUDA(cudaStreamSynchronize(c->stream));
    s->total_traj_iters = (int64_t)h[0];
    return LM_OK;
}

} // extern "C"
