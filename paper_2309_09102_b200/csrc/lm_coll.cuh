// lm_coll.cuh -- collision rows of the trajectory-level step (sm_100a): robot-robot
// (capsule-capsule, below) and robot-environment (capsule-cuboid: segment_box_closest).
//
// "each robot is represented as a set of capsules with endpoints (a, b) and radius c ... the minimum distance
//  between a capsule pair [is] the minimum cost, less c1 + c2, of [the] convex quadratic program
//  min |(a1 + (b1 - a1) t1) - (a2 + (b2 - a2) t2)|^2, 0 <= t1, t2 <= 1"
// Per waypoint and listed pair one hinge row  r = w_coll * max(0, d_safe - dist)  (C4)
// with  d r / d q = -w_coll n^T (J_p1 - J_p2),  n = (p1 - p2) / |p1 - p2|  (C5): the closest points are held
// fixed on their links, which is what forward-mode differentiation through the QP solution gives
// (PAPER.md:L168).  Joints that move BOTH links of a pair move the two points rigidly together and drop
// out, so only the joints between the two links contribute.
//
// The box-constrained 2-variable QP is solved in closed form (the active set is found by clamping:
// interior stationary point, else the edge minimisers), thread per waypoint; capsule endpoints are
// carried into the world frame by a frame sink of the FK loop (lm_device.cuh).
#pragma once
#include "lm_device.cuh"

namespace lmk {

constexpr int MAX_CAPS = 16, MAX_PAIRS = 32, MAX_OBS = 8;

struct KCaps {
    int32_t ncaps, npairs;
    float w_coll, d_safe;
    int8_t link[MAX_CAPS];          // -1 = base frame, j = frame moved by joint j
    uint16_t on_link[MAX_DOF + 1];  // bit k of on_link[j + 1]: capsule k rides on frame j (the frame sink visits only those)
    float a[MAX_CAPS][3], b[MAX_CAPS][3], c[MAX_CAPS];
    float hl[MAX_CAPS];             // half length |b - a| / 2 (bounding sphere of the axis, for culling)
    uint8_t pair[MAX_PAIRS][2];
    // robot-environment rows: cuboids given by their frame in the world (Ro row-major, box axes
    // as columns; origin to) and extents pmin / pmax in that frame; env_pair = (capsule, obstacle)
    int32_t nobs, nenv;
    float w_env, d_safe_env;
    float Ro[MAX_OBS][9], to[MAX_OBS][3], pmin[MAX_OBS][3], pmax[MAX_OBS][3];
    uint8_t env_pair[MAX_PAIRS][2];
    float oc[MAX_OBS][3], orad[MAX_OBS]; // bounding sphere of every cuboid in the world frame (for culling)
};

// world endpoints of the capsules: filled link by link while FK runs
struct CapsWorld {
    float wa[MAX_CAPS][3], wb[MAX_CAPS][3];
};

struct CapsSink {
    const KCaps &C;
    CapsWorld &W;
    __device__ __forceinline__ CapsSink(const KCaps &c, CapsWorld &w) : C(c), W(w) {}
    __device__ __forceinline__ void base() const { // capsules on the base link: the world frame
        for (uint32_t m = C.on_link[0]; m; m &= m - 1u) {
            const int k = __ffs(m) - 1;
#pragma unroll
            for (int i = 0; i < 3; ++i) { W.wa[k][i] = C.a[k][i]; W.wb[k][i] = C.b[k][i]; }
        }
    }
    __device__ __forceinline__ void operator()(int j, const float (&X)[3], const float (&Y)[3], const float (&Z)[3],
                                               const float (&o)[3]) const {
        for (uint32_t m = C.on_link[j + 1]; m; m &= m - 1u) { // warp-uniform: the model is the same for every lane
            const int k = __ffs(m) - 1;
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                W.wa[k][i] = fma_(Z[i], C.a[k][2], fma_(Y[i], C.a[k][1], fma_(X[i], C.a[k][0], o[i])));
                W.wb[k][i] = fma_(Z[i], C.b[k][2], fma_(Y[i], C.b[k][1], fma_(X[i], C.b[k][0], o[i])));
            }
        }
    }
};

__device__ __forceinline__ float dot3(const float (&x)[3], const float (&y)[3]) {
    return fma_(x[2], y[2], fma_(x[1], y[1], mul(x[0], y[0])));
}
__device__ __forceinline__ float clamp01(float x) { return fminf(fmaxf(x, 0.f), 1.f); }

// minimiser (t1, t2) of |r + d1 t1 - d2 t2|^2 on the unit box, r = a1 - a2: the interior stationary point when
// it is feasible, otherwise the better of the clamped edge minimisers (a convex quadratic on a box)
__device__ __forceinline__ void segment_closest(const float (&a1)[3], const float (&b1)[3], const float (&a2)[3],
                                                const float (&b2)[3], float &t1, float &t2) {
    float d1[3], d2[3], r[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) { d1[i] = sub(b1[i], a1[i]); d2[i] = sub(b2[i], a2[i]); r[i] = sub(a1[i], a2[i]); }
    const float A = dot3(d1, d1), B = dot3(d1, d2), E = dot3(d2, d2), C = dot3(d1, r), F = dot3(d2, r);
    const float det = fma_(A, E, -mul(B, B));
    float s1 = 0.f, s2 = 0.f;
    bool interior = false;
    if (det > 1e-6f * mul(A, E)) {
        const float inv = __fdividef(1.0f, det);
        s1 = mul(fma_(B, F, -mul(C, E)), inv);
        s2 = mul(fma_(A, F, -mul(B, C)), inv);
        interior = (s1 >= 0.f) && (s1 <= 1.f) && (s2 >= 0.f) && (s2 <= 1.f);
    }
    if (!interior) {
        const float iA = A > 0.f ? __fdividef(1.0f, A) : 0.f, iE = E > 0.f ? __fdividef(1.0f, E) : 0.f;
        float best = 3.0e38f;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            float u1, u2;
            if (e < 2) { u1 = (float)e; u2 = clamp01(mul(fma_(B, u1, F), iE)); }
            else { u2 = (float)(e - 2); u1 = clamp01(mul(fma_(B, u2, -C), iA)); }
            float cst = 0.f;
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                const float v = fma_(-d2[i], u2, fma_(d1[i], u1, r[i]));
                cst = fma_(v, v, cst);
            }
            if (cst < best) { best = cst; s1 = u1; s2 = u2; }
        }
    }
    t1 = s1; t2 = s2;
}

// min over t in [0,1], p in [pmin, pmax] of |p - (a + (b-a) t)|^2 (box frame): for fixed t the best p is the clamp of
// the segment point, so the cost is a convex piecewise quadratic in t with breakpoints where a coordinate crosses a
// face plane.  Half its derivative, gder(t) = sum_i d_i * (excess of coordinate i over the box), is non-decreasing:
// the breakpoints on either side of its sign change bracket ONE quadratic piece, whose stationary point is exact.
__device__ __forceinline__ float segment_box_closest(const float (&a)[3], const float (&b)[3], const float (&pmin)[3],
                                                     const float (&pmax)[3]) {
    float d[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) d[i] = sub(b[i], a[i]);
    auto gder = [&](float t) {
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const float x = fma_(d[i], t, a[i]);
            const float ex = (x > pmax[i]) ? sub(x, pmax[i]) : (x < pmin[i]) ? sub(x, pmin[i]) : 0.f;
            s = fma_(d[i], ex, s);
        }
        return s;
    };
    if (gder(0.f) >= 0.f) return 0.f;
    if (gder(1.f) <= 0.f) return 1.f;
    float tl = 0.f, th = 1.f;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const float id = (d[i] != 0.f) ? __fdividef(1.0f, d[i]) : 0.f;
#pragma unroll
        for (int side = 0; side < 2; ++side) {
            const float c = clamp01(mul(sub(side ? pmax[i] : pmin[i], a[i]), id));
            if (gder(c) <= 0.f) tl = fmaxf(tl, c); else th = fminf(th, c);
        }
    }
    const float mid = mul(0.5f, add(tl, th));
    float num = 0.f, den = 0.f;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const float x = fma_(d[i], mid, a[i]);
        if (x > pmax[i]) { num = fma_(d[i], sub(a[i], pmax[i]), num); den = fma_(d[i], d[i], den); }
        else if (x < pmin[i]) { num = fma_(d[i], sub(a[i], pmin[i]), num); den = fma_(d[i], d[i], den); }
    }
    const float ts = den > 0.f ? -__fdividef(num, den) : tl;
    return fminf(fmaxf(ts, tl), th);
}

// ---- the two halves of a pair's work.  *_qp: the closest-point problem (divergent, expensive; a pure function of the
// capsule endpoints and the obstacle).  *_finish: distance, hinge test and the row, with the frames of the owning lane.
struct EnvQp { float t, eb[3]; };  // parameter of the closest axis point, (axis point - box point) in the box frame
__device__ __forceinline__ EnvQp env_qp(const KCaps &C, int ob, const float (&wa)[3], const float (&wb)[3]) {
    float ab[3], bb[3], pmin[3], pmax[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) { pmin[i] = C.pmin[ob][i]; pmax[i] = C.pmax[ob][i]; }
#pragma unroll
    for (int i = 0; i < 3; ++i) { // x_box = Ro^T (x - to)
        float sa = 0.f, sb = 0.f;
#pragma unroll
        for (int kk = 0; kk < 3; ++kk) {
            sa = fma_(C.Ro[ob][3 * kk + i], sub(wa[kk], C.to[ob][kk]), sa);
            sb = fma_(C.Ro[ob][3 * kk + i], sub(wb[kk], C.to[ob][kk]), sb);
        }
        ab[i] = sa; bb[i] = sb;
    }
    EnvQp o;
    o.t = segment_box_closest(ab, bb, pmin, pmax);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const float x = fma_(sub(bb[i], ab[i]), o.t, ab[i]);
        o.eb[i] = sub(x, fminf(fmaxf(x, pmin[i]), pmax[i]));
    }
    return o;
}
template <int D, typename SpecT, bool CLEAR_ONLY, typename F>
__device__ __forceinline__ void env_finish(const KChain &ch, const KCaps &C, int k, int ob, const float (&wa)[3], const float (&wb)[3],
                                           const EnvQp &qp, const Pose<D> &Fr, F &&f, float *min_clear) {
    constexpr ChainSpec S = SpecT::spec;
    float ps[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) ps[i] = fma_(sub(wb[i], wa[i]), qp.t, wa[i]);
    const float len = sqrtf(dot3(qp.eb, qp.eb));
    const float dist = sub(len, C.c[k]);
    if (CLEAR_ONLY) { *min_clear = fminf(*min_clear, dist); return; }
    if (!(dist < C.d_safe_env)) return;
    const float r = mul(C.w_env, sub(C.d_safe_env, dist));
    const float il = (len > 0.f) ? __fdividef(1.0f, len) : 0.f; // axis inside the box: no direction, the row keeps its value
    float n[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) n[i] = mul(il, fma_(C.Ro[ob][3 * i + 2], qp.eb[2], fma_(C.Ro[ob][3 * i + 1], qp.eb[1], mul(C.Ro[ob][3 * i], qp.eb[0]))));
    const int L = C.link[k];
    float g[D];
#pragma unroll
    for (int j = 0; j < D; ++j) {
        float gj = 0.f;
        if (j <= L) {
            const bool pris = S.generic ? (((ch.prismatic_mask >> j) & 1u) != 0) : (((S.pris >> j) & 1u) != 0);
            const float z[3] = {Fr.Jw[j][0], Fr.Jw[j][1], Fr.Jw[j][2]};
            float col[3];
            if (pris) { col[0] = z[0]; col[1] = z[1]; col[2] = z[2]; }
            else {
                const float dd[3] = {sub(ps[0], Fr.Jv[j][0]), sub(ps[1], Fr.Jv[j][1]), sub(ps[2], Fr.Jv[j][2])};
                col[0] = fma_(z[1], dd[2], -mul(z[2], dd[1]));
                col[1] = fma_(z[2], dd[0], -mul(z[0], dd[2]));
                col[2] = fma_(z[0], dd[1], -mul(z[1], dd[0]));
            }
            gj = mul(-C.w_env, dot3(n, col));
        }
        g[j] = gj;
    }
    f(g, r);
}
template <int D, typename SpecT, bool CLEAR_ONLY, typename F>
__device__ __forceinline__ void self_finish(const KChain &ch, const KCaps &C, int k1, int k2, const float (&a1)[3], const float (&b1)[3],
                                            const float (&a2)[3], const float (&b2)[3], float t1, float t2, const Pose<D> &Fr, F &&f,
                                            float *min_clear) {
    constexpr ChainSpec S = SpecT::spec;
    float p1[3], p2[3], e[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        p1[i] = fma_(sub(b1[i], a1[i]), t1, a1[i]);
        p2[i] = fma_(sub(b2[i], a2[i]), t2, a2[i]);
        e[i] = sub(p1[i], p2[i]);
    }
    const float len = sqrtf(dot3(e, e));
    const float dist = sub(sub(len, C.c[k1]), C.c[k2]);
    if (CLEAR_ONLY) { *min_clear = fminf(*min_clear, dist); return; }
    if (!(dist < C.d_safe)) return;
    const float r = mul(C.w_coll, sub(C.d_safe, dist));
    const float il = (len > 0.f) ? __fdividef(1.0f, len) : 0.f; // the axes touch: no direction, the row keeps its value
    const float n[3] = {mul(e[0], il), mul(e[1], il), mul(e[2], il)};
    const int L1 = C.link[k1], L2 = C.link[k2];
    const int lo = min(L1, L2), hi = max(L1, L2);
    // the point on the link farther down the chain; its motion relative to the other point
    const float sgn = (L1 > L2) ? -C.w_coll : C.w_coll; // d r / d q_j = -w n.c1 (L1 farther) or +w n.c2 (L2 farther)
    float g[D];
#pragma unroll
    for (int j = 0; j < D; ++j) {
        float gj = 0.f;
        if (j > lo && j <= hi) {
            const bool pris = S.generic ? (((ch.prismatic_mask >> j) & 1u) != 0) : (((S.pris >> j) & 1u) != 0);
            const float z[3] = {Fr.Jw[j][0], Fr.Jw[j][1], Fr.Jw[j][2]};
            float col[3];
            if (pris) { col[0] = z[0]; col[1] = z[1]; col[2] = z[2]; }
            else {
                float d[3];
#pragma unroll
                for (int i = 0; i < 3; ++i) d[i] = sub((L1 > L2) ? p1[i] : p2[i], Fr.Jv[j][i]);
                col[0] = fma_(z[1], d[2], -mul(z[2], d[1]));
                col[1] = fma_(z[2], d[0], -mul(z[0], d[2]));
                col[2] = fma_(z[0], d[1], -mul(z[1], d[0]));
            }
            gj = mul(sgn, dot3(n, col));
        }
        g[j] = gj;
    }
    f(g, r);
}

// culling by bounding volumes: one bit per pair that may have a row (all lanes in step: the model is uniform)
__device__ __forceinline__ void coll_cull(const KCaps &C, const CapsWorld &W, uint32_t &need_env, uint32_t &need_self) {
    need_env = 0u; need_self = 0u; // MAX_PAIRS = 32 of each kind
    for (int p = 0; p < C.nenv; ++p) { // axis midpoint against the box
        const int k = C.env_pair[p][0], ob = C.env_pair[p][1];
        float mw[3], e2 = 0.f;
#pragma unroll
        for (int i = 0; i < 3; ++i) mw[i] = sub(mul(0.5f, add(W.wa[k][i], W.wb[k][i])), C.to[ob][i]);
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const float x = fma_(C.Ro[ob][6 + i], mw[2], fma_(C.Ro[ob][3 + i], mw[1], mul(C.Ro[ob][i], mw[0])));
            const float ex = sub(x, fminf(fmaxf(x, C.pmin[ob][i]), C.pmax[ob][i]));
            e2 = fma_(ex, ex, e2);
        }
        const float reach = add(add(C.hl[k], C.c[k]), add(C.d_safe_env, 1e-4f));
        if (!(e2 > mul(reach, reach))) need_env |= 1u << p;
    }
    for (int p = 0; p < C.npairs; ++p) { // bounding spheres of the two axes
        const int k1 = C.pair[p][0], k2 = C.pair[p][1];
        float cc[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) cc[i] = mul(0.5f, sub(add(W.wa[k1][i], W.wb[k1][i]), add(W.wa[k2][i], W.wb[k2][i])));
        const float reach = add(add(add(C.hl[k1], C.c[k1]), add(C.hl[k2], C.c[k2])), add(C.d_safe, 1e-4f));
        if (!(dot3(cc, cc) > mul(reach, reach))) need_self |= 1u << p;
    }
}

// Calls f(g, r) for every pair whose hinge is active at this waypoint: g[D] = d r / d q, r = the residual.
// Fr = frames retained by FK (Fr.Jw[j] = z_j, Fr.Jv[j] = o_j: eval_pose with WITH_JAC = false).
// CLEAR_ONLY: no rows; *min_clear receives the smallest clearance `dist` over all listed pairs (lm_plan_*: a valid
// trajectory must be collision free).
template <int D, typename SpecT, bool CLEAR_ONLY = false, typename F>
__device__ __forceinline__ void coll_rows(const KChain &ch, const KCaps &C, const CapsWorld &W, const Pose<D> &Fr, F &&f,
                                          float *min_clear = nullptr) {
    // ---- one robot-environment pair: the obstacle does not move
    auto env_item = [&](int p) {
        const int k = C.env_pair[p][0], ob = C.env_pair[p][1];
        float wa[3], wb[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) { wa[i] = W.wa[k][i]; wb[i] = W.wb[k][i]; }
        const EnvQp qp = env_qp(C, ob, wa, wb);
        env_finish<D, SpecT, CLEAR_ONLY>(ch, C, k, ob, wa, wb, qp, Fr, f, min_clear);
    };
    // ---- one robot-robot pair
    auto self_item = [&](int p) {
        const int k1 = C.pair[p][0], k2 = C.pair[p][1];
        float a1[3], b1[3], a2[3], b2[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) { a1[i] = W.wa[k1][i]; b1[i] = W.wb[k1][i]; a2[i] = W.wa[k2][i]; b2[i] = W.wb[k2][i]; }
        float t1, t2;
        segment_closest(a1, b1, a2, b2, t1, t2);
        self_finish<D, SpecT, CLEAR_ONLY>(ch, C, k1, k2, a1, b1, a2, b2, t1, t2, Fr, f, min_clear);
    };
    if (CLEAR_ONLY) { // every listed pair counts towards the clearance
        for (int p = 0; p < C.nenv; ++p) env_item(p);
        for (int p = 0; p < C.npairs; ++p) self_item(p);
        return;
    }
    // ---- culling by bounding volumes, all lanes in step (uniform): one bit per pair that may have a row.  Then the
    // QP and the row for the survivors, every lane through ITS OWN list in ascending order: the lanes of a warp are 32
    // different trajectories (uncorrelated), so a loop over the listed pairs in step would run every pair for the two or
    // three lanes that need it; with the lists the warp iterates max-over-lanes times instead, and a lane's rows still
    // arrive in the order of a plain loop over the pairs (bitwise the same sums).  Measured (C4, all 19 pairs, us per
    // iteration): in-step loop 1225 -> lists 1054; a second, tighter culling level inside the lists (2 or 4 sample
    // points per axis, clearance >= min_j dist(sample_j, body) - hl / K) costs more than it saves (1108 / 1096).
    uint32_t need_env, need_self;
    coll_cull(C, W, need_env, need_self);
    while (need_env) {
        const int p = __ffs(need_env) - 1;
        need_env &= need_env - 1u;
        env_item(p);
    }
    while (need_self) {
        const int p = __ffs(need_self) - 1;
        need_self &= need_self - 1u;
        self_item(p);
    }
}

// Tried and removed (round 2, commit "Collision rows: found once per point ..."): compacting the closest-point problems
// over the warp (items in shared memory, every lane solves one per round, owners finish in their own order; bitwise the
// same).  A warp holds only ~6 items per waypoint on the bench scene, so a round still runs with ~6 lanes: 223 M -> 190 M
// warp instructions, 338 -> 328 us for the cost kernel with 19 pairs, and slower with 9 pairs (0.521 -> 0.551 ms per iteration).

} // namespace lmk
