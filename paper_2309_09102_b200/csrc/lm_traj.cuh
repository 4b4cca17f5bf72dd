// lm_traj.cuh -- kernels of the trajectory-level LM step (sm_100a): the stacked residual
//   r = [w_pose r_pose ; w_diff (q_{k+1} - q_k)_k]            (Fig. 6)
// whose Jacobian has the kinematic Jacobian J_i on the pose rows of waypoint i and
// -I / +I on the differencing rows, so that per trajectory
//   J^T J + lambda I = block-tridiag( T_i , -w_d^2 I ),   T_i = w_p^2 J_i^T J_i + (c_i w_d^2 + lambda) I,
//   c_i = 1 at the two ends, 2 inside (0 for n = 1).
// The block structure is kept (include/lm.h): block Gaussian elimination
// along the waypoint index,
//   S_i = T_i - w_d^4 S_prev^-1,  z_i = S_i^-1 (g_i + w_d^2 z_prev),  x_i = z_i + w_d^2 S_i^-1 x_next,  delta = -x,
// run from BOTH ends of the trajectory towards the middle waypoint (tl_solve_kernel), one LANE per
// trajectory (the recurrence is sequential in i, the trajectories are the parallel dimension), d x d
// symmetric blocks in registers, S_i^-1 by the symmetric sweep operator.  Everything per-waypoint
// (FK, Jacobian, J^T J, J^T r, collision rows, trial cost) runs one thread per waypoint.
//
// Layout ("tile order"): trajectories are grouped in tiles of 32 (one warp); the record of
// waypoint i of tile bt is the chunk  wid = bt * n + i,  and component c of lane l (trajectory
// b = 32 bt + l) of a C-component array lives at  (wid * C + c) * 32 + l.  A warp therefore reads
// or writes a chunk as C consecutive 128-byte lines, a tile's chunks for i = 0..n-1 are one
// contiguous stream.  The normal equations of a waypoint never go to HBM: producer warps of the solve
// kernel evaluate FK, the Jacobian and w_p^2 J^T J, g (or the refinement residual) of the next
// waypoints straight into a shared-memory ring several waypoints ahead of the recurrence; what the
// substitution reads back (-S^-1, z) arrives by bulk-async copies (cp.async.bulk + mbarrier).  Lanes of
// the last tile beyond B are padding: they compute on whatever the workspace holds and never store.
// Determinism: fixed summation orders, no float atomics; explicit round-to-nearest intrinsics.
#pragma once
#include "lm_coll.cuh"
#include "lm_device.cuh"
#include "lm_kernels.cuh"

namespace lmk {

struct TArgs {
    KChain ch;
    float w_pos, w_rot;            // pose residual weights (lm_params)
    float wp2, wd2, wd4;           // w_pose^2, w_diff^2, w_diff^4
    float nu_up, inv_nu_down, lambda_min, lambda_max;
    int64_t B, Bt, nS;             // trajectories, tiles = ceil(B / 32), slots = Bt * n * 32
    int32_t n;
    int32_t shared_targets;
    int32_t max_total;             // iteration cap per trajectory (mask width)
    int32_t cost_by_waypoints;     // collision rows: 1 = tl_cost_window_kernel (lanes along the path), 0 = tl_cost_kernel (tile order)
    const float *tp, *tq;          // targets: tile order [3], [4] comps; when shared: plain [3][n], [4][n]
    float *tp_w, *tq_w;            // the same arrays, writable (pack kernel)
    float *q;                      // [2] x D comps     current / candidate joint values (`sel` says which is current)
    float *cst;                    // 3                 cost terms of the point last evaluated by tl_cost_kernel:
                                   //                   |r_pose,i|^2, |q_{i+1} - q_i|^2 (0 for the last waypoint), collision cost
    float *Ag;                     // NA + D            unfused path only: w_p^2 J^T J (packed lower), then g of the stacked residual
    float *rho;                    // D                 unfused path only: refinement residual
    float *rows;                   // [2] x TL_RMAX x (D + 1)  collision rows (g, r) of the point in q buffer 0 / 1, as tl_cost_kernel found them
    int32_t *rcnt;                 // [2] x 1           how many (TL_ROWS_OVERFLOW: more than TL_RMAX, recompute)
    float *V;                      // NA                -(S_i)^-1
    float *z;                      // D
    float *delta;                  // D
    float *lam, *F, *Fp, *Fd, *Fc; // [Bt * 32] per trajectory
    uint32_t *its;                 // iters | status << 8
    unsigned long long *mask;
    int32_t *sel;                  // which of the two buffers holds the trajectory's current point
    int32_t *ok;                   // this iteration's solve succeeded
    KCaps caps;                    // self-collision capsules (npairs = 0: none), lm_coll.cuh
    const int32_t *gate;           // nullable: only trajectories with gate[b] != 0 take the step (lm_plan_run)
    float *trace_q, *trace_F;      // nullable: trial point [D][W] in w-order (w = b n + i), (F, F+) [2][B]
    const float *src_q;            // pack: [D][W] w-order
    const float *src_tp, *src_tq;  // pack: [3][W], [4][W] w-order
    float *dst_q;                  // unpack: [D][W] w-order
    float *clear_out;              // tl_clearance_kernel: [W] w-order, smallest capsule clearance of the waypoint
};

template <int D> struct Tri { static constexpr int NA = D * (D + 1) / 2; };
__host__ __device__ constexpr int tri(int r, int c) { return r >= c ? r * (r + 1) / 2 + c : c * (c + 1) / 2 + r; }

// which (tile, waypoint, trajectory) a thread of a per-waypoint kernel owns
struct Slot {
    int64_t wid; // chunk index bt * n + i
    int lane;
    int i;       // waypoint
    int64_t b;   // trajectory
    bool valid;
};
__device__ __forceinline__ Slot slot_of_thread(const TArgs &A) {
    Slot s;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    s.lane = (int)(t & 31);
    s.wid = t >> 5;
    const int64_t bt = s.wid / A.n;
    s.i = (int)(s.wid - bt * A.n);
    s.b = bt * 32 + s.lane;
    s.valid = (s.wid < A.Bt * A.n) && (s.b < A.B);
    return s;
}
template <int C> __device__ __forceinline__ int64_t toff(int64_t wid, int c, int lane) { return (wid * C + c) * 32 + lane; }

// ---- w-order -> tile order (targets once per attach, q at the start of every lm_traj_run)
template <int D>
__global__ void __launch_bounds__(256) tl_pack_kernel(const __grid_constant__ TArgs A, int what) {
    const Slot s = slot_of_thread(A);
    if (!s.valid) return;
    const int64_t W = A.B * A.n, w = s.b * A.n + s.i;
    if (what == 0) { // joint values into the buffer the trajectory currently selects
        float *dst = A.q + (int64_t)A.sel[s.b] * D * A.nS;
#pragma unroll
        for (int j = 0; j < D; ++j) dst[toff<D>(s.wid, j, s.lane)] = A.src_q[(int64_t)j * W + w];
    } else if (!A.shared_targets) {
#pragma unroll
        for (int c = 0; c < 3; ++c) A.tp_w[toff<3>(s.wid, c, s.lane)] = A.src_tp[(int64_t)c * W + w];
#pragma unroll
        for (int c = 0; c < 4; ++c) A.tq_w[toff<4>(s.wid, c, s.lane)] = A.src_tq[(int64_t)c * W + w];
    }
}

template <int D>
__global__ void __launch_bounds__(256) tl_unpack_kernel(const __grid_constant__ TArgs A) {
    const Slot s = slot_of_thread(A);
    if (!s.valid) return;
    const int64_t W = A.B * A.n, w = s.b * A.n + s.i;
    const float *src = A.q + (int64_t)A.sel[s.b] * D * A.nS;
#pragma unroll
    for (int j = 0; j < D; ++j) A.dst_q[(int64_t)j * W + w] = src[toff<D>(s.wid, j, s.lane)];
}

// load the target of a slot and convert the quaternion (DESIGN R11)
__device__ __forceinline__ void tl_load_target(const TArgs &A, const Slot &s, float (&pt)[3], float (&Rt)[3][3]) {
    float qv[4];
    if (A.shared_targets) {
#pragma unroll
        for (int c = 0; c < 3; ++c) pt[c] = __ldg(A.tp + (int64_t)c * A.n + s.i);
#pragma unroll
        for (int c = 0; c < 4; ++c) qv[c] = __ldg(A.tq + (int64_t)c * A.n + s.i);
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) pt[c] = __ldg(A.tp + toff<3>(s.wid, c, s.lane));
#pragma unroll
        for (int c = 0; c < 4; ++c) qv[c] = __ldg(A.tq + toff<4>(s.wid, c, s.lane));
    }
    quat_to_cols(qv[0], qv[1], qv[2], qv[3], Rt);
}

// ---- collision rows of a waypoint.  The pair loops (culling, the box-constrained QPs) are divergent and
// expensive, and one point is visited three times per iteration (its cost as a trial point, then -- if accepted -- the
// assembly and the refinement residual): tl_cost_kernel, which sees every point first, keeps the rows it finds
// (g = d r / d q, r), up to TL_RMAX per waypoint, next to the joint buffer it writes; the other two read them back in the
// same order (bitwise the same sums).  A waypoint with more active rows is marked TL_ROWS_OVERFLOW and recomputed.
#ifndef LM_TL_RMAX
#define LM_TL_RMAX 6
#endif
constexpr int TL_RMAX = LM_TL_RMAX, TL_ROWS_OVERFLOW = 255;
template <int D> __host__ __device__ constexpr int tl_row_comps() { return TL_RMAX * (D + 1); }

// the stored rows of one waypoint, requested before the FK pass that precedes their use (two dependent round trips --
// count, then rows -- overlap with it instead of following it)
template <int D>
struct StoredRows {
    int cnt;
    float v[TL_RMAX][D + 1];
};
template <int D>
__device__ __forceinline__ void tl_rows_fetch(const TArgs &A, int buf, int64_t wid, int lane, StoredRows<D> &R) {
    constexpr int RC = tl_row_comps<D>();
    R.cnt = A.rcnt[(int64_t)buf * A.nS + wid * 32 + lane];
    const float *rw = A.rows + (int64_t)buf * RC * A.nS;
#pragma unroll
    for (int r = 0; r < TL_RMAX; ++r) {
        const bool have = r < R.cnt && R.cnt != TL_ROWS_OVERFLOW;
#pragma unroll
        for (int c = 0; c <= D; ++c) R.v[r][c] = have ? rw[toff<RC>(wid, r * (D + 1) + c, lane)] : 0.f;
    }
}
// f(g, r) for every active row of the waypoint, in the order tl_cost_kernel found them
template <int D, bool WEIGHTED, typename SpecT, typename F>
__device__ __forceinline__ void tl_rows_apply(const TArgs &A, const StoredRows<D> &R, const float (&q)[D], const float (&pt)[3],
                                              const float (&Rt)[3][3], F &&f) {
    if (R.cnt == TL_ROWS_OVERFLOW) { // rare: recompute (frames by an FK pass with the capsule sink, then the pair loops)
        Pose<D> Fr;
        CapsWorld W;
        CapsSink sink(A.caps, W);
        sink.base();
        eval_pose<D, false, WEIGHTED, SpecT, false, CapsSink>(A.ch, q, pt, Rt, A.w_pos, A.w_rot, Fr, nullptr, nullptr, nullptr, sink);
        coll_rows<D, SpecT>(A.ch, A.caps, W, Fr, f);
        return;
    }
#pragma unroll
    for (int r = 0; r < TL_RMAX; ++r) {
        if (__ballot_sync(__activemask(), r < R.cnt) == 0u) break;
        if (r < R.cnt) {
            float g[D];
#pragma unroll
            for (int j = 0; j < D; ++j) g[j] = R.v[r][j];
            f(g, R.v[r][D]);
        }
    }
}

// ---- smallest clearance over all listed capsule pairs at the joint values src_q (w-order): thread per waypoint.
//      Used by lm_plan_run: a valid trajectory is collision free.
template <int D, typename SpecT>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) tl_clearance_kernel(const __grid_constant__ TArgs A) {
    const int64_t W = A.B * A.n;
    const int64_t w = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= W) return;
    float q[D];
#pragma unroll
    for (int j = 0; j < D; ++j) q[j] = A.src_q[(int64_t)j * W + w];
    const float pt[3] = {0.f, 0.f, 0.f};
    const float Rt[3][3] = {{1.f, 0.f, 0.f}, {0.f, 1.f, 0.f}, {0.f, 0.f, 1.f}};
    Pose<D> Fr;
    CapsWorld Wc;
    CapsSink sink(A.caps, Wc);
    sink.base();
    eval_pose<D, false, false, SpecT, false, CapsSink>(A.ch, q, pt, Rt, 1.f, 1.f, Fr, nullptr, nullptr, nullptr, sink);
    float mc = 3.0e38f;
    coll_rows<D, SpecT, true>(A.ch, A.caps, Wc, Fr, [](const float (&)[D], float) {}, &mc);
    A.clear_out[w] = mc;
}

// ---- what a producer warp of the solve kernel computes for waypoint i of its tile (lane = trajectory) into a ring
// stage `st` ([C][32] floats, component c of lane l at st[c * 32 + l]); `qs` = the lane's CURRENT joint buffer.
//   tl_chunk_normal: w_p^2 J^T J (+ collision rows; packed lower, NA entries) and
//                    g = w_p^2 J^T r + w_d^2 (c_i y_i - y_{i-1} - y_{i+1}) (+ J_c^T r_c),  y = the joint values
// the inputs of a chunk, loaded ahead of its turn by the fused producers (joint values of waypoints i-1, i, i+1 and the target)
template <int D>
struct ChunkIn {
    float q[D], qm[D], qn[D], tg[7];
};
template <int D>
__device__ __forceinline__ void tl_chunk_load(const TArgs &A, const float *qs, int64_t w0, int i, int lane, ChunkIn<D> &in) {
    const int n = A.n;
    const int64_t wid = w0 + i;
#pragma unroll
    for (int j = 0; j < D; ++j) {
        in.q[j] = qs[toff<D>(wid, j, lane)];
        in.qm[j] = (i > 0) ? qs[toff<D>(wid - 1, j, lane)] : 0.f;
        in.qn[j] = (i + 1 < n) ? qs[toff<D>(wid + 1, j, lane)] : 0.f;
    }
    if (A.shared_targets) {
#pragma unroll
        for (int c = 0; c < 3; ++c) in.tg[c] = __ldg(A.tp + (int64_t)c * n + i);
#pragma unroll
        for (int c = 0; c < 4; ++c) in.tg[3 + c] = __ldg(A.tq + (int64_t)c * n + i);
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) in.tg[c] = __ldg(A.tp + toff<3>(wid, c, lane));
#pragma unroll
        for (int c = 0; c < 4; ++c) in.tg[3 + c] = __ldg(A.tq + toff<4>(wid, c, lane));
    }
}

template <int D, bool WEIGHTED, typename SpecT, bool COLL>
__device__ __forceinline__ void tl_chunk_normal(const TArgs &A, const ChunkIn<D> &in, int buf, int64_t w0, int i, int lane, float *st) {
    constexpr int NA = Tri<D>::NA;
    const int n = A.n;
    const float (&q)[D] = in.q, (&qm)[D] = in.qm, (&qn)[D] = in.qn;
    const float pt[3] = {in.tg[0], in.tg[1], in.tg[2]};
    float Rt[3][3];
    quat_to_cols(in.tg[3], in.tg[4], in.tg[5], in.tg[6], Rt);
    StoredRows<D> SR;
    if (COLL) tl_rows_fetch<D>(A, buf, w0 + i, lane, SR);
    Pose<D> P;
    eval_pose<D, false, WEIGHTED, SpecT>(A.ch, q, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr);
    float Ac[NA], gc[D];
#pragma unroll
    for (int t = 0; t < NA; ++t) Ac[t] = 0.f;
#pragma unroll
    for (int j = 0; j < D; ++j) gc[j] = 0.f;
    if (COLL) {
        tl_rows_apply<D, WEIGHTED, SpecT>(A, SR, q, pt, Rt, [&](const float (&g)[D], float r) {
#pragma unroll
            for (int a = 0; a < D; ++a) {
#pragma unroll
                for (int b = 0; b <= a; ++b) Ac[tri(a, b)] = fma_(g[a], g[b], Ac[tri(a, b)]);
                gc[a] = fma_(g[a], r, gc[a]);
            }
        });
    }
    const float ci = (n == 1) ? 0.f : ((i == 0 || i == n - 1) ? 1.f : 2.f);
#pragma unroll
    for (int r = 0; r < D; ++r) {
#pragma unroll
        for (int c = 0; c <= r; ++c) st[tri(r, c) * 32 + lane] = fma_(A.wp2, coldot<D>(P, r, c), Ac[tri(r, c)]);
        const float dd = sub(sub(mul(ci, q[r]), qm[r]), qn[r]);
        st[(NA + r) * 32 + lane] = fma_(A.wd2, dd, fma_(A.wp2, colvec<D>(P, r, P.r), gc[r]));
    }
}

//   tl_chunk_rho: the refinement residual (DESIGN R4 carried over to the stacked system)
//     rho_i = -[ w_p^2 J_i^T (r_i + J_i delta_i) + w_d^2 (D^T D (q + delta))_i + lambda delta_i
//               + sum over active collision pairs of g (r_c + g . delta_i) ]                  into st[0 .. D)
template <int D, bool WEIGHTED, typename SpecT, bool COLL>
__device__ __forceinline__ void tl_chunk_rho(const TArgs &A, const ChunkIn<D> &in, int buf, float lam, int64_t w0, int i, int lane, float *st) {
    const int n = A.n;
    const int64_t wid = w0 + i;
    const float ci = (n == 1) ? 0.f : ((i == 0 || i == n - 1) ? 1.f : 2.f);
    const float (&q)[D] = in.q;
    float dl[D], dd[D];
#pragma unroll
    for (int j = 0; j < D; ++j) {
        dl[j] = A.delta[toff<D>(wid, j, lane)];
        const float yc = add(q[j], dl[j]);
        const float ym = (i > 0) ? add(in.qm[j], A.delta[toff<D>(wid - 1, j, lane)]) : 0.f;
        const float yn = (i + 1 < n) ? add(in.qn[j], A.delta[toff<D>(wid + 1, j, lane)]) : 0.f;
        dd[j] = sub(sub(mul(ci, yc), ym), yn);
    }
    const float pt[3] = {in.tg[0], in.tg[1], in.tg[2]};
    float Rt[3][3];
    quat_to_cols(in.tg[3], in.tg[4], in.tg[5], in.tg[6], Rt);
    Pose<D> P;
    float ec[D]; // collision rows: sum over the active pairs of g (r + g . delta)
#pragma unroll
    for (int j = 0; j < D; ++j) ec[j] = 0.f;
    StoredRows<D> SR;
    if (COLL) tl_rows_fetch<D>(A, buf, wid, lane, SR);
    eval_pose<D, false, WEIGHTED, SpecT>(A.ch, q, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr);
    if (COLL) {
        tl_rows_apply<D, WEIGHTED, SpecT>(A, SR, q, pt, Rt, [&](const float (&g)[D], float r) {
            float u = r;
#pragma unroll
            for (int j = 0; j < D; ++j) u = fma_(g[j], dl[j], u);
#pragma unroll
            for (int j = 0; j < D; ++j) ec[j] = fma_(g[j], u, ec[j]);
        });
    }
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
        const float acc = add(fma_(lam, dl[j], fma_(A.wd2, dd[j], mul(A.wp2, colvec<D>(P, j, t)))), ec[j]);
        st[j * 32 + lane] = -acc;
    }
}

// ---- the unfused path (collision rows, or fewer tiles than the producers of a block can serve: lm_traj_api.cu): the same
// chunks, one thread per waypoint, written to HBM (A.Ag / A.rho, one chunk = one "stage" in tile order) for the solve
// kernel's producers to fetch with bulk-async copies.  Same functions, same bits as the fused path.
template <int D, bool FAST, bool WEIGHTED, typename SpecT, bool COLL>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) tl_assemble_kernel(const __grid_constant__ TArgs A) {
    const Slot s = slot_of_thread(A);
    if (!s.valid) return;
    const uint32_t pk = A.its[s.b];
    if ((pk & 0xffu) >= (uint32_t)A.max_total || (A.gate != nullptr && A.gate[s.b] == 0)) return;
    constexpr int C = Tri<D>::NA + D;
    const int sel = A.sel[s.b];
    const float *qs = A.q + (int64_t)sel * D * A.nS;
    ChunkIn<D> in;
    tl_chunk_load<D>(A, qs, s.wid - s.i, s.i, s.lane, in);
    tl_chunk_normal<D, WEIGHTED, SpecT, COLL>(A, in, sel, s.wid - s.i, s.i, s.lane, A.Ag + s.wid * C * 32);
}
template <int D, bool FAST, bool WEIGHTED, typename SpecT, bool COLL>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) tl_rho_kernel(const __grid_constant__ TArgs A) {
    const Slot s = slot_of_thread(A);
    if (!s.valid) return;
    const uint32_t pk = A.its[s.b];
    if ((pk & 0xffu) >= (uint32_t)A.max_total || !A.ok[s.b] || (A.gate != nullptr && A.gate[s.b] == 0)) return;
    const int sel = A.sel[s.b];
    const float *qs = A.q + (int64_t)sel * D * A.nS;
    ChunkIn<D> in;
    tl_chunk_load<D>(A, qs, s.wid - s.i, s.i, s.lane, in);
    tl_chunk_rho<D, WEIGHTED, SpecT, COLL>(A, in, sel, A.lam[s.b], s.wid - s.i, s.i, s.lane, A.rho + s.wid * D * 32);
}

// Kahan-compensated sum step (explicit intrinsics: the compiler cannot simplify the compensation away)
__device__ __forceinline__ void kahan_add(float &s, float &c, float x) {
    const float y = sub(x, c);
    const float t = add(s, y);
    c = sub(sub(t, s), y);
    s = t;
}

// Total cost of the point tl_cost_kernel evaluated last (tile = blockIdx.x, lane): a block of TL_SUM_WARPS warps
// per tile; warp w sums the waypoints of segment w in order (Kahan), the segment sums are then added
// in segment order.  The summation order depends on n only, never on the batch.  All threads of the
// block must call; the result is valid in warp 0.
constexpr int TL_SUM_WARPS = 8;
__device__ __forceinline__ void tl_sum_cost(const TArgs &A, float (*part)[3][32], float &Fp, float &Fd, float &Fc, float &F) {
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    const float *cp = A.cst;
    const int64_t w0 = (int64_t)blockIdx.x * A.n;
    const int seg = (A.n + TL_SUM_WARPS - 1) / TL_SUM_WARPS;
    const int i0 = wp * seg, i1 = min(A.n, i0 + seg);
    float sm[3] = {0.f, 0.f, 0.f}, cm[3] = {0.f, 0.f, 0.f};
    int i = i0;
    for (; i + 16 <= i1; i += 16) { // 48 independent loads in flight, then the sums in order
        float a[16][3];
#pragma unroll
        for (int u = 0; u < 16; ++u)
#pragma unroll
            for (int c = 0; c < 3; ++c) a[u][c] = cp[toff<3>(w0 + i + u, c, lane)];
#pragma unroll
        for (int u = 0; u < 16; ++u)
#pragma unroll
            for (int c = 0; c < 3; ++c) kahan_add(sm[c], cm[c], a[u][c]);
    }
    for (; i + 4 <= i1; i += 4) {
        float a[4][3];
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int c = 0; c < 3; ++c) a[u][c] = cp[toff<3>(w0 + i + u, c, lane)];
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int c = 0; c < 3; ++c) kahan_add(sm[c], cm[c], a[u][c]);
    }
    for (; i < i1; ++i)
#pragma unroll
        for (int c = 0; c < 3; ++c) kahan_add(sm[c], cm[c], cp[toff<3>(w0 + i, c, lane)]);
#pragma unroll
    for (int c = 0; c < 3; ++c) part[wp][c][lane] = sm[c];
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        sm[c] = 0.f; cm[c] = 0.f;
#pragma unroll
        for (int u = 0; u < TL_SUM_WARPS; ++u) kahan_add(sm[c], cm[c], part[u][c][lane]);
    }
    Fp = sm[0]; Fd = sm[1]; Fc = sm[2];
    F = add(fma_(A.wd2, sm[1], mul(A.wp2, sm[0])), sm[2]);
}

#ifdef LM_TRAJ_PLAIN_KERNELS // non-template kernels: defined in exactly one translation unit (lm_traj_api.cu)
// ---- cost of the current point (entry of lm_traj_run): block of TL_SUM_WARPS warps per tile
__global__ void __launch_bounds__(TL_SUM_WARPS * 32) tl_init_cost_kernel(const __grid_constant__ TArgs A) {
    __shared__ float part[TL_SUM_WARPS][3][32];
    const int64_t b = (int64_t)blockIdx.x * 32 + (threadIdx.x & 31);
    const bool valid = b < A.B;
    float Fp, Fd, Fc, F;
    tl_sum_cost(A, part, Fp, Fd, Fc, F);
    if (!valid || threadIdx.x >= 32) return;
    A.Fp[b] = Fp; A.Fd[b] = Fd; A.Fc[b] = Fc; A.F[b] = F;
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

// ---- bulk-async copy + mbarrier primitives (sm_90+ PTX; one warp is both producer and consumer)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t done = 0;
    while (!done) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    }
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

#ifndef LM_TL_STAGE_BUDGET
#define LM_TL_STAGE_BUDGET (200 * 1024) // shared memory one solve block may spend on its rings
#endif

// One ring stage (floats): [0, NA*32) matrix, then vector 1 (D*32) and, in MODE 1, vector 2 (D*32).
// Each of the two chain warps of a block has its own ring.
template <int D, int MODE> __host__ __device__ constexpr int tl_stage_floats() { return (Tri<D>::NA + (MODE == 0 ? D : 2 * D)) * 32; }
// Waypoints in flight per chain warp in the solve kernel: TL_STAGES_WANT, cut to what the shared-memory budget holds
// (a power of two is not required).  Round 1, when the stages were filled from HBM (n = 300, us per iteration at
// B = 4096 / 16384): 2 stages 486 / 1276, 4: 403 / 1279, 8: 387 / --.
#ifndef LM_TL_STAGES
#define LM_TL_STAGES 8
#endif
constexpr int TL_STAGES_WANT = LM_TL_STAGES;
// Block shapes of the solve kernel (chosen per launch, lm_traj_launch.h): warps 0, 1 are the chains, every further warp is
// a producer and serves chain (warp & 1).  Measured on B200, n = 300, ms per iteration with one refinement step (fused
// path; threads per block = 32 (2 + 2 producers per chain)):      256      320      384      512
//                                     4096 trajectories (128 tiles, one block per SM)     0.341    0.340    0.326    0.328
//                                     16384 trajectories (512 tiles)                      1.102    1.350    1.300    1.299
// Keeping the producers off the two scheduler partitions the chains run on (idle warps in between) made no difference
// (0.336 with 4 producers per chain).  A producer warp is never two ring turns ahead of its own last wait as long as
// producers per chain <= ring stages.
constexpr int TL_SOLVE_MAX_THREADS = 512;
constexpr int TL_SOLVE_THREADS_MANY_TILES = 256; // more tiles than SMs: 2 chains + 3 producers each, two blocks per SM
constexpr int TL_SOLVE_THREADS_FEW_TILES = 384;  // at most one block per SM: 2 chains + 5 producers each
constexpr int TL_SOLVE_THREADS_HBM = 128;        // unfused: 2 chains + 1 copy-issuing producer each
static_assert((TL_SOLVE_THREADS_FEW_TILES / 32 - 2) / 2 <= TL_STAGES_WANT, "more producers per chain than ring stages");
template <int D, int MODE> __host__ __device__ constexpr int tl_stages() {
    const size_t per_stage = (size_t)2 * tl_stage_floats<D, MODE>() * sizeof(float);
    const int fit = (int)((size_t)LM_TL_STAGE_BUDGET / per_stage);
    return fit > TL_STAGES_WANT ? TL_STAGES_WANT : fit;
}
template <int D, int MODE> __host__ __device__ constexpr size_t tl_solve_smem_bytes() {
    return (size_t)2 * tl_stages<D, MODE>() * tl_stage_floats<D, MODE>() * sizeof(float);
}

// ---- block-tridiagonal solve: one block per tile of 32 trajectories -- two chain warps and a few producer warps for
// each of them -- lane = trajectory.
// Two-sided ("twisted") block elimination halves the sequential chain: with m = n / 2,
//   warp 0 eliminates i = 0, 1, .., m-1      (S_i = T_i - w_d^4 S_{i-1}^-1,  h_i = g_i + w_d^2 z_{i-1}),
//   warp 1 eliminates i = n-1, n-2, .., m+1  (S_i = T_i - w_d^4 S_{i+1}^-1,  h_i = g_i + w_d^2 z_{i+1}),
//   z_i = S_i^-1 h_i; they meet at the middle block
//   S_m = T_m - w_d^4 (S_{m-1}^-1 + S_{m+1}^-1),  x_m = S_m^-1 (g_m + w_d^2 (z_{m-1} + z_{m+1})),
// and both substitute outwards from x_m:  x_i = z_i + w_d^2 S_i^-1 x_{i+-1}.
//   MODE 0: factor (stores W_i = -S_i^-1) and solve for g;                      delta  = -x
//   MODE 1: re-solve with the stored W_i for rho (iterative refinement);        delta +=  x
// What a chain consumes is PRODUCED IN THE BLOCK, not fetched: the producer warps of a chain take the waypoints of its
// sequence round robin and write T_i (without the diagonal shift) and g_i (MODE 0: tl_chunk_normal) or rho_i (MODE 1:
// tl_chunk_rho, next to the bulk-async copy of W_i) into the chain's shared-memory ring, up to TL_STAGES waypoints ahead of the
// recurrence; w_p^2 J^T J, g and rho never exist in HBM.  Per stage an "empty" mbarrier (armed by the consumer's lane 0
// once all its lanes have read the stage) and a "full" one (the producer's lane 0 arrives after its warp's stores; the
// byte count of a bulk copy is posted on the same barrier).  For the substitution phase producer 0 of each chain issues
// the bulk-async copies of W_i, z_i (and the old delta_i) as before.  The chains only wait, load and compute.
// fewer tiles than this: the unfused path (every SM assembles) beats a few producer warps per chain (lm_traj_api.cu)
#ifndef LM_TL_FUSED_MIN_TILES
#define LM_TL_FUSED_MIN_TILES 96
#endif
constexpr int64_t TL_FUSED_MIN_TILES = LM_TL_FUSED_MIN_TILES;
// FUSED = false: the chunks come from HBM instead (A.Ag / A.rho, written by tl_assemble_kernel / tl_rho_kernel): producer
// 0 of each chain fetches them with bulk-async copies, the other producer warps idle.
template <int D, int MODE, bool FUSED, bool WEIGHTED, typename SpecT>
__global__ void __launch_bounds__(TL_SOLVE_MAX_THREADS) tl_solve_kernel(const __grid_constant__ TArgs A) {
    constexpr int NA = Tri<D>::NA, SF = tl_stage_floats<D, MODE>();
    constexpr int TL_STAGES = tl_stages<D, MODE>();
    // the mbarrier parity argument (above) on the stage count this instantiation really has, not the wanted one
    static_assert(!FUSED || (TL_SOLVE_THREADS_FEW_TILES / 32 - 2) / 2 <= TL_STAGES, "more producers per chain than ring stages");
    static_assert(TL_STAGES >= 1, "no ring stage fits the shared-memory budget");
    constexpr uint32_t FULL_COUNT = (FUSED && MODE == 1) ? 2u : 1u; // fused MODE 1: the poster of the copy's byte count + the writer of rho
    extern __shared__ __align__(128) float smem[];
    __shared__ __align__(8) uint64_t full_all[2][TL_STAGES], empty_all[2][TL_STAGES];
    __shared__ float xch[NA + D][32]; // warp 1 -> warp 0: W_{m+1}, z_{m+1}
    __shared__ float xmid[D][32];     // warp 0 -> both: x_m
    __shared__ int okx[2][32];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5; // warps 0, 1: the two chains; warps 2..: their producers
    const int npw = ((int)(blockDim.x >> 5) - 2) / 2; // producer warps per chain
    const int pq = wp & 1, pi = (wp - 2) >> 1;         // a producer's chain and its index among that chain's producers
    const int64_t bt = blockIdx.x;
    const int64_t b = bt * 32 + lane;
    const bool valid = b < A.B;
    const uint32_t pk = valid ? A.its[b] : 0xffu;
    const bool active = valid && ((pk & 0xffu) < (uint32_t)A.max_total) && (MODE == 0 || A.ok[b] != 0) &&
                        (A.gate == nullptr || A.gate[b] != 0);
    if (!__any_sync(0xffffffffu, active)) return; // the same lanes in every warp: block-uniform
    const int sel = valid ? A.sel[b] : 0;
    const int n = A.n;
    const int64_t w0 = bt * n;
    const int m = n / 2;
    // sequence of warp q: q = 0 eliminates 0 .. m-1 and then the middle block m; q = 1 eliminates n-1 .. m+1
    auto len_of = [&](int q) { return q == 0 ? m : n - 1 - m; };          // waypoints warp q eliminates
    auto uses1_of = [&](int q) { return len_of(q) + (q == 0 ? 1 : 0); };  // ring uses of its elimination phase
    auto idx_of = [&](int q, int k) { return q == 0 ? k : n - 1 - k; };   // k-th waypoint of its sequence (idx(0, m) = m)

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < TL_STAGES; ++s) {
            mbar_init(&full_all[0][s], FULL_COUNT); mbar_init(&full_all[1][s], FULL_COUNT);
            mbar_init(&empty_all[0][s], 1); mbar_init(&empty_all[1][s], 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (wp >= 2) { // ---- the producers: warps 2, 4, 6, .. feed the ring of warp 0, warps 3, 5, 7, .. that of warp 1
        const int q = pq;
        float *ring_q = smem + (size_t)q * TL_STAGES * SF;
        const float *qs = A.q + (int64_t)sel * D * A.nS; // the lane's current joint buffer
        const float lam = valid ? A.lam[b] : 1.f;
        // use u of a stage may be filled once use u - TL_STAGES has been released (uses are numbered per chain, both
        // phases).  A producer is never two ring turns ahead of the consumer (producers per chain <= TL_STAGES), so the parity is unambiguous.
        auto wait_free = [&](int k) {
            if (k >= TL_STAGES) {
                if (lane == 0) mbar_wait(&empty_all[q][k % TL_STAGES], (uint32_t)(((k / TL_STAGES) - 1) & 1));
                __syncwarp();
            }
        };
        const int u = uses1_of(q);
        if (FUSED) {
            // the inputs of a producer's NEXT chunk are requested before it waits for / computes the current one
            ChunkIn<D> nxt;
            if (pi < u) tl_chunk_load<D>(A, qs, w0, idx_of(q, pi), lane, nxt);
            for (int k = pi; k < u; k += npw) {
                const int s = k % TL_STAGES;
                const ChunkIn<D> cur = nxt;
                if (k + npw < u) tl_chunk_load<D>(A, qs, w0, idx_of(q, k + npw), lane, nxt);
                wait_free(k);
                float *st = ring_q + (size_t)s * SF;
                const int i = idx_of(q, k);
                if (MODE == 0) {
                    tl_chunk_normal<D, WEIGHTED, SpecT, false>(A, cur, sel, w0, i, lane, st);
                } else {
                    if (lane == 0) {
                        mbar_expect_tx(&full_all[q][s], NA * 128u);
                        bulk_g2s(st, A.V + (w0 + i) * NA * 32, NA * 128u, &full_all[q][s]);
                    }
                    tl_chunk_rho<D, WEIGHTED, SpecT, false>(A, cur, sel, lam, w0, i, lane, st + NA * 32);
                }
                __syncwarp(); // every lane's stores precede the arrival below
                if (lane == 0) mbar_arrive(&full_all[q][s]);
            }
        } else if (pi == 0 && lane == 0) {
            for (int k = 0; k < u; ++k) {
                const int s = k % TL_STAGES;
                if (k >= TL_STAGES) mbar_wait(&empty_all[q][s], (uint32_t)(((k / TL_STAGES) - 1) & 1));
                uint64_t *bar = &full_all[q][s];
                float *dst = ring_q + (size_t)s * SF;
                const int64_t wid = w0 + idx_of(q, k);
                mbar_expect_tx(bar, (NA + D) * 128u);
                if (MODE == 0) {
                    bulk_g2s(dst, A.Ag + wid * (NA + D) * 32, (NA + D) * 128u, bar);
                } else {
                    bulk_g2s(dst, A.V + wid * NA * 32, NA * 128u, bar);
                    bulk_g2s(dst + NA * 32, A.rho + wid * D * 32, D * 128u, bar);
                }
            }
        }
        __syncthreads(); // (1) warp 1 has handed its last block to warp 0
        __syncthreads(); // (2) the chunks written by the elimination are ordered before the copies below
        fence_proxy_async();
        if (pi == 0 && lane == 0) {
            const int l = len_of(q);
            for (int j = 0; j < l; ++j) {
                const int kk = u + j, s = kk % TL_STAGES;
                if (kk >= TL_STAGES) mbar_wait(&empty_all[q][s], (uint32_t)(((kk / TL_STAGES) - 1) & 1));
                uint64_t *bar = &full_all[q][s];
                float *dst = ring_q + (size_t)s * SF;
                const int64_t wid = w0 + idx_of(q, l - 1 - j);
                mbar_expect_tx(bar, (NA + D + (MODE == 1 ? D : 0)) * 128u);
                bulk_g2s(dst, A.V + wid * NA * 32, NA * 128u, bar);
                bulk_g2s(dst + NA * 32, A.z + wid * D * 32, D * 128u, bar);
                if (MODE == 1) bulk_g2s(dst + (NA + D) * 32, A.delta + wid * D * 32, D * 128u, bar);
                if (FULL_COUNT == 2u) mbar_arrive(bar); // the barrier counts two arrivals per use in the fused MODE 1
            }
        }
        __syncthreads(); // (3) the verdicts of the two chains
        return;
    }

    // ---- the two chains
    const float lam = valid ? A.lam[b] : 1.f;
    float *ring = smem + (size_t)wp * TL_STAGES * SF;
    uint64_t *bars = full_all[wp], *empt = empty_all[wp];
    const int len = len_of(wp);
    const int uses1 = uses1_of(wp);
    auto idx = [&](int k) { return idx_of(wp, k); };

    float W[NA], zp[D];
#pragma unroll
    for (int t = 0; t < NA; ++t) W[t] = 0.f;
#pragma unroll
    for (int j = 0; j < D; ++j) zp[j] = 0.f;
    bool ok = true;

    // one elimination step on the chunk in stage k of this warp's ring; `Wo`, `zo`: the contribution of the
    // other side (only at the middle block), zero otherwise
    auto eliminate = [&](int k, int i, const float (&Wo)[NA], const float (&zo)[D], bool middle) {
        const int s = k % TL_STAGES;
        mbar_wait(&bars[s], (uint32_t)((k / TL_STAGES) & 1));
        const float *st = ring + (size_t)s * SF;
        float S[NA], rhs[D];
#pragma unroll
        for (int t = 0; t < NA; ++t) S[t] = st[t * 32 + lane];
#pragma unroll
        for (int r = 0; r < D; ++r) rhs[r] = st[(NA + r) * 32 + lane];
        __syncwarp(); // every lane has read the stage: it may be refilled (the copy lands long after these loads)
        if (lane == 0) mbar_arrive(&empt[s]);
        const int64_t wid = w0 + i;
        if (MODE == 0) {
            const float ci = (n == 1) ? 0.f : ((i == 0 || i == n - 1) ? 1.f : 2.f);
            const float dg = fma_(ci, A.wd2, lam);
#pragma unroll
            for (int r = 0; r < D; ++r) S[tri(r, r)] = add(S[tri(r, r)], dg);
            // S_i = T_i - w_d^4 S_prev^-1 = T_i + w_d^4 W_prev (+ the other side's at the middle)
#pragma unroll
            for (int t = 0; t < NA; ++t) S[t] = fma_(A.wd4, W[t], S[t]);
            if (middle) {
#pragma unroll
                for (int t = 0; t < NA; ++t) S[t] = fma_(A.wd4, Wo[t], S[t]);
            }
            ok = sweep_neg_inverse<D>(S) && ok;
            if (active) {
#pragma unroll
                for (int t = 0; t < NA; ++t) A.V[toff<NA>(wid, t, lane)] = S[t];
            }
        }
#pragma unroll
        for (int t = 0; t < NA; ++t) W[t] = S[t];
        // h_i = rhs_i + w_d^2 z_prev;  z_i = S_i^-1 h_i = -(W_i h_i)
        float h[D], y[D];
#pragma unroll
        for (int r = 0; r < D; ++r) {
            h[r] = fma_(A.wd2, zp[r], rhs[r]);
            if (middle) h[r] = fma_(A.wd2, zo[r], h[r]);
        }
        symv<D>(W, h, y);
#pragma unroll
        for (int r = 0; r < D; ++r) zp[r] = -y[r];
        if (active && !middle) {
#pragma unroll
            for (int r = 0; r < D; ++r) A.z[toff<D>(wid, r, lane)] = zp[r];
        }
    };

    // ---- elimination from both ends
    {
        float Wz[NA], zz[D];
#pragma unroll
        for (int t = 0; t < NA; ++t) Wz[t] = 0.f;
#pragma unroll
        for (int r = 0; r < D; ++r) zz[r] = 0.f;
        for (int k = 0; k < len; ++k) eliminate(k, idx(k), Wz, zz, false);
    }
    if (wp == 1) { // hand W_{m+1}, z_{m+1} (zeros when this warp had nothing to eliminate) to warp 0
#pragma unroll
        for (int t = 0; t < NA; ++t) xch[t][lane] = W[t];
#pragma unroll
        for (int r = 0; r < D; ++r) xch[NA + r][lane] = zp[r];
    }
    __syncthreads();
    float amax = 0.f;
    if (wp == 0) { // the middle block: x_m
        float Wo[NA], zo[D];
#pragma unroll
        for (int t = 0; t < NA; ++t) Wo[t] = xch[t][lane];
#pragma unroll
        for (int r = 0; r < D; ++r) zo[r] = xch[NA + r][lane];
        eliminate(len, m, Wo, zo, true);
        const int64_t wid = w0 + m;
#pragma unroll
        for (int r = 0; r < D; ++r) {
            xmid[r][lane] = zp[r];
            const float dv = (MODE == 0) ? -zp[r] : add(active ? A.delta[toff<D>(wid, r, lane)] : 0.f, zp[r]);
            if (active) A.delta[toff<D>(wid, r, lane)] = dv;
            amax = fmaxf(amax, fabsf(dv));
        }
    }
    // the chunks written above are read back by bulk-async copies: order the generic writes before them
    __threadfence();
    fence_proxy_async();
    __syncthreads();

    // ---- substitution outwards from the middle: x_i = z_i + w_d^2 S_i^-1 x_next = z_i - w_d^2 W_i x_next
    float x[D];
#pragma unroll
    for (int r = 0; r < D; ++r) x[r] = xmid[r][lane];
    for (int j = 0; j < len; ++j) {
        const int kk = uses1 + j;
        const int s = kk % TL_STAGES;
        const int i = idx(len - 1 - j);
        mbar_wait(&bars[s], (uint32_t)((kk / TL_STAGES) & 1));
        const float *st = ring + (size_t)s * SF;
        float zi[D], dold[D];
#pragma unroll
        for (int t = 0; t < NA; ++t) W[t] = st[t * 32 + lane];
#pragma unroll
        for (int r = 0; r < D; ++r) {
            zi[r] = st[(NA + r) * 32 + lane];
            dold[r] = (MODE == 1) ? st[(NA + D + r) * 32 + lane] : 0.f;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empt[s]);
        float y[D];
        symv<D>(W, x, y);
        const int64_t wid = w0 + i;
#pragma unroll
        for (int r = 0; r < D; ++r) {
            x[r] = fma_(-A.wd2, y[r], zi[r]);
            const float dv = (MODE == 0) ? -x[r] : add(dold[r], x[r]);
            if (active) A.delta[toff<D>(wid, r, lane)] = dv;
            amax = fmaxf(amax, fabsf(dv));
        }
    }
    ok = ok && (amax < 1e30f); // NaN compares false
    okx[wp][lane] = ok ? 1 : 0;
    __syncthreads();
    if (wp == 0 && active) {
        const bool both = okx[0][lane] && okx[1][lane];
        if (MODE == 0) A.ok[b] = both ? 1 : 0;
        else if (!both) A.ok[b] = 0;
    }
}

// ---- cost of a point: thread per waypoint.
//   INIT = false: the trial point q+ = clamp(q + delta) -> the candidate joint buffer (1 - sel), its cost
//                 terms -> cst.  Only FK and the residual are evaluated: the Jacobian of an accepted point is formed by the
//                 next solve's producers.
//   INIT = true:  the cost terms of the current point (entry of lm_traj_run).
template <int D, bool FAST, bool WEIGHTED, typename SpecT, bool COLL, bool INIT>
__global__ void __launch_bounds__(LM_MAX_THREADS, LM_MIN_BLOCKS) tl_cost_kernel(const __grid_constant__ TArgs A) {
    const Slot s = slot_of_thread(A);
    if (!s.valid) return;
    // every load below is issued before the first use: the joint values of BOTH buffers are fetched and the
    // trajectory's `sel` picks afterwards (a dependent address would cost one more DRAM round trip)
    const uint32_t pk = A.its[s.b];
    const int sel = A.sel[s.b];
    const bool ok = INIT ? false : (A.ok[s.b] != 0);
    const float *q0 = A.q, *q1 = A.q + (int64_t)D * A.nS;
    float ra[2][D], rb[2][D], rd[2][D]; // this waypoint and the next one (the differencing cost of row i)
#pragma unroll
    for (int u = 0; u < 2; ++u) {
        const bool there = (u == 0) || (s.i + 1 < A.n);
        const int64_t wid = s.wid + u;
#pragma unroll
        for (int j = 0; j < D; ++j) {
            ra[u][j] = there ? q0[toff<D>(wid, j, s.lane)] : 0.f;
            rb[u][j] = there ? q1[toff<D>(wid, j, s.lane)] : 0.f;
            rd[u][j] = (there && !INIT) ? A.delta[toff<D>(wid, j, s.lane)] : 0.f;
        }
    }
    float pt[3], Rt[3][3];
    tl_load_target(A, s, pt, Rt);
    if (!INIT && ((pk & 0xffu) >= (uint32_t)A.max_total || (A.gate != nullptr && A.gate[s.b] == 0))) return;
    float qt[D], qn[D];
    bool clamped = false;
    auto point_of = [&](int u, int j, bool &cl) {
        const float qv = sel ? rb[u][j] : ra[u][j];
        if (INIT) return qv;
        const float t = ok ? add(qv, rd[u][j]) : qv;
        const float c = fminf(fmaxf(t, A.ch.lo[j]), A.ch.hi[j]);
        cl = cl || (c != t);
        return c;
    };
    float fd = 0.f;
#pragma unroll
    for (int j = 0; j < D; ++j) {
        bool dummy = false;
        qt[j] = point_of(0, j, clamped);
        qn[j] = (s.i + 1 < A.n) ? point_of(1, j, dummy) : 0.f;
        if (!INIT) A.q[(int64_t)(1 - sel) * D * A.nS + toff<D>(s.wid, j, s.lane)] = qt[j];
        if (s.i + 1 < A.n) {
            const float t = sub(qn[j], qt[j]);
            fd = fma_(t, t, fd);
        }
    }
    // "a trial point of this trajectory was clamped": integer atomic (order-free), skipped once the bit is seen set
    if (!INIT && clamped && !((__ldcg(A.its + s.b) >> 8) & 32u)) atomicOr(A.its + s.b, 32u << 8);
    float fc = 0.f;
    Pose<D> P;
    if (COLL) { // lanes = trajectories (tile order); tl_cost_window_kernel is the same with lanes = consecutive waypoints
        CapsWorld W;
        CapsSink sink(A.caps, W);
        sink.base();
        eval_pose<D, FAST, WEIGHTED, SpecT, false, CapsSink>(A.ch, qt, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr, nullptr, sink);
        // the rows of this point, kept for the assembly and the refinement residual (tl_rows_fetch)
        constexpr int RC = tl_row_comps<D>();
        const int dst = INIT ? sel : 1 - sel;
        float *rw = A.rows + (int64_t)dst * RC * A.nS + toff<RC>(s.wid, 0, s.lane); // component c at rw[c * 32]
        int cnt = 0;
        coll_rows<D, SpecT>(A.ch, A.caps, W, P, [&](const float (&g)[D], float r) {
            fc = fma_(r, r, fc);
            if (cnt < TL_RMAX) {
#pragma unroll
                for (int j = 0; j < D; ++j) rw[j * 32] = g[j];
                rw[D * 32] = r;
                rw += (D + 1) * 32;
            }
            ++cnt;
        });
        A.rcnt[(int64_t)dst * A.nS + s.wid * 32 + s.lane] = cnt > TL_RMAX ? TL_ROWS_OVERFLOW : cnt;
    } else {
        eval_pose<D, FAST, WEIGHTED, SpecT, false>(A.ch, qt, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr);
    }
    A.cst[toff<3>(s.wid, 0, s.lane)] = P.F;
    A.cst[toff<3>(s.wid, 1, s.lane)] = fd;
    A.cst[toff<3>(s.wid, 2, s.lane)] = fc;
    if (!INIT && A.trace_q != nullptr) {
        const int64_t W = A.B * A.n, w = s.b * A.n + s.i;
#pragma unroll
        for (int j = 0; j < D; ++j) A.trace_q[(int64_t)j * W + w] = qt[j];
    }
}

// ---- the same for the step WITH collision rows, lanes along the PATH.  In tile order the 32 lanes of a warp are 32
// different trajectories at one waypoint index: their surviving pair lists are uncorrelated and the pair loops run with a
// handful of lanes (ncu, round 2: 13.8 of 32 threads per instruction, 5800 warp-instructions per chunk).  Consecutive
// waypoints of ONE trajectory are millimetres apart and see the same obstacles, so here a block takes a tile and a window
// of 32 waypoints, transposes it through shared memory, and every warp walks 32 consecutive waypoints of one trajectory
// (lane = waypoint): the lists of its lanes are nearly the same and the loops run full.  Same per-waypoint functions as
// tl_cost_kernel, so every output has the same bits.
//   phase 1 (lane = trajectory, coalesced): trial point of the window's 33 chunks -> shared memory (and the candidate
//            joint buffer, the "clamped" bit), targets -> shared memory
//   phase 2 (lane = waypoint): FK with the capsule sink, pair loops, rows -> HBM (sparse), cost terms and row count ->
//            shared memory
//   phase 3 (lane = trajectory, coalesced): cost terms and row counts -> HBM
constexpr int TL_CW = 32;            // waypoints per window
constexpr int TL_CW_THREADS = 256;   // 8 warps: 4 trajectories each in phase 2
template <int D> __host__ __device__ constexpr size_t tl_cost_window_smem() {
    return sizeof(float) * ((size_t)(TL_CW + 1) * D * 33 + (size_t)TL_CW * 7 * 33); // the outputs reuse the targets' columns
}
template <int D, bool WEIGHTED, typename SpecT, bool INIT>
__global__ void __launch_bounds__(TL_CW_THREADS, 3) tl_cost_window_kernel(const __grid_constant__ TArgs A) {
    extern __shared__ __align__(16) float smem_cw[];
    float *qs = smem_cw;                                  // [TL_CW + 1][D][33]: trial point of waypoint i0 + l, joint j, trajectory b
    float *tg = qs + (TL_CW + 1) * D * 33;                // [TL_CW][7][33]: targets
    float *co = tg;                                       // [TL_CW][4][33]: F_pose, diff, coll, row count (as int bits) -- column b of the
                                                          // targets is dead once the warp that owns trajectory b has read it
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int nwin = (A.n + TL_CW - 1) / TL_CW;
    const int64_t bt = blockIdx.x / nwin;
    const int i0 = (int)(blockIdx.x - bt * nwin) * TL_CW;
    const int n = A.n;
    // ---- phase 1: lane = trajectory
    {
        const int64_t b = bt * 32 + lane;
        const bool valid = b < A.B;
        const uint32_t pk = valid ? A.its[b] : 0xffu;
        const int sel = valid ? A.sel[b] : 0;
        const bool ok = INIT ? false : (valid && A.ok[b] != 0);
        const bool live = valid && (INIT || !((pk & 0xffu) >= (uint32_t)A.max_total || (A.gate != nullptr && A.gate[b] == 0)));
        const float *qcur = A.q + (int64_t)sel * D * A.nS;
        float *qcand = A.q + (int64_t)(1 - sel) * D * A.nS;
        bool clamped = false;
        for (int l = wp; l <= TL_CW; l += nw) {
            const int i = i0 + l;
            if (i >= n) continue;
            const int64_t wid = bt * n + i;
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const float qv = qcur[toff<D>(wid, j, lane)];
                float c = qv;
                if (!INIT) {
                    const float t = ok ? add(qv, A.delta[toff<D>(wid, j, lane)]) : qv;
                    c = fminf(fmaxf(t, A.ch.lo[j]), A.ch.hi[j]);
                    if (l < TL_CW) {
                        clamped = clamped || (c != t);
                        if (live) qcand[toff<D>(wid, j, lane)] = c;
                    }
                }
                qs[(l * D + j) * 33 + lane] = c;
            }
            if (l < TL_CW) {
                if (A.shared_targets) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) tg[(l * 7 + c) * 33 + lane] = __ldg(A.tp + (int64_t)c * n + i);
#pragma unroll
                    for (int c = 0; c < 4; ++c) tg[(l * 7 + 3 + c) * 33 + lane] = __ldg(A.tq + (int64_t)c * n + i);
                } else {
#pragma unroll
                    for (int c = 0; c < 3; ++c) tg[(l * 7 + c) * 33 + lane] = __ldg(A.tp + toff<3>(wid, c, lane));
#pragma unroll
                    for (int c = 0; c < 4; ++c) tg[(l * 7 + 3 + c) * 33 + lane] = __ldg(A.tq + toff<4>(wid, c, lane));
                }
            }
        }
        // "a trial point of this trajectory was clamped": integer atomic (order-free), skipped once the bit is seen set
        if (!INIT && live && clamped && !((__ldcg(A.its + b) >> 8) & 32u)) atomicOr(A.its + b, 32u << 8);
    }
    __syncthreads();
    // ---- phase 2: lane = waypoint i0 + lane of trajectory bb (warp-uniform)
    for (int tb = wp; tb < 32; tb += nw) {
        const int64_t bb = bt * 32 + tb;
        if (bb >= A.B) break;
        const uint32_t pk = A.its[bb];
        if (!INIT && ((pk & 0xffu) >= (uint32_t)A.max_total || (A.gate != nullptr && A.gate[bb] == 0))) continue;
        const int sel = A.sel[bb];
        const int i = i0 + lane;
        const bool have = i < n;
        const int lc = have ? lane : 0; // lanes beyond the end of the path shadow the window's first waypoint, never store
        float qt[D], qn[D], fd = 0.f;
#pragma unroll
        for (int j = 0; j < D; ++j) {
            qt[j] = qs[(lc * D + j) * 33 + tb];
            qn[j] = (have && i + 1 < n) ? qs[((lc + 1) * D + j) * 33 + tb] : 0.f;
            if (have && i + 1 < n) {
                const float t = sub(qn[j], qt[j]);
                fd = fma_(t, t, fd);
            }
        }
        const float pt[3] = {tg[(lc * 7 + 0) * 33 + tb], tg[(lc * 7 + 1) * 33 + tb], tg[(lc * 7 + 2) * 33 + tb]};
        float Rt[3][3];
        quat_to_cols(tg[(lc * 7 + 3) * 33 + tb], tg[(lc * 7 + 4) * 33 + tb], tg[(lc * 7 + 5) * 33 + tb], tg[(lc * 7 + 6) * 33 + tb], Rt);
        Pose<D> P;
        CapsWorld W;
        CapsSink sink(A.caps, W);
        sink.base();
        eval_pose<D, false, WEIGHTED, SpecT, false, CapsSink>(A.ch, qt, pt, Rt, A.w_pos, A.w_rot, P, nullptr, nullptr, nullptr, sink);
        // the rows of this point, kept for the assembly and the refinement residual (tl_rows_fetch)
        constexpr int RC = tl_row_comps<D>();
        const int dst = INIT ? sel : 1 - sel;
        const int64_t wid = bt * n + (have ? i : i0);
        float *rw = A.rows + (int64_t)dst * RC * A.nS + toff<RC>(wid, 0, tb); // component c at rw[c * 32]
        int cnt = 0;
        float fc = 0.f;
        coll_rows<D, SpecT>(A.ch, A.caps, W, P, [&](const float (&g)[D], float r) {
            fc = fma_(r, r, fc);
            if (cnt < TL_RMAX && have) {
#pragma unroll
                for (int j = 0; j < D; ++j) rw[j * 32] = g[j];
                rw[D * 32] = r;
                rw += (D + 1) * 32;
            }
            ++cnt;
        });
        __syncwarp(); // every lane of this warp has read its target from column tb: the column may be overwritten
        if (have) {
            co[(lane * 4 + 0) * 33 + tb] = P.F;
            co[(lane * 4 + 1) * 33 + tb] = fd;
            co[(lane * 4 + 2) * 33 + tb] = fc;
            co[(lane * 4 + 3) * 33 + tb] = __int_as_float(cnt > TL_RMAX ? TL_ROWS_OVERFLOW : cnt);
            if (!INIT && A.trace_q != nullptr) {
                const int64_t Wn = A.B * n, w = bb * n + i;
#pragma unroll
                for (int j = 0; j < D; ++j) A.trace_q[(int64_t)j * Wn + w] = qt[j];
            }
        }
    }
    __syncthreads();
    // ---- phase 3: lane = trajectory
    {
        const int64_t b = bt * 32 + lane;
        const bool valid = b < A.B;
        const uint32_t pk = valid ? A.its[b] : 0xffu;
        const bool live = valid && (INIT || !((pk & 0xffu) >= (uint32_t)A.max_total || (A.gate != nullptr && A.gate[b] == 0)));
        const int sel = valid ? A.sel[b] : 0;
        const int dst = INIT ? sel : 1 - sel;
        if (live) {
            for (int l = wp; l < TL_CW; l += nw) {
                const int i = i0 + l;
                if (i >= n) break;
                const int64_t wid = bt * n + i;
#pragma unroll
                for (int c = 0; c < 3; ++c) A.cst[toff<3>(wid, c, lane)] = co[(l * 4 + c) * 33 + lane];
                A.rcnt[(int64_t)dst * A.nS + wid * 32 + lane] = __float_as_int(co[(l * 4 + 3) * 33 + lane]);
            }
        }
    }
}

#ifdef LM_TRAJ_PLAIN_KERNELS
// ---- accept / reject and the lambda update, per trajectory (DESIGN T3 = R5 on the total cost)
__global__ void __launch_bounds__(TL_SUM_WARPS * 32) tl_decide_kernel(const __grid_constant__ TArgs A) {
    __shared__ float part[TL_SUM_WARPS][3][32];
    const int64_t b = (int64_t)blockIdx.x * 32 + (threadIdx.x & 31);
    const bool valid = b < A.B;
    const int s = valid ? A.sel[b] : 0;
    float Fp, Fd, Fc, Ft;
    tl_sum_cost(A, part, Fp, Fd, Fc, Ft);
    if (!valid || threadIdx.x >= 32) return;
    uint32_t pk = A.its[b];
    uint32_t k = pk & 0xffu, st = pk >> 8;
    if (k >= (uint32_t)A.max_total || (A.gate != nullptr && A.gate[b] == 0)) return;
    const bool ok = A.ok[b] != 0;
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
        A.F[b] = Ft; A.Fp[b] = Fp; A.Fd[b] = Fd; A.Fc[b] = Fc;
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
    if (b >= A.Bt * 32) return;
    A.lam[b] = (lam_in && b < A.B) ? lam_in[b] : lambda0;
    A.its[b] = 0u;
    A.mask[b] = 0ull;
    A.sel[b] = 0;
    A.ok[b] = 0;
}
#endif

} // namespace lmk
