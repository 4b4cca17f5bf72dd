// lm_search_api.cu -- C ABI of the global discrete search over K candidate trajectories of one path
// (include/lm.h, lm_search*; sec. III-B).
//
// Two kernels.  search_edges_kernel is the parallel part: block (i, y) holds the K configurations of
// timesteps i-1 and i in shared memory and writes a slice of the K x K edge costs max_j |dq_j| (coalesced);
// the y = 0 blocks also write the K node penalties of timestep i.  search_dp_kernel is the sequential part: one thread-block cluster
// walks the n layers, G lanes per node scan its K incoming edges (L2-resident), then CTA 0 picks the cheapest
// end node, reads the path back through the stored predecessors and gathers xi_search.  Every
// subtraction and addition is a single fp32 operation rounded to nearest, max and < are exact, ties go
// to the lowest candidate index: the choice is reproducible bit for bit.
#include "lm_ctx.h"

#include <cooperative_groups.h>
#include <cmath>
#include <cstring>
#include <mutex>

namespace cg = cooperative_groups;

using namespace lmk;

namespace {

constexpr int EDGE_THREADS = 256;
constexpr int DP_THREADS = 512;
constexpr int DP_CLUSTER = 8;   // portable maximum
constexpr int DP_BATCH = 12;    // edge costs per lane prefetched into registers before the wait that closes a layer
constexpr size_t SMEM_OPT_IN = 232448; // 227 KB

struct SLayout {
    size_t edges, pen, clear, pred, choice, xi, result, all;
};

struct DpShape { int KC, G, KP, threads; };
// KC nodes per CTA, G lanes per node (a power of two, KC * G <= DP_THREADS), KP = row stride of the edge costs and
// length of the cost vectors: K rounded up so that every lane reads whole batches; the padding holds +inf.
DpShape dp_shape(int64_t K) {
    DpShape s{};
    s.KC = (int)((K + DP_CLUSTER - 1) / DP_CLUSTER);
    s.G = 1;
    while (s.G < 32 && 2 * s.G * s.KC <= DP_THREADS) s.G *= 2;
    const int chunk = s.G * DP_BATCH;
    s.KP = (int)((K + chunk - 1) / chunk * chunk);
    s.threads = (s.KC * s.G + 31) / 32 * 32;
    return s;
}

SLayout make_slayout(int d, int64_t K, int64_t n) {
    SLayout L{};
    const size_t KP = (size_t)dp_shape(K).KP;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
    L.edges = take(4 * (size_t)(n > 1 ? n - 1 : 1) * (size_t)K * KP);
    L.pen = take(4 * (size_t)n * (size_t)K);
    L.clear = take(4 * (size_t)n * (size_t)K);
    L.pred = take(2 * (size_t)n * (size_t)K);
    L.choice = take(4 * (size_t)n);
    L.xi = take(4 * (size_t)n * (size_t)d);
    L.result = take(16);
    L.all = off;
    return L;
}

struct SArgs {
    int32_t dof, n, K, KP, KC, pred_in_smem, use_clear;
    int64_t W;
    uint32_t prismatic_mask;
    float margin_rev, margin_pris, pen_limit, pen_collision;
    float lo[MAX_DOF], hi[MAX_DOF];
    const float *q;     // [d][W], w = k * n + i
    const float *clear; // [W]
    float *edges;       // [n-1][K][KP]: edges[(i-1)][k][k'] = step from (i-1, k') to (i, k); +inf for k' >= K
    float *pen;         // [n][K]
    uint16_t *pred;     // [n][K]
    int32_t *choice;    // [n]
    float *xi;          // [d][n]
    float *result;      // [2]
};

// Block (i, y): for i >= 1 the edge costs between layers i-1 and i into a slice of the nodes k; blocks with y = 0
// also write the penalties of layer i.  A thread owns one predecessor k' (its D joint values stay in registers) and
// walks the rows k of the slice: per edge D broadcast shared-memory reads, D subtractions, D max.
template <int D>
__global__ void __launch_bounds__(EDGE_THREADS) search_edges_kernel(const SArgs A) {
    extern __shared__ float sm[];
    const int K = A.K, KP = A.KP, i = blockIdx.x, t = threadIdx.x;
    float *qa = sm;          // [D][K] layer i-1
    float *qb = sm + D * K;  // [D][K] layer i
    for (int e = t; e < D * K; e += EDGE_THREADS) {
        const int j = e / K, k = e - j * K;
        const int64_t w = (int64_t)j * A.W + (int64_t)k * A.n + i;
        qb[e] = A.q[w];
        qa[e] = i > 0 ? A.q[w - 1] : 0.f;
    }
    __syncthreads();
    if (blockIdx.y == 0) {
        for (int k = t; k < K; k += EDGE_THREADS) {
            bool near = false;
#pragma unroll
            for (int j = 0; j < D; ++j) {
                const float m = ((A.prismatic_mask >> j) & 1u) ? A.margin_pris : A.margin_rev;
                const float v = qb[j * K + k];
                near = near || (__fsub_rn(v, A.lo[j]) < m) || (__fsub_rn(A.hi[j], v) < m);
            }
            float p = near ? A.pen_limit : 0.f;
            if (A.use_clear && A.clear[(int64_t)k * A.n + i] < 0.f) p = __fadd_rn(p, A.pen_collision);
            A.pen[(int64_t)i * K + k] = p;
        }
    }
    if (i == 0) return;
    float *out = A.edges + (size_t)(i - 1) * K * KP;
    const int rows = (K + gridDim.y - 1) / gridDim.y, k0 = blockIdx.y * rows, k1 = min(K, k0 + rows);
    for (int kp = t; kp < KP; kp += EDGE_THREADS) {
        if (kp >= K) { // the padding of every row: never chosen
            for (int k = k0; k < k1; ++k) out[(size_t)k * KP + kp] = __int_as_float(0x7f800000);
            continue;
        }
        float qp[D];
#pragma unroll
        for (int j = 0; j < D; ++j) qp[j] = qa[j * K + kp];
        for (int k = k0; k < k1; ++k) {
            float s = 0.f;
#pragma unroll
            for (int j = 0; j < D; ++j) s = fmaxf(s, fabsf(__fsub_rn(qb[j * K + k], qp[j])));
            out[(size_t)k * KP + kp] = s;
        }
    }
}

__device__ __forceinline__ void take_min(float &best, int &arg, float v, int a) { // first minimum: smaller value, then smaller index
    if (v < best || (v == best && a < arg)) { best = v; arg = a; }
}

__device__ __forceinline__ uint32_t map_cluster(uint32_t saddr, uint32_t rank) { // shared::cta address -> shared::cluster address in CTA `rank`
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
// One 4-byte store into another CTA's shared memory that also counts 4 bytes on that CTA's mbarrier.
__device__ __forceinline__ void st_async_f32(uint32_t raddr, float v, uint32_t rbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];" ::"r"(raddr), "r"(__float_as_uint(v)), "r"(rbar)
                 : "memory");
}

// The sequential part, on one thread-block cluster of DP_CLUSTER CTAs.  CTA r owns the nodes [r * KC, (r + 1) * KC)
// of every layer, G lanes per node.  Every CTA keeps the whole cost vector c[i-1] in its own shared memory; the
// owner of a node sends its new cost to all CTAs with st.async, each store counting 4 bytes on the receiver's
// mbarrier of that layer's parity, and a CTA starts layer i+1 when all 4 K bytes of layer i have arrived: no
// cluster-wide barrier (and no memory fence that would wait for the prefetch) inside the loop.  Two buffers and two
// mbarriers are enough: nobody can send layer i+1 before it has received every node of layer i, i.e. before every
// owner has finished reading layer i-1.  That argument paces OWNERS only, so only CTAs and warps that own a node
// take part in the layer loop: a CTA without nodes (K <= 7; K = 9 gives KC = 2 and ranks 5-7 empty) is sent nothing
// and a warp without nodes (the tail of the last active rank) never waits -- nobody would wait for either, and one
// that fell two layers behind would see layer i+2 counted on the mbarrier phase of layer i.  Both go straight to
// the cluster barrier after the loop.  The edge costs do not depend on the DP, so the first NB per lane of the
// NEXT layer are loaded before the wait and their L2 latency hides behind it.  Predecessors stay in the owner's
// shared memory and are gathered into CTA 0 after the last layer (or go to global memory when n * K of them do not
// fit); CTA 0 picks the end node, walks back and gathers xi_search.
template <int G, int NB>
__global__ void __launch_bounds__(DP_THREADS) search_dp_kernel(const SArgs A) {
    extern __shared__ float sm[];
    __shared__ float s_red[DP_THREADS / 32];
    __shared__ __align__(8) uint64_t bars[2];
    cg::cluster_group cl = cg::this_cluster();
    const int rank = (int)cl.block_rank();
    const int K = A.K, KP = A.KP, n = A.n, KC = A.KC, t = threadIdx.x, nthr = blockDim.x;
    float *c0 = sm, *c1 = sm + KP;                                                    // c[i] lives in c0 for even i
    uint16_t *pred_mine = reinterpret_cast<uint16_t *>(sm + 2 * KP);                  // [n][KC] this CTA's nodes
    uint16_t *pred_all = pred_mine + (size_t)n * KC;                                  // [n][K], filled in CTA 0 at the end
    const int kl = t / G, g = t % G;
    const int k = rank * KC + kl;
    const bool node = kl < KC && k < K;
    const bool owner = node && g == 0;
    const int nact = (K + KC - 1) / KC;                         // ranks 0 .. nact-1 own nodes (rank 0 always does)
    const int kw = rank * KC + (t & ~31) / G;                   // first node of this warp: the warp takes part in the
    const bool in_loop = rank < nact && (t & ~31) / G < KC && kw < K; // layer loop iff it owns at least one node
    const float INF = __int_as_float(0x7f800000);
    if (t == 0) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int x = t; x < KP; x += nthr) {
        c0[x] = x < K ? A.pen[x] : 0.f; // the padding is only ever combined with an edge cost of +inf
        c1[x] = 0.f;
    }
    // this lane's slice of the incoming edges of its node: columns g, g + G, ...; lanes without a node read row 0
    const float *__restrict__ rp = A.edges + (size_t)(node ? k : 0) * KP + g;
    const size_t layer = (size_t)K * KP;
    const int nbatch = KP / (G * NB);
    float e[NB], pn = 0.f;
    auto load_batch = [&](int b) {
#pragma unroll
        for (int u = 0; u < NB; ++u) e[u] = __ldg(rp + (b * NB + u) * G);
    };
    uint32_t rdst[DP_CLUSTER], rbar[DP_CLUSTER]; // where this node's cost and its byte count go, in every CTA (parity 0)
#pragma unroll
    for (int r = 0; r < DP_CLUSTER; ++r) {
        rdst[r] = map_cluster(smem_u32(c0 + (node ? k : 0)), r);
        rbar[r] = map_cluster(smem_u32(&bars[0]), r);
    }
    if (n > 1) {
        load_batch(0);
        if (owner) pn = __ldg(A.pen + (size_t)K + k);
    }
    cl.sync(); // mbarriers initialised everywhere, c[0] in place
    for (int i = 1; in_loop && i < n; ++i) { // in_loop is warp-uniform; thread 0 (node 0 of its rank) is always in
        const int par = i & 1;
        if (t == 0) mbar_expect_tx(&bars[par], 4u * (uint32_t)K); // layer i: one 4-byte store per node, from its owner
        const float *cprev = (par ? c0 : c1) + g;
        float best = INF;
        int arg = 0x7fffffff;
        for (int b = 0; b < nbatch; ++b) {
#pragma unroll
            for (int u = 0; u < NB; ++u) {
                const int off = (b * NB + u) * G;
                const float v = fmaxf(cprev[off], e[u]);
                if (v < best) { best = v; arg = off + g; } // the index increases: the first minimum of this lane's subsequence stays
            }
            if (b + 1 < nbatch) load_batch(b + 1);
        }
#pragma unroll
        for (int s = 1; s < G; s <<= 1) {
            const float ob = __shfl_xor_sync(0xffffffffu, best, s);
            const int oa = __shfl_xor_sync(0xffffffffu, arg, s);
            take_min(best, arg, ob, oa);
        }
        if (owner) {
            if (arg == 0x7fffffff) arg = 0; // every incoming cost was +inf
            const float cnew = __fadd_rn(best, pn);
            const uint32_t shift = par ? 4u * (uint32_t)KP : 0u, bshift = par ? 8u : 0u;
#pragma unroll
            for (int r = 0; r < DP_CLUSTER; ++r)
                if (r < nact) st_async_f32(rdst[r] + shift, cnew, rbar[r] + bshift);
            if (A.pred_in_smem) pred_mine[(size_t)i * KC + kl] = (uint16_t)arg;
            else A.pred[(size_t)i * K + k] = (uint16_t)arg;
        }
        if (i + 1 < n) {
            rp += layer;
            load_batch(0);
            if (owner) pn = __ldg(A.pen + (size_t)(i + 1) * K + k);
        }
        mbar_wait(&bars[par], (uint32_t)(((i - 1) >> 1) & 1)); // bars[par] is used every other layer
    }
    cl.sync(); // every CTA is past its last wait: predecessor slices complete, global predecessors visible
    if (A.pred_in_smem) {
        uint16_t *dst = cl.map_shared_rank(pred_all, 0);
        for (int x = t; x < n * KC; x += nthr) {
            const int i = x / KC, l = x - i * KC, kk = rank * KC + l;
            if (i > 0 && kk < K) dst[(size_t)i * K + kk] = pred_mine[x];
        }
        cl.sync();
    }
    if (rank != 0) return;
    const float *cend = ((n - 1) & 1) ? c1 : c0;
    const uint16_t *pred = A.pred_in_smem ? pred_all : A.pred;
    // cheapest end node (warp 0), then the path back (one thread: n dependent reads)
    if (t < 32) {
        float best = INF;
        int arg = 0x7fffffff;
        for (int x = t; x < K; x += 32) {
            const float v = cend[x];
            if (v < best) { best = v; arg = x; }
        }
        for (int s = 1; s < 32; s <<= 1) {
            const float ob = __shfl_xor_sync(0xffffffffu, best, s);
            const int oa = __shfl_xor_sync(0xffffffffu, arg, s);
            take_min(best, arg, ob, oa);
        }
        if (t == 0) {
            if (arg == 0x7fffffff) arg = 0;
            A.result[0] = cend[arg];
            int cur = arg;
            A.choice[n - 1] = cur;
            for (int i = n - 1; i > 0; --i) {
                cur = pred[(size_t)i * K + cur];
                A.choice[i - 1] = cur;
            }
        }
    }
    __syncthreads(); // block-wide: also orders thread 0's global writes of choice[] before the reads below
    // xi_search and its mjac
    float mj = 0.f;
    for (int i = t; i < n; i += nthr) {
        const int ka = A.choice[i];
        const int kb = i + 1 < n ? A.choice[i + 1] : 0;
        for (int j = 0; j < A.dof; ++j) {
            const float a = A.q[(int64_t)j * A.W + (int64_t)ka * n + i];
            A.xi[(int64_t)j * n + i] = a;
            if (i + 1 < n) mj = fmaxf(mj, fabsf(__fsub_rn(A.q[(int64_t)j * A.W + (int64_t)kb * n + i + 1], a)));
        }
    }
    for (int s = 16; s > 0; s >>= 1) mj = fmaxf(mj, __shfl_xor_sync(0xffffffffu, mj, s));
    if ((t & 31) == 0) s_red[t >> 5] = mj;
    __syncthreads();
    if (t == 0) {
        for (int x = 1; x < nthr / 32; ++x) mj = fmaxf(mj, s_red[x]);
        A.result[1] = mj;
    }
}

} // namespace

extern "C" {

size_t lm_search_workspace_bytes(int32_t dof, int64_t K, int64_t n) {
    if (dof < 1 || dof > LM_MAX_DOF || K <= 0 || K > LM_SEARCH_MAX_K || n <= 0) return 0;
    return make_slayout(dof, K, n).all;
}

int lm_search_default_params(lm_search_params *out) {
    if (!out) return LM_EINVAL;
    out->margin_rev = (float)(1.5 * 3.14159265358979323846 / 180.0);
    out->margin_pris = 0.03f;
    out->pen_limit = 10.f;
    out->pen_collision = 100.f;
    out->use_clearance = 0;
    return LM_OK;
}

int lm_search(lm_ctx *c, const lm_search_params *p, void *workspace, size_t bytes, int32_t *choice_out,
              float *xi_out, float *result_out) {
    if (!c || !p || !workspace) return LM_EINVAL;
    if ((reinterpret_cast<uintptr_t>(workspace) & 255u) != 0) return LM_EINVAL;
    if (c->B > LM_SEARCH_MAX_K || c->n > 0x7fffffff) return LM_EINVAL;
    if (!(p->margin_rev >= 0.f) || !(p->margin_pris >= 0.f) || !(p->pen_limit >= 0.f) || !(p->pen_collision >= 0.f)) return LM_EINVAL;
    const bool use_clear = p->use_clearance != 0;
    if (use_clear && !(c->traj.attached && (c->traj.args.caps.npairs + c->traj.args.caps.nenv) > 0)) return LM_EINVAL;
    const int K = (int)c->B, d = c->dof;
    const SLayout L = make_slayout(d, c->B, c->n);
    if (bytes < L.all) return LM_ENOMEM;
    int rc = materialize_state(c);
    if (rc != LM_OK) return rc;
    char *ws = static_cast<char *>(workspace);
    SArgs a{};
    a.dof = d; a.n = (int32_t)c->n; a.K = K; a.W = c->W;
    const DpShape shp = dp_shape(K);
    a.KC = shp.KC;
    a.KP = shp.KP;
    a.prismatic_mask = c->args.ch.prismatic_mask;
    a.margin_rev = p->margin_rev; a.margin_pris = p->margin_pris; a.pen_limit = p->pen_limit; a.pen_collision = p->pen_collision;
    std::memcpy(a.lo, c->args.ch.lo, sizeof(a.lo));
    std::memcpy(a.hi, c->args.ch.hi, sizeof(a.hi));
    a.use_clear = use_clear ? 1 : 0;
    a.q = c->args.q;
    a.clear = reinterpret_cast<float *>(ws + L.clear);
    a.edges = reinterpret_cast<float *>(ws + L.edges);
    a.pen = reinterpret_cast<float *>(ws + L.pen);
    a.pred = reinterpret_cast<uint16_t *>(ws + L.pred);
    a.choice = reinterpret_cast<int32_t *>(ws + L.choice);
    a.xi = reinterpret_cast<float *>(ws + L.xi);
    a.result = reinterpret_cast<float *>(ws + L.result);
    if (use_clear) {
        rc = launch_clearance(c, reinterpret_cast<float *>(ws + L.clear));
        if (rc != LM_OK) return rc;
    }
    const size_t edge_smem = 2 * sizeof(float) * (size_t)d * K;
    size_t dp_smem = 2 * sizeof(float) * (size_t)a.KP;
    const size_t pred_bytes = 2 * (size_t)c->n * ((size_t)a.KC + (size_t)K); // the owner's slice + CTA 0's gathered copy
    a.pred_in_smem = (dp_smem + pred_bytes + 2048 <= SMEM_OPT_IN) ? 1 : 0;
    if (a.pred_in_smem) dp_smem += pred_bytes;
    launch_counter().fetch_add(2);
    {
        int split = (int)((4 * 148 + c->n - 1) / c->n); // about four blocks per SM, more when the trajectory is short
        if (split > K) split = K;
        if (split < 1) split = 1;
        const dim3 grid((unsigned)c->n, (unsigned)split);
#define LM_EDGE_LAUNCH(DD)                                                                                                  \
    case DD:                                                                                                                \
        LM_CUDA(cudaFuncSetAttribute(search_edges_kernel<DD>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536));         \
        search_edges_kernel<DD><<<grid, EDGE_THREADS, edge_smem, c->stream>>>(a);                                           \
        break;
        switch (d) {
            LM_EDGE_LAUNCH(1) LM_EDGE_LAUNCH(2) LM_EDGE_LAUNCH(3) LM_EDGE_LAUNCH(4)
            LM_EDGE_LAUNCH(5) LM_EDGE_LAUNCH(6) LM_EDGE_LAUNCH(7) LM_EDGE_LAUNCH(8)
            default: return LM_EINVAL;
        }
#undef LM_EDGE_LAUNCH
        LM_CUDA(cudaGetLastError());
    }
    {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(DP_CLUSTER);
        cfg.blockDim = dim3((unsigned)shp.threads);
        cfg.dynamicSmemBytes = dp_smem;
        cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = DP_CLUSTER;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        const int smem_max = (int)(SMEM_OPT_IN - 2048);
#define LM_DP_LAUNCH(GG)                                                                                                      \
    case GG:                                                                                                                  \
        LM_CUDA(cudaFuncSetAttribute(search_dp_kernel<GG, DP_BATCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max)); \
        LM_CUDA(cudaLaunchKernelEx(&cfg, search_dp_kernel<GG, DP_BATCH>, a));                                                 \
        break;
        switch (shp.G) {
            LM_DP_LAUNCH(1) LM_DP_LAUNCH(2) LM_DP_LAUNCH(4) LM_DP_LAUNCH(8) LM_DP_LAUNCH(16) LM_DP_LAUNCH(32)
            default: return LM_EINVAL;
        }
#undef LM_DP_LAUNCH
    }
    if (choice_out) LM_CUDA(cudaMemcpyAsync(choice_out, a.choice, 4 * (size_t)c->n, cudaMemcpyDefault, c->stream));
    if (xi_out) LM_CUDA(cudaMemcpyAsync(xi_out, a.xi, 4 * (size_t)c->n * d, cudaMemcpyDefault, c->stream));
    if (result_out) LM_CUDA(cudaMemcpyAsync(result_out, a.result, 8, cudaMemcpyDefault, c->stream));
    LM_CUDA(cudaStreamSynchronize(c->stream));
    return LM_OK;
}

} // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// lm_search_static: the same two kernels, for callers that cannot obtain device memory at all (include/lm.h has the
// user-facing description).  Every intermediate array of the search -- edge costs, penalties, predecessors, the chosen
// path -- lives in ONE fixed array that is part of the library image, so the call path below contains no cudaMalloc,
// no cudaFree, no host allocation and no library routine that allocates.
//
// g_search_static is a device variable.  In HOST code its name is only a handle for the runtime (a host-side shadow),
// not an address the GPU can use: the device address is looked up with cudaGetSymbolAddress, once per device and with
// that device current, and it is that looked-up pointer the kernels receive.
namespace {

static __device__ __align__(256) unsigned char g_search_static[LM_SEARCH_STATIC_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
char *g_static_ptr[STATIC_MAX_DEVICES];   // device address of g_search_static on device i, nullptr = not looked up yet
std::mutex g_static_mutex;

// Device address of the static scratch on the CURRENT device; the first call on a device performs the look-up.
int static_scratch(char **out) {
    int dev = -1;
    LM_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return LM_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        LM_CUDA(cudaGetSymbolAddress(&p, g_search_static));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u) != 0) return LM_EINVAL;
        g_static_ptr[dev] = static_cast<char *>(p);
    }
    *out = g_static_ptr[dev];
    return LM_OK;
}

float limit_inward(double x, bool lower) { // the fp32 limit lm_init derives from an fp64 one: never outside it
    float f = (float)x;
    if (lower && (double)f < x) f = nextafterf(f, INFINITY);
    if (!lower && (double)f > x) f = nextafterf(f, -INFINITY);
    return f;
}

} // namespace

extern "C" {

int lm_search_static_fits(int32_t dof, int64_t K, int64_t n) {
    if (dof < 1 || dof > LM_MAX_DOF || K <= 0 || K > LM_SEARCH_MAX_K || n <= 0 || n > 0x7fffffff) return 0;
    // K * KP * 4 bytes per layer >= 4 bytes: n beyond the capacity cannot fit, and the product below cannot overflow
    if ((uint64_t)n > (uint64_t)LM_SEARCH_STATIC_BYTES) return 0;
    return make_slayout(dof, K, n).all <= (size_t)LM_SEARCH_STATIC_BYTES ? 1 : 0;
}

int lm_search_static(const lm_chain *chain, int64_t K, int64_t n, const float *q, const lm_search_params *p,
                     void *cuda_stream, int32_t *choice_out, float *xi_out, float *result_out) {
    if (!chain || !q || !p) return LM_EINVAL;
    const int d = chain->dof;
    if (d < 1 || d > LM_MAX_DOF || !chain->joint_type || !chain->q_lo || !chain->q_hi) return LM_EINVAL;
    if (K <= 0 || K > LM_SEARCH_MAX_K || n <= 0 || n > 0x7fffffff) return LM_EINVAL;
    if (!(p->margin_rev >= 0.f) || !(p->margin_pris >= 0.f) || !(p->pen_limit >= 0.f) || !(p->pen_collision >= 0.f)) return LM_EINVAL;
    if (p->use_clearance) return LM_EINVAL; // the clearance needs a capsule model, i.e. a context
    if (!lm_search_static_fits(d, K, n)) return LM_ECAPACITY;
    char *ws = nullptr;
    int rc = static_scratch(&ws);
    if (rc != LM_OK) return rc;
    { // q must be memory of the device whose copy of the scratch the kernels are about to use
        int dev = -1;
        LM_CUDA(cudaGetDevice(&dev));
        cudaPointerAttributes at{};
        if (cudaPointerGetAttributes(&at, q) != cudaSuccess) { (void)cudaGetLastError(); return LM_EINVAL; }
        if (!(at.type == cudaMemoryTypeManaged || (at.type == cudaMemoryTypeDevice && at.device == dev))) return LM_EINVAL;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const SLayout L = make_slayout(d, K, n);
    SArgs a{};
    a.dof = d; a.n = (int32_t)n; a.K = (int32_t)K; a.W = K * n;
    const DpShape shp = dp_shape(K);
    a.KC = shp.KC;
    a.KP = shp.KP;
    for (int j = 0; j < d; ++j) {
        if (!(chain->q_lo[j] <= chain->q_hi[j]) || chain->joint_type[j] > 1) return LM_EINVAL;
        a.lo[j] = limit_inward(chain->q_lo[j], true);
        a.hi[j] = limit_inward(chain->q_hi[j], false);
        if (a.lo[j] > a.hi[j]) a.lo[j] = a.hi[j] = (float)chain->q_lo[j];
        if (chain->joint_type[j]) a.prismatic_mask |= 1u << j;
    }
    a.margin_rev = p->margin_rev; a.margin_pris = p->margin_pris; a.pen_limit = p->pen_limit; a.pen_collision = p->pen_collision;
    a.use_clear = 0;
    a.q = q;
    // Nothing below needs the scratch to start at zero: each of these regions is written in full by this call's own
    // kernels (edge rows including their +inf padding, all n * K penalties, the predecessors of layers 1 .. n-1, the
    // path, xi, the two results) before anything reads it, so what an earlier call left behind is never seen.
    a.clear = reinterpret_cast<float *>(ws + L.clear);
    a.edges = reinterpret_cast<float *>(ws + L.edges);
    a.pen = reinterpret_cast<float *>(ws + L.pen);
    a.pred = reinterpret_cast<uint16_t *>(ws + L.pred);
    a.choice = reinterpret_cast<int32_t *>(ws + L.choice);
    a.xi = reinterpret_cast<float *>(ws + L.xi);
    a.result = reinterpret_cast<float *>(ws + L.result);
    const size_t edge_smem = 2 * sizeof(float) * (size_t)d * (size_t)K;
    size_t dp_smem = 2 * sizeof(float) * (size_t)a.KP;
    const size_t pred_bytes = 2 * (size_t)n * ((size_t)a.KC + (size_t)K);
    a.pred_in_smem = (dp_smem + pred_bytes + 2048 <= SMEM_OPT_IN) ? 1 : 0;
    if (a.pred_in_smem) dp_smem += pred_bytes;
    launch_counter().fetch_add(2);
    {
        int split = (int)((4 * 148 + n - 1) / n);
        if (split > (int)K) split = (int)K;
        if (split < 1) split = 1;
        const dim3 grid((unsigned)n, (unsigned)split);
#define LM_EDGE_LAUNCH(DD)                                                                                                  \
    case DD:                                                                                                                \
        LM_CUDA(cudaFuncSetAttribute(search_edges_kernel<DD>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536));         \
        search_edges_kernel<DD><<<grid, EDGE_THREADS, edge_smem, stream>>>(a);                                              \
        break;
        switch (d) {
            LM_EDGE_LAUNCH(1) LM_EDGE_LAUNCH(2) LM_EDGE_LAUNCH(3) LM_EDGE_LAUNCH(4)
            LM_EDGE_LAUNCH(5) LM_EDGE_LAUNCH(6) LM_EDGE_LAUNCH(7) LM_EDGE_LAUNCH(8)
            default: return LM_EINVAL;
        }
#undef LM_EDGE_LAUNCH
        LM_CUDA(cudaGetLastError());
    }
    {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(DP_CLUSTER);
        cfg.blockDim = dim3((unsigned)shp.threads);
        cfg.dynamicSmemBytes = dp_smem;
        cfg.stream = stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = DP_CLUSTER;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        const int smem_max = (int)(SMEM_OPT_IN - 2048);
#define LM_DP_LAUNCH(GG)                                                                                                      \
    case GG:                                                                                                                  \
        LM_CUDA(cudaFuncSetAttribute(search_dp_kernel<GG, DP_BATCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max)); \
        LM_CUDA(cudaLaunchKernelEx(&cfg, search_dp_kernel<GG, DP_BATCH>, a));                                                 \
        break;
        switch (shp.G) {
            LM_DP_LAUNCH(1) LM_DP_LAUNCH(2) LM_DP_LAUNCH(4) LM_DP_LAUNCH(8) LM_DP_LAUNCH(16) LM_DP_LAUNCH(32)
            default: return LM_EINVAL;
        }
#undef LM_DP_LAUNCH
    }
    if (choice_out) LM_CUDA(cudaMemcpyAsync(choice_out, a.choice, 4 * (size_t)n, cudaMemcpyDefault, stream));
    if (xi_out) LM_CUDA(cudaMemcpyAsync(xi_out, a.xi, 4 * (size_t)n * d, cudaMemcpyDefault, stream));
    if (result_out) LM_CUDA(cudaMemcpyAsync(result_out, a.result, 8, cudaMemcpyDefault, stream));
    LM_CUDA(cudaStreamSynchronize(stream));
    return LM_OK;
}

} // extern "C"
