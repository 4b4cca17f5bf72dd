// lm_traj_launch.h -- launch entry points of the trajectory-level kernels (lm_traj.cuh); one
// translation unit per group of instantiations so that the build compiles them in parallel.
#pragma once
#include "lm_specs.cuh"
#include "lm_traj.cuh"

namespace lmk {

enum TrajPoseKernel : int { TK_COST_INIT = 0, TK_COST = 1, TK_CLEARANCE = 2, TK_SOLVE_FACTOR = 3, TK_SOLVE_REFINE = 4, TK_ASSEMBLE = 5, TK_RHO = 6 };
enum TrajPlainKernel : int { TK_PACK_Q = 0, TK_PACK_TARGETS = 1, TK_UNPACK = 2, TK_SOLVE_FACTOR_HBM = 3, TK_SOLVE_REFINE_HBM = 4 };

// kernels that evaluate FK (chain-structure specialised or generic): the per-waypoint cost kernels and the solve kernels,
// whose producer warps assemble the normal equations (fused path), and the per-waypoint assemble / rho kernels of the
// unfused path.  `grid` is ignored for the solve kernels (one block per tile).
cudaError_t launch_traj_pose_spec(int which, int spec_id, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);
cudaError_t launch_traj_pose_generic_lo(int which, int dof, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);
cudaError_t launch_traj_pose_generic_hi(int which, int dof, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);
// kernels that depend on the dof only
cudaError_t launch_traj_plain(int which, int dof, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);

template <int D, int MODE, bool FUSED, bool WEIGHTED, typename SpecT>
cudaError_t launch_traj_solve_t(cudaStream_t s, const TArgs &a) {
    // the rings need more than the default 48 KB; the attribute is per DEVICE: set it on every launch (cheap)
    cudaError_t e = cudaFuncSetAttribute(tl_solve_kernel<D, MODE, FUSED, WEIGHTED, SpecT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)tl_solve_smem_bytes<D, MODE>());
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    // block shape (lm_traj.cuh): more producer warps while every SM holds at most one block
    const unsigned threads = !FUSED ? TL_SOLVE_THREADS_HBM : a.Bt <= (int64_t)sms ? TL_SOLVE_THREADS_FEW_TILES : TL_SOLVE_THREADS_MANY_TILES;
    tl_solve_kernel<D, MODE, FUSED, WEIGHTED, SpecT><<<(unsigned)a.Bt, threads, tl_solve_smem_bytes<D, MODE>(), s>>>(a);
    return cudaGetLastError();
}

template <int D, typename SpecT>
cudaError_t launch_traj_pose_t(int which, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    const bool coll = a.caps.npairs + a.caps.nenv > 0; // collision rows: their own instantiations (lm_coll.cuh)
#define LM_TL_DISPATCH(CALL)                                               \
    do {                                                                   \
        if (weighted) { if (coll) { CALL(true, true); } else { CALL(true, false); } }   \
        else { if (coll) { CALL(false, true); } else { CALL(false, false); } }          \
    } while (0)
    // with collision rows: the window kernel (lanes along the path); its transposition buffers need more than 48 KB
    const unsigned wgrid = (unsigned)(a.Bt * ((a.n + TL_CW - 1) / TL_CW));
#define LM_TL_COST_WINDOW(W, I)                                                                                                    \
    do {                                                                                                                           \
        cudaError_t e_ = cudaFuncSetAttribute(tl_cost_window_kernel<D, W, SpecT, I>, cudaFuncAttributeMaxDynamicSharedMemorySize,  \
                                              (int)tl_cost_window_smem<D>());                                                      \
        if (e_ != cudaSuccess) return e_;                                                                                          \
        tl_cost_window_kernel<D, W, SpecT, I><<<wgrid, TL_CW_THREADS, tl_cost_window_smem<D>(), s>>>(a);                           \
    } while (0)
#define LM_TL_COST_INIT(W, C) do { if (C && a.cost_by_waypoints) LM_TL_COST_WINDOW(W, true); else tl_cost_kernel<D, false, W, SpecT, C, true><<<grid, block, 0, s>>>(a); } while (0)
#define LM_TL_COST(W, C) do { if (C && a.cost_by_waypoints) LM_TL_COST_WINDOW(W, false); else tl_cost_kernel<D, false, W, SpecT, C, false><<<grid, block, 0, s>>>(a); } while (0)
#define LM_TL_ASSEMBLE(W, C) tl_assemble_kernel<D, false, W, SpecT, C><<<grid, block, 0, s>>>(a)
#define LM_TL_RHO(W, C) tl_rho_kernel<D, false, W, SpecT, C><<<grid, block, 0, s>>>(a)
    switch (which) {
    case TK_COST_INIT: LM_TL_DISPATCH(LM_TL_COST_INIT); break;
    case TK_COST: LM_TL_DISPATCH(LM_TL_COST); break;
    case TK_CLEARANCE: tl_clearance_kernel<D, SpecT><<<grid, block, 0, s>>>(a); break;
    case TK_ASSEMBLE: LM_TL_DISPATCH(LM_TL_ASSEMBLE); break;
    case TK_RHO: LM_TL_DISPATCH(LM_TL_RHO); break;
    case TK_SOLVE_FACTOR: // fused: the producers assemble; never with collision rows (lm_traj_api.cu)
        if (coll) return cudaErrorInvalidValue;
        return weighted ? launch_traj_solve_t<D, 0, true, true, SpecT>(s, a) : launch_traj_solve_t<D, 0, true, false, SpecT>(s, a);
    case TK_SOLVE_REFINE:
        if (coll) return cudaErrorInvalidValue;
        return weighted ? launch_traj_solve_t<D, 1, true, true, SpecT>(s, a) : launch_traj_solve_t<D, 1, true, false, SpecT>(s, a);
    default: return cudaErrorInvalidValue;
    }
#undef LM_TL_DISPATCH
#undef LM_TL_COST_INIT
#undef LM_TL_COST
#undef LM_TL_COST_WINDOW
#undef LM_TL_ASSEMBLE
#undef LM_TL_RHO
    return cudaGetLastError();
}

template <int D>
cudaError_t launch_traj_plain_t(int which, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    switch (which) {
    case TK_PACK_Q: tl_pack_kernel<D><<<grid, block, 0, s>>>(a, 0); break;
    case TK_PACK_TARGETS: tl_pack_kernel<D><<<grid, block, 0, s>>>(a, 1); break;
    case TK_UNPACK: tl_unpack_kernel<D><<<grid, block, 0, s>>>(a); break;
    case TK_SOLVE_FACTOR_HBM: return launch_traj_solve_t<D, 0, false, false, NoSpec>(s, a);
    case TK_SOLVE_REFINE_HBM: return launch_traj_solve_t<D, 1, false, false, NoSpec>(s, a);
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

} // namespace lmk
