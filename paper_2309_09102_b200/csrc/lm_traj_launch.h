// lm_traj_launch.h -- launch entry points of the trajectory-level kernels (lm_traj.cuh); one
// translation unit per group of instantiations so that the build compiles them in parallel.
#pragma once
#include "lm_specs.cuh"
#include "lm_traj.cuh"

namespace lmk {

enum TrajPoseKernel : int { TK_ASSEMBLE = 0, TK_RHO = 1, TK_TRIAL = 2, TK_CLEARANCE = 3 };
enum TrajPlainKernel : int { TK_PACK_Q = 0, TK_PACK_TARGETS = 1, TK_UNPACK = 2, TK_SOLVE_FACTOR = 3, TK_SOLVE_REFINE = 4 };

// kernels that evaluate FK (chain-structure specialised or generic), thread per waypoint
cudaError_t launch_traj_pose_spec(int which, int spec_id, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);
cudaError_t launch_traj_pose_generic_lo(int which, int dof, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);
cudaError_t launch_traj_pose_generic_hi(int which, int dof, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);
// kernels that depend on the dof only
cudaError_t launch_traj_plain(int which, int dof, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a);

template <int D, typename SpecT>
cudaError_t launch_traj_pose_t(int which, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    const bool coll = a.caps.npairs + a.caps.nenv > 0; // collision rows: their own instantiations (lm_coll.cuh)
#define LM_TL_LAUNCH(K)                                                                   \
    do {                                                                                  \
        if (weighted) { if (coll) K<D, false, true, SpecT, true><<<grid, block, 0, s>>>(a);   \
                        else K<D, false, true, SpecT, false><<<grid, block, 0, s>>>(a); }     \
        else { if (coll) K<D, false, false, SpecT, true><<<grid, block, 0, s>>>(a);           \
               else K<D, false, false, SpecT, false><<<grid, block, 0, s>>>(a); }             \
    } while (0)
    switch (which) {
    case TK_ASSEMBLE: LM_TL_LAUNCH(tl_assemble_kernel); break;
    case TK_RHO: LM_TL_LAUNCH(tl_rho_kernel); break;
    case TK_TRIAL: LM_TL_LAUNCH(tl_trial_kernel); break;
    case TK_CLEARANCE: tl_clearance_kernel<D, SpecT><<<grid, block, 0, s>>>(a); break;
    default: return cudaErrorInvalidValue;
    }
#undef LM_TL_LAUNCH
    return cudaGetLastError();
}

template <int D>
cudaError_t launch_traj_plain_t(int which, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    switch (which) {
    case TK_PACK_Q: tl_pack_kernel<D><<<grid, block, 0, s>>>(a, 0); break;
    case TK_PACK_TARGETS: tl_pack_kernel<D><<<grid, block, 0, s>>>(a, 1); break;
    case TK_UNPACK: tl_unpack_kernel<D><<<grid, block, 0, s>>>(a); break;
    case TK_SOLVE_FACTOR:  // two chain warps + two producer warps per tile of 32 trajectories; the rings need more than
    case TK_SOLVE_REFINE: { // the default 48 KB.  Ring depth: deep while every SM holds at most one block (lm_traj.cuh)
        int dev = 0, sms = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        const bool deep = grid <= (unsigned)sms;
#define LM_SOLVE_LAUNCH(MODE, WANT)                                                                                          \
    {                                                                                                                        \
        /* the attribute is per DEVICE: set it on every launch (cheap), never once per process */                           \
        e = cudaFuncSetAttribute(tl_solve_kernel<D, MODE, WANT>, cudaFuncAttributeMaxDynamicSharedMemorySize,                \
                                 (int)tl_solve_smem_bytes<D, MODE, WANT>());                                                 \
        if (e != cudaSuccess) return e;                                                                                      \
        tl_solve_kernel<D, MODE, WANT><<<grid, TL_SOLVE_THREADS, tl_solve_smem_bytes<D, MODE, WANT>(), s>>>(a);              \
    }
        if (which == TK_SOLVE_FACTOR) {
            if (deep) LM_SOLVE_LAUNCH(0, TL_STAGES_DEEP) else LM_SOLVE_LAUNCH(0, TL_STAGES_SHALLOW)
        } else {
            if (deep) LM_SOLVE_LAUNCH(1, TL_STAGES_DEEP) else LM_SOLVE_LAUNCH(1, TL_STAGES_SHALLOW)
        }
#undef LM_SOLVE_LAUNCH
        break;
    }
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

} // namespace lmk
