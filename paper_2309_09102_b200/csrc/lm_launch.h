// lm_launch.h -- launch entry points of the kernel instantiations (one translation unit each, so
// that the build can compile them in parallel).
#pragma once
#include "lm_kernels.cuh"
#include "lm_specs.cuh"

namespace lmk {
// generic kernels, dof 1..4 / 5..8
cudaError_t launch_iterate_generic_lo(int dof, bool fast, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a);
cudaError_t launch_iterate_generic_hi(int dof, bool fast, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a);
cudaError_t launch_fk_generic(int dof, bool fast, unsigned grid, unsigned block, cudaStream_t s, const KFkArgs &a);
// specialised kernels (spec_id != SPEC_GENERIC)
cudaError_t launch_iterate_spec(int spec_id, bool fast, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a);
cudaError_t launch_fk_spec(int spec_id, bool fast, unsigned grid, unsigned block, cudaStream_t s, const KFkArgs &a);

// lane-group form (G = 2, 4 lanes per waypoint) of the registered chains; plain residual, unweighted, exact sincos only
cudaError_t launch_iterate_lanegroup(int spec_id, int lanes, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a);

// ---- launch helpers used by the instantiation units
template <int D, typename SpecT>
cudaError_t launch_iterate_t(bool fast, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a) {
    if (a.variant == LM_VAR_DUAL || a.variant == LM_VAR_RPY) { // disclosed variants: their own instantiations, the hot path's kernels are untouched
#define LM_IT_LAUNCH(V)                                                                                \
    do {                                                                                               \
        if (fast) { if (weighted) lm_iterate_kernel<D, true, true, SpecT, V><<<grid, block, 0, s>>>(a);   \
                    else lm_iterate_kernel<D, true, false, SpecT, V><<<grid, block, 0, s>>>(a); }         \
        else { if (weighted) lm_iterate_kernel<D, false, true, SpecT, V><<<grid, block, 0, s>>>(a);       \
               else lm_iterate_kernel<D, false, false, SpecT, V><<<grid, block, 0, s>>>(a); }             \
    } while (0)
        if (a.variant == LM_VAR_DUAL) LM_IT_LAUNCH(LM_VAR_DUAL); else LM_IT_LAUNCH(LM_VAR_RPY);
#undef LM_IT_LAUNCH
    } else if (fast) {
        if (weighted) lm_iterate_kernel<D, true, true, SpecT><<<grid, block, 0, s>>>(a);
        else lm_iterate_kernel<D, true, false, SpecT><<<grid, block, 0, s>>>(a);
    } else if (!SpecT::spec.generic && a.refine == 1 && a.trace_q == nullptr) { // the HOT instantiations (lm_kernels.cuh)
        if (weighted) lm_iterate_kernel<D, false, true, SpecT, 0, 1, true><<<grid, block, 0, s>>>(a);
        else lm_iterate_kernel<D, false, false, SpecT, 0, 1, true><<<grid, block, 0, s>>>(a);
    } else {
        if (weighted) lm_iterate_kernel<D, false, true, SpecT><<<grid, block, 0, s>>>(a);
        else lm_iterate_kernel<D, false, false, SpecT><<<grid, block, 0, s>>>(a);
    }
    return cudaGetLastError();
}

template <int D, typename SpecT>
cudaError_t launch_fk_t(bool fast, unsigned grid, unsigned block, cudaStream_t s, const KFkArgs &a) {
    if (fast) lm_fk_kernel<D, true, SpecT><<<grid, block, 0, s>>>(a);
    else lm_fk_kernel<D, false, SpecT><<<grid, block, 0, s>>>(a);
    return cudaGetLastError();
}

} // namespace lmk
