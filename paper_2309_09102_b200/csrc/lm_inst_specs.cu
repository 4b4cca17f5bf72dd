// LM and FK kernels specialised at compile time for the registered chain structures (lm_specs.cuh)
#include "lm_launch.h"
namespace lmk {
cudaError_t launch_iterate_spec(int spec_id, bool fast, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a) {
    switch (spec_id) {
    case SPEC_PANDA: return launch_iterate_t<7, PandaSpec>(fast, weighted, grid, block, s, a);
    case SPEC_RAND8: return launch_iterate_t<8, Rand8Spec>(fast, weighted, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
cudaError_t launch_fk_spec(int spec_id, bool fast, unsigned grid, unsigned block, cudaStream_t s, const KFkArgs &a) {
    switch (spec_id) {
    case SPEC_PANDA: return launch_fk_t<7, PandaSpec>(fast, grid, block, s, a);
    case SPEC_RAND8: return launch_fk_t<8, Rand8Spec>(fast, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
} // namespace lmk
