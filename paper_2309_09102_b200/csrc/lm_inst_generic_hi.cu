// generic (run-time chain structure) LM kernels, dof 5..8
#include "lm_launch.h"
namespace lmk {
cudaError_t launch_iterate_generic_hi(int dof, bool fast, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a) {
    switch (dof) {
    case 5: return launch_iterate_t<5, GenericSpec<5>>(fast, weighted, grid, block, s, a);
    case 6: return launch_iterate_t<6, GenericSpec<6>>(fast, weighted, grid, block, s, a);
    case 7: return launch_iterate_t<7, GenericSpec<7>>(fast, weighted, grid, block, s, a);
    case 8: return launch_iterate_t<8, GenericSpec<8>>(fast, weighted, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
} // namespace lmk
