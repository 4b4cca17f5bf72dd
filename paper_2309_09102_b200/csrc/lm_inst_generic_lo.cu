// generic (run-time chain structure) LM kernels, dof 1..4, and every generic FK kernel
#include "lm_launch.h"
namespace lmk {
cudaError_t launch_iterate_generic_lo(int dof, bool fast, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a) {
    switch (dof) {
    case 1: return launch_iterate_t<1, GenericSpec<1>>(fast, weighted, grid, block, s, a);
    case 2: return launch_iterate_t<2, GenericSpec<2>>(fast, weighted, grid, block, s, a);
    case 3: return launch_iterate_t<3, GenericSpec<3>>(fast, weighted, grid, block, s, a);
    case 4: return launch_iterate_t<4, GenericSpec<4>>(fast, weighted, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
cudaError_t launch_fk_generic(int dof, bool fast, unsigned grid, unsigned block, cudaStream_t s, const KFkArgs &a) {
    switch (dof) {
    case 1: return launch_fk_t<1, GenericSpec<1>>(fast, grid, block, s, a);
    case 2: return launch_fk_t<2, GenericSpec<2>>(fast, grid, block, s, a);
    case 3: return launch_fk_t<3, GenericSpec<3>>(fast, grid, block, s, a);
    case 4: return launch_fk_t<4, GenericSpec<4>>(fast, grid, block, s, a);
    case 5: return launch_fk_t<5, GenericSpec<5>>(fast, grid, block, s, a);
    case 6: return launch_fk_t<6, GenericSpec<6>>(fast, grid, block, s, a);
    case 7: return launch_fk_t<7, GenericSpec<7>>(fast, grid, block, s, a);
    case 8: return launch_fk_t<8, GenericSpec<8>>(fast, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
} // namespace lmk
