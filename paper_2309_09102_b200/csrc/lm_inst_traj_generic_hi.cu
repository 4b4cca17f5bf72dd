// generic trajectory-level kernels, dof 5..8
#include "lm_traj_launch.h"
namespace lmk {
cudaError_t launch_traj_pose_generic_hi(int which, int dof, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    switch (dof) {
    case 5: return launch_traj_pose_t<5, GenericSpec<5>>(which, weighted, grid, block, s, a);
    case 6: return launch_traj_pose_t<6, GenericSpec<6>>(which, weighted, grid, block, s, a);
    case 7: return launch_traj_pose_t<7, GenericSpec<7>>(which, weighted, grid, block, s, a);
    case 8: return launch_traj_pose_t<8, GenericSpec<8>>(which, weighted, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
} // namespace lmk
