// generic trajectory-level kernels, dof 1..4, and the dof-only kernels (pack / unpack / block-tridiagonal solve)
#include "lm_traj_launch.h"
namespace lmk {
cudaError_t launch_traj_pose_generic_lo(int which, int dof, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    switch (dof) {
    case 1: return launch_traj_pose_t<1, GenericSpec<1>>(which, weighted, grid, block, s, a);
    case 2: return launch_traj_pose_t<2, GenericSpec<2>>(which, weighted, grid, block, s, a);
    case 3: return launch_traj_pose_t<3, GenericSpec<3>>(which, weighted, grid, block, s, a);
    case 4: return launch_traj_pose_t<4, GenericSpec<4>>(which, weighted, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
cudaError_t launch_traj_plain(int which, int dof, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    switch (dof) {
    case 1: return launch_traj_plain_t<1>(which, grid, block, s, a);
    case 2: return launch_traj_plain_t<2>(which, grid, block, s, a);
    case 3: return launch_traj_plain_t<3>(which, grid, block, s, a);
    case 4: return launch_traj_plain_t<4>(which, grid, block, s, a);
    case 5: return launch_traj_plain_t<5>(which, grid, block, s, a);
    case 6: return launch_traj_plain_t<6>(which, grid, block, s, a);
    case 7: return launch_traj_plain_t<7>(which, grid, block, s, a);
    case 8: return launch_traj_plain_t<8>(which, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
} // namespace lmk
