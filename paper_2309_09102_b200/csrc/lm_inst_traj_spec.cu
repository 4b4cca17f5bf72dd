// trajectory-level kernels specialised for the registered chain structures (lm_specs.cuh)
#include "lm_traj_launch.h"
namespace lmk {
cudaError_t launch_traj_pose_spec(int which, int spec_id, bool weighted, unsigned grid, unsigned block, cudaStream_t s, const TArgs &a) {
    switch (spec_id) {
    case SPEC_PANDA: return launch_traj_pose_t<7, PandaSpec>(which, weighted, grid, block, s, a);
    case SPEC_RAND8: return launch_traj_pose_t<8, Rand8Spec>(which, weighted, grid, block, s, a);
    default: return cudaErrorInvalidValue;
    }
}
} // namespace lmk
