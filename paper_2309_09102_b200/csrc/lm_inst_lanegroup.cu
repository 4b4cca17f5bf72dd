// lane-group LM kernels (2 / 4 lanes per waypoint, lm_delta_lg) for the registered chain structures: the measured
// alternative to one thread per waypoint that BASELINE.json's north_star names
#include "lm_launch.h"
namespace lmk {
cudaError_t launch_iterate_lanegroup(int spec_id, int lanes, unsigned grid, unsigned block, cudaStream_t s, const KArgs &a) {
    if (spec_id == SPEC_PANDA && lanes == 2) lm_iterate_kernel<7, false, false, PandaSpec, 0, 2><<<grid, block, 0, s>>>(a);
    else if (spec_id == SPEC_PANDA && lanes == 4) lm_iterate_kernel<7, false, false, PandaSpec, 0, 4><<<grid, block, 0, s>>>(a);
    else if (spec_id == SPEC_RAND8 && lanes == 2) lm_iterate_kernel<8, false, false, Rand8Spec, 0, 2><<<grid, block, 0, s>>>(a);
    else if (spec_id == SPEC_RAND8 && lanes == 4) lm_iterate_kernel<8, false, false, Rand8Spec, 0, 4><<<grid, block, 0, s>>>(a);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}
} // namespace lmk
