// launch_map_x.cu -- instantiations and launchers of k_cells_map4 (temperature maps under the cubic-in-log-T strategies)
// and k_cells_map32 (temperature maps with FP32 interpolation).
#include "ppm_launch.h"
#include "ppm_cells_map4.cuh"
#include "ppm_cells_map32.cuh"

namespace ppm {

template <int EPL>
static cudaError_t map4_npl(const LaunchShape& L, const CellArgs& a, StarD* stars_rw)
{
    if (L.npl == 1) PPM_LAUNCH_KERNEL((k_cells_map4<EPL, 1>), a, stars_rw);
    PPM_LAUNCH_KERNEL((k_cells_map4<EPL, 3>), a, stars_rw);
}

template <int EPL>
static cudaError_t map32_npl(const LaunchShape& L, const CellArgs& a, StarD* stars_rw)
{
    switch (L.npl) {
    case 1:  PPM_LAUNCH_KERNEL((k_cells_map32<EPL, 1>), a, stars_rw);
    case 3:  PPM_LAUNCH_KERNEL((k_cells_map32<EPL, 3>), a, stars_rw);
    case 5:  PPM_LAUNCH_KERNEL((k_cells_map32<EPL, 5>), a, stars_rw);
    case 7:  PPM_LAUNCH_KERNEL((k_cells_map32<EPL, 7>), a, stars_rw);
    default: PPM_LAUNCH_KERNEL((k_cells_map32<EPL, 9>), a, stars_rw);
    }
}

cudaError_t launch_cells_map4(const LaunchShape& L, const CellArgs& a, StarD* stars_rw) { PPM_SWITCH_EPL(map4_npl, L, a, stars_rw) }
cudaError_t launch_cells_map32(const LaunchShape& L, const CellArgs& a, StarD* stars_rw) { PPM_SWITCH_EPL(map32_npl, L, a, stars_rw) }

}  // namespace ppm
