// launch_map.cu -- instantiations and launcher of k_cells_map (temperature maps, strategy d, FP64): the windowed 16-warp
// kernel (stepped coordinate on log-uniform grids with EPL >= 4) and the full-width 8-warp kernel.
#include "ppm_launch.h"
#include "ppm_cells_map.cuh"

namespace ppm {

template <int EPL, int NPL>
static cudaError_t map_one(const LaunchShape& L, const CellArgs& a, bool windowed)
{
    if (windowed) {
        if constexpr (EPL >= 4) {
            if (a.uniform_e) PPM_LAUNCH_KERNEL((k_cells_map<EPL, NPL, true, true>), a);
        }
        PPM_LAUNCH_KERNEL((k_cells_map<EPL, NPL, true, false>), a);
    }
    PPM_LAUNCH_KERNEL((k_cells_map<EPL, NPL, false, false>), a);
}

template <int EPL>
static cudaError_t map_npl(const LaunchShape& L, const CellArgs& a, bool windowed)
{
    switch (L.npl) {
    case 1:  return map_one<EPL, 1>(L, a, windowed);
    case 3:  return map_one<EPL, 3>(L, a, windowed);
    case 5:  return map_one<EPL, 5>(L, a, windowed);
    case 7:  return map_one<EPL, 7>(L, a, windowed);
    default: return map_one<EPL, 9>(L, a, windowed);
    }
}

cudaError_t launch_cells_map(const LaunchShape& L, const CellArgs& a, bool windowed) { PPM_SWITCH_EPL(map_npl, L, a, windowed) }

}  // namespace ppm
