// launch_aux.cu -- instantiations and launchers of k_cells_lin (intensity-domain interpolation), k_cells_tab32 (FP32
// interpolation) and k_cells_bb (closed-form blackbody).
#include "ppm_launch.h"
#include "ppm_cells32.cuh"
#include "ppm_cells_lin.cuh"

namespace ppm {

template <int EPL>
static cudaError_t lin_npl(const LaunchShape& L, const CellArgs& a)
{
    switch (L.npl) {
    case 1:  PPM_LAUNCH_KERNEL((k_cells_lin<EPL, 1>), a);
    case 3:  PPM_LAUNCH_KERNEL((k_cells_lin<EPL, 3>), a);
    case 5:  PPM_LAUNCH_KERNEL((k_cells_lin<EPL, 5>), a);
    case 7:  PPM_LAUNCH_KERNEL((k_cells_lin<EPL, 7>), a);
    default: PPM_LAUNCH_KERNEL((k_cells_lin<EPL, 9>), a);
    }
}

template <int EPL>
static cudaError_t tab32_npl(const LaunchShape& L, const CellArgs& a)
{
    switch (L.npl) {
    case 1:  PPM_LAUNCH_KERNEL((k_cells_tab32<EPL, 1>), a);
    case 3:  PPM_LAUNCH_KERNEL((k_cells_tab32<EPL, 3>), a);
    case 5:  PPM_LAUNCH_KERNEL((k_cells_tab32<EPL, 5>), a);
    case 7:  PPM_LAUNCH_KERNEL((k_cells_tab32<EPL, 7>), a);
    default: PPM_LAUNCH_KERNEL((k_cells_tab32<EPL, 9>), a);
    }
}

template <int EPL>
static cudaError_t bb_one(const LaunchShape& L, const CellArgs& a) { PPM_LAUNCH_KERNEL((k_cells_bb<EPL>), a); }

cudaError_t launch_cells_lin(const LaunchShape& L, const CellArgs& a) { PPM_SWITCH_EPL(lin_npl, L, a) }
cudaError_t launch_cells_tab32(const LaunchShape& L, const CellArgs& a) { PPM_SWITCH_EPL(tab32_npl, L, a) }
cudaError_t launch_cells_bb(const LaunchShape& L, const CellArgs& a) { PPM_SWITCH_EPL(bb_one, L, a) }

}  // namespace ppm
