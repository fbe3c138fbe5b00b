// launch_tab.cu -- instantiations and launcher of k_cells_tab (FP64 table emission, the dominant kernel).
#include "ppm_launch.h"

namespace ppm {

template <int EPL, int NPL>
static cudaError_t tab_uni(const LaunchShape& L, const CellArgs& a)
{
    if constexpr (EPL >= 2) {
        if (a.uniform_e) PPM_LAUNCH_KERNEL((k_cells_tab<EPL, NPL, true>), a);
    }
    PPM_LAUNCH_KERNEL((k_cells_tab<EPL, NPL, false>), a);
}

template <int EPL>
static cudaError_t tab_npl(const LaunchShape& L, const CellArgs& a)
{
    switch (L.npl) {
    case 1:  return tab_uni<EPL, 1>(L, a);
    case 3:  return tab_uni<EPL, 3>(L, a);
    case 5:  return tab_uni<EPL, 5>(L, a);
    case 7:  return tab_uni<EPL, 7>(L, a);
    default: return tab_uni<EPL, 9>(L, a);
    }
}

cudaError_t launch_cells_tab(const LaunchShape& L, const CellArgs& a) { PPM_SWITCH_EPL(tab_npl, L, a) }

}  // namespace ppm
