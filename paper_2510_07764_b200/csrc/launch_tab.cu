// launch_tab.cu -- instantiations and launcher of k_cells_tab (FP64 table emission, the dominant kernel).
#include "ppm_launch.h"

namespace ppm {

// node exchange (k_cells_tab<.., NX = true>): measured on the same box against the record form -- 4 energies per lane
// (128-energy grids: C3 -2.3 %, the Table 3 geometries -6.5 %), 2 energies per lane +5 % (C2), so EPL = 4 only
static bool use_node_exchange(int epl, const CellArgs&) { return epl == 4; }

template <int EPL, int NPL>
static cudaError_t tab_uni(const LaunchShape& L, const CellArgs& a)
{
    if constexpr (EPL == 4) {
        if (use_node_exchange(EPL, a)) {
            if constexpr (EPL >= 2) {
                if (a.uniform_e) PPM_LAUNCH_KERNEL((k_cells_tab<EPL, NPL, true, true>), a);
            }
            PPM_LAUNCH_KERNEL((k_cells_tab<EPL, NPL, false, true>), a);
        }
    }
    if constexpr (EPL >= 2) {
        if (a.uniform_e) PPM_LAUNCH_KERNEL((k_cells_tab<EPL, NPL, true, false>), a);
    }
    PPM_LAUNCH_KERNEL((k_cells_tab<EPL, NPL, false, false>), a);
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
