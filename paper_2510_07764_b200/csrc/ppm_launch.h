// ppm_launch.h -- launchers of the cell-kernel families.  Each family's template instantiations (energies per lane
// EPL in {1, 2, 4, 5, 8, 10} x window nodes per lane NPL in {1, 3, 5, 7, 9}) live in their own translation unit
// (launch_*.cu) so that the library builds in parallel; ppm.cu sees only these declarations.  Every launcher sets the
// kernel's dynamic shared-memory limit, launches on `stream` and returns the CUDA status of that (launch errors surface
// at the caller's cudaGetLastError).  Product path (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include "ppm_cells.cuh"

namespace ppm {

struct LaunchShape {
    cudaStream_t stream;
    dim3 grid;
    int threads;
    size_t smem;
    int epl, npl;
};

cudaError_t launch_cells_tab(const LaunchShape& L, const CellArgs& a);      // k_cells_tab (a.uniform_e picks the stepped coordinate)
cudaError_t launch_cells_lin(const LaunchShape& L, const CellArgs& a);      // k_cells_lin   (interp_domain = 1)
cudaError_t launch_cells_tab32(const LaunchShape& L, const CellArgs& a);    // k_cells_tab32 (precision = 1)
cudaError_t launch_cells_bb(const LaunchShape& L, const CellArgs& a);       // k_cells_bb    (closed-form blackbody)
cudaError_t launch_cells_map(const LaunchShape& L, const CellArgs& a, bool windowed);      // k_cells_map
cudaError_t launch_cells_map4(const LaunchShape& L, const CellArgs& a, StarD* stars_rw);   // k_cells_map4 (NPL 1 or 3)
cudaError_t launch_cells_map32(const LaunchShape& L, const CellArgs& a, StarD* stars_rw);  // k_cells_map32

// the two switches every launcher is made of
#define PPM_LAUNCH_KERNEL(KERNEL, ...)                                                                                     \
    do {                                                                                                                   \
        cudaError_t e_ = cudaFuncSetAttribute(KERNEL, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem);           \
        if (e_ != cudaSuccess) return e_;                                                                                  \
        KERNEL<<<L.grid, L.threads, L.smem, L.stream>>>(__VA_ARGS__);                                                      \
        return cudaSuccess;                                                                                                \
    } while (0)

#define PPM_SWITCH_EPL(FN, ...)                                                                                            \
    switch (L.epl) {                                                                                                       \
    case 1:  return FN<1>(__VA_ARGS__);                                                                                    \
    case 2:  return FN<2>(__VA_ARGS__);                                                                                    \
    case 4:  return FN<4>(__VA_ARGS__);                                                                                    \
    case 5:  return FN<5>(__VA_ARGS__);                                                                                    \
    case 8:  return FN<8>(__VA_ARGS__);                                                                                    \
    default: return FN<10>(__VA_ARGS__);                                                                                   \
    }

}  // namespace ppm
