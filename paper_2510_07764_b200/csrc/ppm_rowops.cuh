// ppm_rowops.cuh -- the two plain kernels around the cell kernels: k_slice collapses the 4-D atmosphere table to each
// row's (mu x logx) slice (S4, before the cell kernel), k_reduce sums the per-chunk partial tiles in a fixed order
// (S5, after it).  Included by ppm.cu only (the cell kernels' launchers live in their own translation units).
// Product path (sm_100a).
#pragma once
#include "ppm_common.cuh"

namespace ppm {

// ---- K4: collapse the 4-D table to the row's (mu x logx) slice: T is per spot, g per row -------
struct SliceArgs {
    const SpotD* spots; const RowD* rows; const double* values; double* slices;
    int n_theta, nT, ng, nmu, nx;
    int domain;              // 0: weighted sum of the tabulated log10(I/T^3) (reading R13a); 1: of I/T^3 = 10^table (R13g)
};

__global__ void __launch_bounds__(256) k_slice(SliceArgs A)
{
    const int rid = blockIdx.y;
    const RowD& r = A.rows[rid];
    if (r.n_active == 0 || !r.visible) return;
    const SpotD& sp = A.spots[rid / A.n_theta];
    const int plane = A.nmu * A.nx;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= plane) return;
    double v = 0.0;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const double wa = sp.wT[a];
        if (wa == 0.0) continue;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double wb = r.wg[b];
            if (wb == 0.0) continue;
            const double node = __ldg(A.values + ((size_t)(sp.bT + a) * A.ng + (r.bg + b)) * plane + i);
            v = fma(wa * wb, A.domain ? exp10(node) : node, v);
        }
    }
    A.slices[(size_t)rid * plane + i] = v;
}

// ---- K6: F_t[b][k][e] = sum over chunks, fixed order (deterministic); NaN for rejected vectors ----
__global__ void __launch_bounds__(256) k_reduce(const double* __restrict__ partial, const StarD* __restrict__ stars,
                                                int nchunk, int n_out, double* __restrict__ flux, int* status)
{
    const int b = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int stt = stars[b].status;
    if (i == 0 && status) status[b] = stt;
    if (i >= n_out) return;
    double s = 0.0;
    if (stt) s = nan("");
    else {
        const double* p = partial + (size_t)b * nchunk * n_out + i;
        for (int c = 0; c < nchunk; ++c) s += p[(size_t)c * n_out];
    }
    flux[(size_t)b * n_out + i] = s;
}

}  // namespace ppm
