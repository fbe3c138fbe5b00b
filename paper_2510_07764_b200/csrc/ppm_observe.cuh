// ppm_observe.cuh -- S6 + S7 of DESIGN.md: ISM attenuation x banded response fold (PAPER.md:267-276,
// 449-472; Eq 22-23, 51-55) and the Poisson log-likelihood (reading R14), plus the
// DFMA-chain microbenchmark that measures the FP64 roofline denominator.  Product path (sm_100a).
#pragma once
#include "ppm_common.cuh"

namespace ppm {

// ---- K7: gather form of the banded fold.  Channel c receives the energies e_lo[c] .. e_hi[c]-1 (a
// contiguous range, found once in ppm_set_response); summed in increasing e, no atomics.
// Block = (channel tile of 128, phase k, vector b); the attenuated flux row sits in shared memory.
struct FoldArgs {
    const double* flux; const double* params; const double* band; const double* tau;
    const int* first; const int* e_lo; const int* e_hi;
    double* counts;
    int P, n_phase, nE, n_channel, band_w;
};

__global__ void __launch_bounds__(128) k_fold(FoldArgs A)
{
    extern __shared__ __align__(16) double sm[];     // [nE] attenuated flux of (b, k)
    const int k = blockIdx.y, b = blockIdx.z;
    const double NH = A.params[(size_t)b * A.P + 5];
    const double* f = A.flux + ((size_t)b * A.n_phase + k) * A.nE;
    for (int e = threadIdx.x; e < A.nE; e += blockDim.x) sm[e] = f[e] * exp(-NH * A.tau[e]);   // Eq 22/51
    __syncthreads();
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= A.n_channel) return;
    double s = 0.0;
    const int lo = A.e_lo[c], hi = A.e_hi[c];
    for (int e = lo; e < hi; ++e) {
        const int wdx = c - A.first[e];
        if (wdx >= 0 && wdx < A.band_w) s += sm[e] * A.band[(size_t)e * A.band_w + wdx];
    }
    A.counts[((size_t)b * A.n_phase + k) * A.n_channel + c] = s;
}

// ---- K8: Poisson ln L.  One block per vector, fixed-shape tree reduction (deterministic).
// lgamma(d+1) depends on the data only and is summed by the same kernel run with mode = 1.
__global__ void __launch_bounds__(512) k_loglike(const double* __restrict__ counts, const double* __restrict__ data,
                                                 const double* __restrict__ bkg, int n_phase, int n_channel,
                                                 double exposure, const double* __restrict__ lgam_sum, int mode,
                                                 double* __restrict__ out)
{
    __shared__ double red[512];
    __shared__ int bad_s;
    const int b = blockIdx.x;
    const size_t n = (size_t)n_phase * n_channel;
    const double* C = counts + (size_t)b * n;
    if (threadIdx.x == 0) bad_s = 0;
    __syncthreads();
    double s = 0.0;
    int bad = 0;
    for (size_t i = threadIdx.x; i < n; i += blockDim.x) {
        const double d = data[i];
        if (mode == 1) { s += lgamma(d + 1.0); continue; }
        const int c = (int)(i % n_channel);
        const double m = exposure * C[i] / n_phase + (bkg ? bkg[c] : 0.0);
        if (!(m == m)) bad = 1;
        if (d > 0.0) {
            if (!(m > 0.0)) bad = 1; else s += d * log(m);
        }
        s -= m;
    }
    red[threadIdx.x] = s;
    if (bad) bad_s = 1;
    __syncthreads();
    for (int h = 256; h > 0; h >>= 1) {
        if (threadIdx.x < h) red[threadIdx.x] += red[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (mode == 1) out[0] = red[0];
        else out[b] = bad_s ? -INFINITY : red[0] - lgam_sum[0];
    }
}

// ---- FP64 peak: 8 independent DFMA chains per thread, all SMs.  flop = blocks*threads*8*iters*2.
__global__ void __launch_bounds__(256) k_dfma_peak(double* out, int iters, double seed)
{
    double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6, a7 = seed + 7;
    const double m = 0.999999, c = 1.0e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 123.456) out[0] = s;      // never true; keeps the chains alive
}

}  // namespace ppm
