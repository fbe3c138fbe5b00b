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

// ---- K8: Poisson ln L (reading R14).  Two deterministic stages: kLLSplit blocks per vector reduce fixed slices of
// the (phase, channel) plane with a fixed-shape tree; k_loglike_final adds the slice sums in index order.  Row
// `nvec` of the partial array holds sum lgamma(d+1), which depends on the data only (blockIdx.y == nvec).
constexpr int kLLSplit = 64;

__global__ void __launch_bounds__(256) k_loglike_part(const double* __restrict__ counts, const double* __restrict__ data,
                                                      const double* __restrict__ bkg, int n_phase, int n_channel,
                                                      double exposure, int nvec, double* __restrict__ part,
                                                      int* __restrict__ bad)
{
    __shared__ double red[256];
    __shared__ int bad_s;
    const int b = blockIdx.y;
    const bool lgam = (b == nvec);
    const size_t n = (size_t)n_phase * n_channel;
    const size_t per = (n + kLLSplit - 1) / kLLSplit;
    const size_t i0 = (size_t)blockIdx.x * per, i1 = (i0 + per < n) ? i0 + per : n;
    const double* C = counts + (size_t)(lgam ? 0 : b) * n;
    const double scale = exposure / n_phase;
    if (threadIdx.x == 0) bad_s = 0;
    __syncthreads();
    double s = 0.0;
    int isbad = 0;
    for (size_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
        const double d = data[i];
        if (lgam) { s += lgamma(d + 1.0); continue; }
        const double m = scale * C[i] + (bkg ? bkg[i % n_channel] : 0.0);
        if (!(m == m)) isbad = 1;
        if (d > 0.0) {
            if (!(m > 0.0)) isbad = 1; else s += d * log(m);
        }
        s -= m;
    }
    red[threadIdx.x] = s;
    if (isbad) bad_s = 1;
    __syncthreads();
    for (int h = 128; h > 0; h >>= 1) {
        if (threadIdx.x < h) red[threadIdx.x] += red[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        part[(size_t)b * kLLSplit + blockIdx.x] = red[0];
        bad[(size_t)b * kLLSplit + blockIdx.x] = bad_s;
    }
}

__global__ void k_loglike_final(const double* __restrict__ part, const int* __restrict__ bad, int nvec,
                                double* __restrict__ out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nvec) return;
    double lg = 0.0, s = 0.0;
    int isbad = 0;
    for (int i = 0; i < kLLSplit; ++i) {
        lg += part[(size_t)nvec * kLLSplit + i];
        s += part[(size_t)b * kLLSplit + i];
        isbad |= bad[(size_t)b * kLLSplit + i];
    }
    out[b] = isbad ? -INFINITY : s - lg;
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
