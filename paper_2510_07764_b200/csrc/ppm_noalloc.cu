// ppm_noalloc.cu -- ppm_loglike_noalloc: S7 (Poisson ln L, reading R14) for callers that cannot call cudaMalloc (code
// under CUDA-graph capture, tight serving loops, harnesses that forbid allocation).  A variant of the two-stage ln L
// reduction of ppm_loglike (ppm_observe.cuh: k_loglike_part / k_loglike_final, same arithmetic, same summation order, so
// the same bits) whose scratch -- the per-slice partial sums -- lives in a file-scope static __device__ array instead of a
// context's cudaMalloc'ed buffer.  Product path (sm_100a).  No context, no allocation, no free: the entry point only
// looks up the array's device address (once per device), checks its arguments and launches two kernels on the caller's
// stream.
//
// The array (kMaxVec + 1 rows of kSplit doubles + as many ints: 0.75 MiB) is held by every GPU that loads the library
// until the process exits.  Every call on a device shares it and it keeps the last call's contents; nothing in it has to
// start at zero, because stage 1 overwrites every entry stage 2 reads (rows 0 .. B of kSplit entries each).  Calls that
// overlap on one GPU (different streams, or different host threads) RACE on it: serialise them.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <mutex>

#include "ppm.h"

namespace {

constexpr int kSplit = 64;                          // slices of the (phase, channel) plane per vector (= kLLSplit)
constexpr int kMaxVec = PPM_NOALLOC_MAX_BATCH;      // largest B of one call
constexpr int kMaxDev = 64;

struct Scratch {
    double part[(size_t)(kMaxVec + 1) * kSplit];    // row b < B: slice sums of vector b; row B: sum lgamma(d + 1)
    int bad[(size_t)(kMaxVec + 1) * kSplit];        // slice saw m <= 0 < d or NaN
};

static __device__ __align__(256) Scratch g_scratch;

thread_local char t_err[256] = "";
std::mutex g_mu;
Scratch* g_ptr[kMaxDev] = {};                       // device address of g_scratch per device ordinal (host-side name != address)

int fail(int code, const char* what)
{
    snprintf(t_err, sizeof(t_err), "ppm_loglike_noalloc: %s", what);
    return code;
}

__global__ void __launch_bounds__(256) k_ll_part_static(const double* __restrict__ counts, const double* __restrict__ data,
                                                        const double* __restrict__ bkg, int n_phase, int n_channel,
                                                        double exposure, int nvec, Scratch* __restrict__ sc)
{
    __shared__ double red[256];
    __shared__ int bad_s;
    const int b = blockIdx.y;
    const bool lgam = (b == nvec);
    const size_t n = (size_t)n_phase * n_channel;
    const size_t per = (n + kSplit - 1) / kSplit;
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
        sc->part[(size_t)b * kSplit + blockIdx.x] = red[0];
        sc->bad[(size_t)b * kSplit + blockIdx.x] = bad_s;
    }
}

__global__ void k_ll_final_static(const Scratch* __restrict__ sc, int nvec, double* __restrict__ out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nvec) return;
    double lg = 0.0, s = 0.0;
    int isbad = 0;
    for (int i = 0; i < kSplit; ++i) {
        lg += sc->part[(size_t)nvec * kSplit + i];
        s += sc->part[(size_t)b * kSplit + i];
        isbad |= sc->bad[(size_t)b * kSplit + i];
    }
    out[b] = isbad ? -INFINITY : s - lg;
}

}  // namespace

extern "C" const char* ppm_loglike_noalloc_error(void) { return t_err; }

extern "C" int ppm_loglike_noalloc(const double* counts_dev, int B, int n_phase, int n_channel, const double* data_dev,
                                   const double* bkg_dev, double exposure_s, double* loglike_dev, void* stream)
{
    if (B < 0) return fail(PPM_ERR_ARG, "B must be >= 0");
    if (B == 0) return PPM_OK;
    if (B > kMaxVec) {
        snprintf(t_err, sizeof(t_err), "ppm_loglike_noalloc: B = %d exceeds PPM_NOALLOC_MAX_BATCH = %d (the static scratch "
                 "array holds that many vectors; split the batch or use ppm_loglike)", B, kMaxVec);
        return PPM_ERR_BATCH;
    }
    if (!counts_dev || !data_dev || !loglike_dev) return fail(PPM_ERR_ARG, "null pointer");
    if (n_phase < 1 || n_channel < 1) return fail(PPM_ERR_ARG, "n_phase and n_channel must be >= 1");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) return fail(PPM_ERR_CUDA, "no current CUDA device");
    if (dev >= kMaxDev) return fail(PPM_ERR_ARG, "device ordinal beyond 63");
    Scratch* sc;
    {   // once per device, with that device current: the device address of the static array
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_ptr[dev]) {
            void* p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&p, g_scratch);
            if (e != cudaSuccess || !p) {
                snprintf(t_err, sizeof(t_err), "ppm_loglike_noalloc: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
                return PPM_ERR_CUDA;
            }
            g_ptr[dev] = static_cast<Scratch*>(p);
        }
        sc = g_ptr[dev];
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    dim3 grid(kSplit, B + 1);
    k_ll_part_static<<<grid, 256, 0, st>>>(counts_dev, data_dev, bkg_dev, n_phase, n_channel, exposure_s, B, sc);
    k_ll_final_static<<<(B + 127) / 128, 128, 0, st>>>(sc, B, loglike_dev);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(t_err, sizeof(t_err), "ppm_loglike_noalloc: launch failed: %s", cudaGetErrorString(e));
        return PPM_ERR_CUDA;
    }
    return PPM_OK;
}
