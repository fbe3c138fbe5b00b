// ppm_chain.cuh -- device-resident sampler loop around the likelihood ("a fully
// GPU-resident parallel-tempered MCMC ... batching likelihood calls within each device"; reading R26 of DESIGN.md):
// W walkers at inverse temperatures beta_w; per step a Gaussian random-walk proposal inside a box prior, Metropolis
// acceptance against beta_w (ln L' - ln L), replica exchange between neighbouring walkers.  The parameter batch, the
// likelihoods and the counters never leave HBM; one step (propose -> S0..S7 -> accept -> exchange) is captured once
// into a CUDA graph and replayed.  Random numbers: Philox4x32-10 keyed by the seed, counter (step, walker, stream).
// Product path (sm_100a); the CPU oracle has its own copy of the same published generator.
#pragma once
#include "ppm_common.cuh"

namespace ppm {

__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1,
                                              unsigned out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// 53-bit uniform in (0, 1) from two words
__device__ __forceinline__ double chain_u01(unsigned a, unsigned b)
{
    const unsigned long long m = ((unsigned long long)(a >> 5) << 26) | (unsigned long long)(b >> 6);
    return ((double)m + 0.5) * (1.0 / 9007199254740992.0);
}

// the two uniforms of counter (t, walker, stream); n0, n1: their Box-Muller normals
__device__ inline void chain_random(unsigned long long seed, unsigned long long t, unsigned walker, unsigned stream,
                                    double& u0, double& u1, double& n0, double& n1)
{
    unsigned x[4];
    philox4x32_10((unsigned)t, (unsigned)(t >> 32), walker, stream, (unsigned)seed, (unsigned)(seed >> 32), x);
    u0 = chain_u01(x[0], x[1]);
    u1 = chain_u01(x[2], x[3]);
    const double r = sqrt(-2.0 * log(u0));
    double s, c;
    sincos(2.0 * kPi * u1, &s, &c);
    n0 = r * c; n1 = r * s;
}

constexpr unsigned kStreamAccept = 0x10000u, kStreamSwap = 0x10001u;

struct ChainArgs {
    double* cur;            // [W][P] current states
    double* prop;           // [W][P] proposals (a walker whose proposal leaves the box gets its current state: evaluated, ignored)
    double* ll;             // [W] ln L of the current states
    double* llp;            // [W] ln L of the proposals
    int* oob;               // [W] 1 = proposal outside the box prior
    const double *lo, *hi, *sigma, *beta;
    long long* accepted;    // [W]
    long long* swapped;     // [W]
    unsigned long long* t;  // step counter
    unsigned long long seed;
    int W, P;
};

__global__ void k_chain_propose(ChainArgs A)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= A.W) return;
    const unsigned long long t = *A.t;
    const double* cur = A.cur + (size_t)w * A.P;
    double* prop = A.prop + (size_t)w * A.P;
    bool inside = true;
    for (int k = 0; k < A.P; k += 2) {
        const double s0 = A.sigma[k], s1 = (k + 1 < A.P) ? A.sigma[k + 1] : 0.0;
        double v0 = cur[k], v1 = (k + 1 < A.P) ? cur[k + 1] : 0.0;
        if (s0 > 0.0 || s1 > 0.0) {
            double u0, u1, n0, n1;
            chain_random(A.seed, t, (unsigned)w, (unsigned)(k / 2), u0, u1, n0, n1);
            if (s0 > 0.0) { v0 += s0 * n0; if (!(v0 >= A.lo[k] && v0 <= A.hi[k])) inside = false; }
            if (s1 > 0.0) { v1 += s1 * n1; if (!(v1 >= A.lo[k + 1] && v1 <= A.hi[k + 1])) inside = false; }
        }
        prop[k] = v0;
        if (k + 1 < A.P) prop[k + 1] = v1;
    }
    A.oob[w] = inside ? 0 : 1;
    if (!inside)
        for (int k = 0; k < A.P; ++k) prop[k] = cur[k];
}

__global__ void k_chain_accept(ChainArgs A)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= A.W) return;
    if (A.oob[w]) return;                                           // zero prior
    double u0, u1, n0, n1;
    chain_random(A.seed, *A.t, (unsigned)w, kStreamAccept, u0, u1, n0, n1);
    const double lp = A.llp[w];
    if (isfinite(lp) && log(u0) < A.beta[w] * (lp - A.ll[w])) {
        double* cur = A.cur + (size_t)w * A.P;
        const double* prop = A.prop + (size_t)w * A.P;
        for (int k = 0; k < A.P; ++k) cur[k] = prop[k];
        A.ll[w] = lp;
        A.accepted[w] += 1;
    }
}

// replica exchange between (i, i+1), i = t mod 2, t mod 2 + 2, ...; then the step counter advances.  One block.
__global__ void k_chain_swap(ChainArgs A)
{
    const unsigned long long t = *A.t;
    for (int i = (int)(t & 1ull) + 2 * (int)threadIdx.x; i + 1 < A.W; i += 2 * (int)blockDim.x) {
        double u0, u1, n0, n1;
        chain_random(A.seed, t, (unsigned)i, kStreamSwap, u0, u1, n0, n1);
        const double la = A.ll[i], lb = A.ll[i + 1];
        if (log(u0) < (A.beta[i] - A.beta[i + 1]) * (lb - la)) {
            double* a = A.cur + (size_t)i * A.P;
            double* b = a + A.P;
            for (int k = 0; k < A.P; ++k) { const double x = a[k]; a[k] = b[k]; b[k] = x; }
            A.ll[i] = lb; A.ll[i + 1] = la;
            A.swapped[i] += 1; A.swapped[i + 1] += 1;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) *A.t = t + 1ull;
}

}  // namespace ppm
