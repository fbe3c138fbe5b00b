// ppm_cells32.cuh -- S4 + S5 with FP32 interpolation and exponential (ppm_config.precision = 1; SURVEY.md 8(a) row S4
// "FP32 variant", north_star tolerance 1e-4 per bin).  Geometry stays FP64: the templates, Eq 45-46, the mu stencil
// weights, the fixed-point logx coordinate and log2(F_p T^3) are computed exactly as in k_cells_tab; what runs in FP32
// is the work per (pair, interval) and per triple: mu contraction, Lagrange -> monomial coefficients, Horner, 2^y by
// MUFU.EX2 (ex2.approx.ftz.f32), and a short FP32 accumulation.  Product path (sm_100a).
//
// Range handling.  y = log2(F_p T^3 10^v) spans hundreds of octaves across energies (Wien tail), far more than FP32
// holds, so every term is formed relative to two integer exponents: n_row (per row: round(log2(T^3 max F))) and
// yoff_e (per row and energy: round(log2(10) v) at mu = 1 and the row's z at phase 0).  FP32 sees
// y - n_row - yoff_e = O(10).  Each lane sums at most 32 terms (one step-A batch) in FP32, then adds
// float_sum * 2^(n_row + yoff_e) to its FP64 accumulator (exact scaling by an exponent add): accumulation error
// <= 32 * 2^-24 per batch, the final sums are FP64.
#pragma once
#include "ppm_cells.cuh"

namespace ppm {

__device__ __forceinline__ float ex2_approx(float y)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y));
    return r;
}

// x * 2^k for a finite float sum x >= 0 and any int k, in double (exponent add; 0 stays 0; tiny results flush to 0)
__device__ __forceinline__ double scale_pow2(float x, int k)
{
    const double d = (double)x;
    const int hi = __double2hiint(d);
    const int e = ((hi >> 20) & 0x7FF) + k;
    if (x == 0.0f || e <= 0) return 0.0;
    return __hiloint2double(hi + (k << 20), __double2loint(d));
}

__device__ __forceinline__ float node_value32(const float* __restrict__ sp0, int nx, float v0, float v1, float v2, float v3,
                                              float qb)
{
    return fmaf(v3, sp0[3 * nx], fmaf(v2, sp0[2 * nx], fmaf(v1, sp0[nx], fmaf(v0, sp0[0], qb))));
}

__device__ __forceinline__ void cubic_coeffs32(float c0, float c1, float c2, float c3, float& k0, float& k1, float& k2,
                                               float& k3)
{
    const float s03 = c0 + c3, s12 = c1 + c2, d30 = c3 - c0, d21 = c2 - c1;
    k0 = fmaf(s03, -0.0625f, s12 * 0.5625f);
    k1 = fmaf(d30, -1.0f / 24.0f, d21 * 1.125f);
    k2 = (s03 - s12) * 0.25f;
    k3 = fmaf(d21, -0.5f, d30 * (1.0f / 6.0f));
}

template <int EPL, int NPL>
__global__ void __launch_bounds__(512, 1) k_cells_tab32(CellArgs A)
{
    extern __shared__ __align__(16) double sm[];
    __shared__ double fmax_s[16];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int chunk = blockIdx.x, pg = blockIdx.y;
    const int b = blockIdx.z / A.n_etile, et = blockIdx.z % A.n_etile;
    const int k = pg * A.nw + w;
    const bool kvalid = k < A.n_phase;
    const int e0 = et * 32 * EPL;
    const int n1 = A.n_fp + 1;
    const int nx = A.nx;
    const int plane = A.nmu * nx;
    // shared layout: per warp { K4 [KW] float4 (k0..k3), R0 [32] double2 (q, pb), R1 [32] float4 (mu weights * log2 10),
    // RI [32] int } | T [4][n1] f64 | MUAX [nmu] f64 | S32 [nmu][nx] f32 (slice * log2 10)
    constexpr int KW = 32 * NPL;
    constexpr int WARP_DBL = 2 * KW + 64 + 64 + 16;
    double* wbase = sm + (size_t)w * WARP_DBL;
    float4* K4 = reinterpret_cast<float4*>(wbase);
    double2* R0 = reinterpret_cast<double2*>(wbase + 2 * KW);
    float4* R1 = reinterpret_cast<float4*>(wbase + 2 * KW + 64);
    int* RI = reinterpret_cast<int*>(wbase + 2 * KW + 128);
    double* T = sm + (size_t)A.nw * WARP_DBL;
    double* MUAX = T + 4 * n1;
    float* S = reinterpret_cast<float*>(MUAX + A.nmu);

    long long uef[EPL];
    float yoff[EPL], acc32[EPL];
    double acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) {
        const int e = e0 + lane + 32 * i;
        uef[i] = A.uef[e < A.nE ? e : A.nE - 1];
        acc[i] = 0.0; acc32[i] = 0.0f; yoff[i] = 0.0f;
    }
    const long long uef_first = A.uef[imin_(e0, A.nE - 1)];
    const long long uef_last = A.uef[imin_(e0 + 32 * EPL, A.nE) - 1];
    const long long s_top = ((long long)(nx - 1) << 52) - 1;
    for (int i = threadIdx.x; i < A.nmu; i += blockDim.x) MUAX[i] = A.axmu[i];

    const StarD& st = A.stars[b];
    const double phi_off = st.phi_off;
    const double phi_out = (double)k / A.n_phase;                               // reading R3
    unsigned npairs = 0;

    for (int ri = 0; ri < A.rows_per_chunk; ++ri) {
        const int rl = chunk + ri * A.nchunk;
        if (rl >= A.RT) break;
        const int rid = b * A.RT + rl;
        const RowD& row = A.rows[rid];
        const int nact = row.n_active;
        if (nact == 0 || !row.visible) continue;
        const SpotD& sp = A.spots[rid / A.n_theta];
        __syncthreads();
        double fmx = 0.0;
        {   // stage the slice as log2(10) * v in FP32, the template in FP64; block maximum of F
            const double* src = A.slices + (size_t)rid * plane;
            for (int i = threadIdx.x; i < plane; i += blockDim.x) S[i] = (float)(src[i] * kLog2_10);
            const double* ts = A.tmpl + (size_t)rid * 4 * n1;
            for (int i = threadIdx.x; i < 4 * n1; i += blockDim.x) {
                const double v = ts[i];
                T[i] = v;
                if (i < n1) fmx = fmax(fmx, v);
            }
#pragma unroll
            for (int m = 16; m > 0; m >>= 1) fmx = fmax(fmx, __shfl_xor_sync(0xffffffffu, fmx, m));
            if (lane == 0) fmax_s[w] = fmx;
        }
        __syncthreads();
        fmx = fmax_s[0];
        for (int i = 1; i < (int)(blockDim.x >> 5); ++i) fmx = fmax(fmx, fmax_s[i]);
        if (!kvalid || !(fmx > 0.0)) continue;
        const double* F = T;
        const double* Z = T + n1;
        const double* PO = T + 2 * n1;
        const double* MU = T + 3 * n1;
        const int* cl = A.cells + (size_t)rid * A.n_phi;
        const double po0 = PO[0];
        // row exponents: n_row and, per owned energy, yoff = round(log2(10) v) at mu = 1, z = Z[0]
        const int n_row = __double2int_rn(sp.log2T3 + log2(fmx));
        {
            const long long q0 = __double2ll_rn(((log10(Z[0]) - sp.log10kT) * A.inv_h - A.x0_over_h) * kTwo52);
#pragma unroll
            for (int i = 0; i < EPL; ++i) {
                long long s = q0 + uef[i];
                s = s < 0 ? 0 : (s > s_top ? s_top : s);
                yoff[i] = rintf(S[(A.nmu - 1) * nx + (int)(s >> 52)]);
            }
        }
        for (int base = 0; base < nact; base += 32) {
            // ---- step A (FP64): lane <-> cell; Eq 45-46 and the per-pair record ----
            const int idx = base + lane;
            double Fp = 0.0, pb = 0.0;
            long long pq = 0;
            double ww[4] = {0.0, 0.0, 0.0, 0.0};
            int info = 0;
            if (idx < nact) {
                const double phi_p = phase_of_cell(phi_out, cell_azimuth(A.mesh, row, sp, cl[idx]), phi_off, po0);   // Eq 45
                double zp, mup;
                template_interp(F, Z, PO, MU, A.n_fp, A.phase_order, phi_p, Fp, zp, mup);                            // Eq 46
                if (!(Fp > 0.0)) Fp = 0.0;
                if (Fp != 0.0) {
                    int flags;
                    pair_table_record(Fp, zp, mup, sp.log10kT, sp.log2T3 - (double)n_row, MUAX, A.nmu, A.mu_rule, nx, A.inv_h,
                                      A.x0_over_h, uef_first, uef_last, s_top, 0.0, 0.0, pq, pb, ww, info, flags);
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) ww[q4] *= 1.0 / kLog2_10;         // the FP32 slice is already scaled by log2(10)
                    if (flags & (PAIR_CLAMP_LO | PAIR_CLAMP_HI)) info |= 0x8000;
                }
            }
            const unsigned valid = __ballot_sync(0xffffffffu, Fp != 0.0);
            const int cnt = __popc(valid);
            npairs += cnt;
            __syncwarp();
            if (Fp != 0.0) {
                const int slot = __popc(valid & ((1u << lane) - 1u));
                R0[slot] = make_double2(__longlong_as_double(pq), pb);
                R1[slot] = make_float4((float)ww[0], (float)ww[1], (float)ww[2], (float)ww[3]);
                RI[slot] = info;
            }
            __syncwarp();
            // ---- step B (FP32): walk the valid pairs ----
            for (int pj = 0; pj < cnt; ++pj) {
                const double2 r0 = R0[pj];
                const float4 wv = R1[pj];
                const int inf = RI[pj];
                const long long q = __double_as_longlong(r0.x);
                const float qb = (float)r0.y;
                const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                const float* srow = S + (inf & 0x7FFF);
                const int n0 = jlo - 1 + NPL * lane;
                const float* sp0 = srow + n0;
                float f[NPL + 3];
#pragma unroll
                for (int jn = 0; jn < NPL; ++jn) f[1 + jn] = node_value32(sp0 + jn, nx, wv.x, wv.y, wv.z, wv.w, qb);
                f[0] = __shfl_up_sync(0xffffffffu, f[NPL], 1);
                if (NPL == 1) {
                    f[2] = __shfl_down_sync(0xffffffffu, f[1], 1);
                    f[3] = __shfl_down_sync(0xffffffffu, f[1], 2);
                } else {
                    f[NPL + 1] = __shfl_down_sync(0xffffffffu, f[1], 1);
                    f[NPL + 2] = __shfl_down_sync(0xffffffffu, f[2], 1);
                }
                float4 kc[NPL];
#pragma unroll
                for (int jn = 0; jn < NPL; ++jn) cubic_coeffs32(f[jn], f[jn + 1], f[jn + 2], f[jn + 3], kc[jn].x, kc[jn].y, kc[jn].z, kc[jn].w);
                if (jlo == 0 || jhi == nx - 2) {      // first / last interval of the axis in the window (warp-uniform)
#pragma unroll
                    for (int jn = 0; jn < NPL; ++jn) {
                        const int c = n0 + jn;
                        if (c != 0 && c != nx - 2) continue;
                        if (A.x_linedge) {
                            kc[jn] = make_float4(0.5f * (f[jn + 1] + f[jn + 2]), f[jn + 2] - f[jn + 1], 0.0f, 0.0f);
                        } else {
                            const int s = (c == 0) ? 0 : nx - 4;
                            float g[4];
#pragma unroll
                            for (int m = 0; m < 4; ++m) g[m] = node_value32(srow + s + m, nx, wv.x, wv.y, wv.z, wv.w, qb);
                            float k0, k1, k2, k3;
                            cubic_coeffs32(g[0], g[1], g[2], g[3], k0, k1, k2, k3);
                            const float d = (float)(c - 1 - s);
                            kc[jn] = make_float4(fmaf(d, fmaf(d, fmaf(d, k3, k2), k1), k0),
                                                 fmaf(d, fmaf(3.0f * d, k3, 2.0f * k2), k1), fmaf(3.0f * d, k3, k2), k3);
                        }
                    }
                }
                __syncwarp();
#pragma unroll
                for (int jn = 0; jn < NPL; ++jn) K4[NPL * lane + jn] = kc[jn];
                __syncwarp();
                const float4* K4q = K4 + (1 - jlo);
                if (!(inf & 0x8000)) {
#pragma unroll
                    for (int i = 0; i < EPL; ++i) {
                        const long long s = q + uef[i];
                        const int shi = (int)(s >> 32);
                        const float4 c4 = K4q[shi >> 20];
                        // top 23 bits of the 52-bit fraction under the exponent of 1.0f: 1 + frac in FP32
                        const float tau = __int_as_float((__funnelshift_l((int)s, shi, 3) & 0x007FFFFF) | 0x3F800000) - 1.5f;
                        const float y = fmaf(fmaf(fmaf(c4.w, tau, c4.z), tau, c4.y), tau, c4.x) - yoff[i];
                        acc32[i] += ex2_approx(y);
                    }
                } else if (q + uef_first >= 0) {
                    // only the upper energies leave the table (the common clamped case): one-sided clamp
#pragma unroll
                    for (int i = 0; i < EPL; ++i) {
                        long long s = q + uef[i];
                        s = s > s_top ? s_top : s;                              // clamp to the table (reading R13b)
                        const int shi = (int)(s >> 32);
                        const float4 c4 = K4q[shi >> 20];
                        const float tau = __int_as_float((__funnelshift_l((int)s, shi, 3) & 0x007FFFFF) | 0x3F800000) - 1.5f;
                        const float y = fmaf(fmaf(fmaf(c4.w, tau, c4.z), tau, c4.y), tau, c4.x) - yoff[i];
                        acc32[i] += ex2_approx(y);
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < EPL; ++i) {
                        long long s = q + uef[i];
                        s = s < 0 ? 0 : (s > s_top ? s_top : s);                 // clamp to the table (reading R13b)
                        const int shi = (int)(s >> 32);
                        const float4 c4 = K4q[shi >> 20];
                        const float tau = __int_as_float((__funnelshift_l((int)s, shi, 3) & 0x007FFFFF) | 0x3F800000) - 1.5f;
                        const float y = fmaf(fmaf(fmaf(c4.w, tau, c4.z), tau, c4.y), tau, c4.x) - yoff[i];
                        acc32[i] += ex2_approx(y);
                    }
                }
            }
            // flush the batch's FP32 sums into the FP64 accumulators (exact power-of-two scaling)
#pragma unroll
            for (int i = 0; i < EPL; ++i) {
                acc[i] += scale_pow2(acc32[i], n_row + (int)yoff[i]);
                acc32[i] = 0.0f;
            }
        }
    }
    if (kvalid && et == 0 && lane == 0 && npairs) atomicAdd(A.pairs, (unsigned long long)npairs);
    if (kvalid) {
        double* out = A.partial + (((size_t)b * A.nchunk + chunk) * A.n_phase + k) * A.nE;
#pragma unroll
        for (int i = 0; i < EPL; ++i) {
            const int e = e0 + lane + 32 * i;
            if (e < A.nE) out[e] = acc[i] / A.en[e];                            // the 1/E_e of Eq 47
        }
    }
}

}  // namespace ppm
