// ppm_cells_map32.cuh -- S4 + S5 for a per-cell effective-temperature map (reading R24) with FP32
// interpolation and exponential (ppm_config.precision = 1, tolerance 1e-4 per bin; the paper's own production precision,
// PAPER.md:569, 690), strategy d (linear in log T).  Product path (sm_100a).
//
// k_cells_tab32's arithmetic (FP32 mu contraction, Lagrange -> monomial coefficients, Horner, MUFU.EX2, short FP32 sums
// scaled into FP64 accumulators by integer exponents; geometry, Eq 45-46, mu weights and the fixed-point logx coordinate
// in FP64) on k_cells_map's row walk: the block visits the row's log T intervals in ascending order (cell list sorted by
// interval, k_rows) with the slices of the interval's two log T nodes in shared memory.  In FP32 both slices fit at full
// width beside 16 warps (2 x 44.5 KB), so there is no windowing and no second launch; the upper node of one interval is
// the lower node of the next (ping-pong, one new slice per step).
// Reference exponents (see ppm_cells32.cuh): per (row, interval) instead of per row -- n_ref = round(log2(T_ref^3 max F))
// and yoff_e = round(log2(10) v) at mu = 1, z(phase 0), T_ref, with T_ref the middle of the interval's cell temperatures
// -- so that FP32 sees O(10) although the cells' temperatures differ.  An interval whose cells span more than 0.5 dex
// (cells far outside the table's log T axis fall into its first / last interval) would leave FP32's exponent range: its
// vector gets PPM_STATUS_MAP_WINDOW and a NaN flux.
#pragma once
#include "ppm_cells32.cuh"
#include "ppm_cells_map.cuh"

namespace ppm {

__device__ __forceinline__ float contract4f(const float* __restrict__ sp0, int nx, float v0, float v1, float v2, float v3, float acc)
{
    return fmaf(v3, sp0[3 * nx], fmaf(v2, sp0[2 * nx], fmaf(v1, sp0[nx], fmaf(v0, sp0[0], acc))));
}

template <int EPL, int NPL>
__global__ void __launch_bounds__(512, 1) k_cells_map32(CellArgs A, StarD* stars_rw)
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
    // shared layout: per warp { K4 [KW] float4 (k0..k3), R0 [32] double2 (q, pb), R1a [32] float4 ((1-t) mu weights),
    // R1b [32] float4 (t mu weights), RI [32] int } | T [4][n1] f64 | MUAX [nmu] f64 | TAX [nT] f64 |
    // S0 [nmu][nx] f32 | S1 [nmu][nx] f32 (slices * log2 10) + tail pad
    constexpr int KW = 32 * NPL;
    constexpr int WARP_DBL = 2 * KW + 64 + 64 + 64 + 16;
    double* wbase = sm + (size_t)w * WARP_DBL;
    float4* K4 = reinterpret_cast<float4*>(wbase);
    double2* R0 = reinterpret_cast<double2*>(wbase + 2 * KW);
    float4* R1a = reinterpret_cast<float4*>(wbase + 2 * KW + 64);
    float4* R1b = reinterpret_cast<float4*>(wbase + 2 * KW + 128);
    int* RI = reinterpret_cast<int*>(wbase + 2 * KW + 192);
    double* T = sm + (size_t)A.nw * WARP_DBL;
    double* MUAX = T + 4 * n1;
    double* TAX = MUAX + A.nmu;
    float* Sb0 = reinterpret_cast<float*>(TAX + A.nT + (A.nT & 1));
    float* Sb1 = Sb0 + plane;

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
    for (int i = threadIdx.x; i < A.nT; i += blockDim.x) TAX[i] = A.axT[i];

    const StarD& st = A.stars[b];
    const double phi_off = st.phi_off;
    const double phi_out = (double)k / A.n_phase;                               // reading R3
    const double log10kB = log10(kKB_keV_K);
    unsigned npairs = 0;

    for (int ri = 0; ri < A.rows_per_chunk; ++ri) {
        const int rl = chunk + ri * A.nchunk;
        if (rl >= A.RT) break;
        const int rid = b * A.RT + rl;
        const RowD& row = A.rows[rid];
        const int nact = row.n_active;
        if (nact == 0 || !row.visible) continue;
        const int it_first = __ffsll((long long)row.tmask) - 1, it_last = 63 - __clzll((long long)row.tmask);
        {   // cell temperatures of the first / last interval may lie outside the axis: FP32 needs their spread bounded
            const double lo_span = A.axT[imin_(it_first + 1, A.nT - 1)] - fmin(row.tmin, A.axT[it_first]);
            const double hi_span = fmax(row.tmax, A.axT[imin_(it_last + 1, A.nT - 1)]) - A.axT[it_last];
            if (lo_span > 0.5 || hi_span > 0.5) {
                if (threadIdx.x == 0) atomicOr(&stars_rw[b].status, 8);          // PPM_STATUS_MAP_WINDOW: k_reduce writes NaN
                continue;
            }
        }
        const SpotD& sp = A.spots[rid / A.n_theta];
        __syncthreads();
        double fmx = 0.0;
        {
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
        if (!(fmx > 0.0)) continue;                                              // (block-uniform)
        const double* F = T;
        const double* Z = T + n1;
        const double* PO = T + 2 * n1;
        const double* MU = T + 3 * n1;
        const int* cl = A.cells + (size_t)rid * A.n_phi;
        const double* tcell = A.tmap + (size_t)rid * A.n_phi;
        int go = 0;                                                              // the row's two log g nodes (strategy d)
        while (go < 2 && row.wg[go] == 0.0) ++go;
        const double wga = row.wg[go] * kLog2_10, wgb = row.wg[go + 1] * kLog2_10;
        const size_t gplane = (size_t)A.nmu * nx;
        int pos = 0;
        int node0 = -1, node1 = -1;                                              // log T node held by slice buffer 0 / 1
        for (unsigned long long tm = row.tmask; tm; tm &= tm - 1) {
            const int it = __ffsll((long long)tm) - 1;                           // log T interval [it, it+1]
            const int pl = (node1 == it) ? 1 : 0;
            __syncthreads();                                                     // readers of the previous interval are done
#pragma unroll
            for (int h = 0; h < 2; ++h) {                                        // h = 0: lower node -> buffer pl; 1: upper -> 1 - pl
                const int buf = h ? 1 - pl : pl, node = it + h;
                if ((buf ? node1 : node0) == node) continue;
                if (buf) node1 = node; else node0 = node;
                float* dst = buf ? Sb1 : Sb0;
                const double* src = A.values + ((size_t)node * A.ng + row.bg + go) * gplane;
                // kDepth passes' loads are issued before their blends (the staging is bound by L2 latency)
                constexpr int kDepth = 6;
                for (int i0 = threadIdx.x; i0 < plane; i0 += kDepth * blockDim.x) {
                    double va[kDepth], vb[kDepth];
#pragma unroll
                    for (int u = 0; u < kDepth; ++u) {
                        const int i = imin_(i0 + u * (int)blockDim.x, plane - 1);
                        va[u] = __ldg(src + i);
                        vb[u] = __ldg(src + gplane + i);
                    }
#pragma unroll
                    for (int u = 0; u < kDepth; ++u) {
                        const int i = i0 + u * (int)blockDim.x;
                        if (i < plane) dst[i] = (float)fma(wgb, vb[u], wga * va[u]);
                    }
                }
            }
            __syncthreads();
            if (!kvalid) continue;
            const float* Slo = pl ? Sb1 : Sb0;
            const float* Shi = pl ? Sb0 : Sb1;
            const double po0 = PO[0];
            // reference temperature of the interval: the middle of its cells' range
            const double t_lo = (it == it_first) ? fmin(row.tmin, TAX[it]) : TAX[it];
            const double t_hi = (it == it_last) ? fmax(row.tmax, TAX[imin_(it + 1, A.nT - 1)]) : TAX[it + 1];
            const double t_ref = 0.5 * (t_lo + t_hi);
            const int n_ref = __double2int_rn(3.0 * t_ref * kLog2_10 + log2(fmx));
            {
                const long long q0 = __double2ll_rn(((log10(Z[0]) - (log10kB + t_ref)) * A.inv_h - A.x0_over_h) * kTwo52);
#pragma unroll
                for (int i = 0; i < EPL; ++i) {
                    long long s = q0 + uef[i];
                    s = s < 0 ? 0 : (s > s_top ? s_top : s);
                    yoff[i] = rintf(Slo[(A.nmu - 1) * nx + (int)(s >> 52)]);
                }
            }
            for (bool more = true; more;) {
                // ---- step A (FP64): lane <-> cell of this interval ----
                const int idx = pos + lane;
                double Fp = 0.0, pb = 0.0, tw = 0.0;
                long long pq = 0;
                double ww[4] = {0.0, 0.0, 0.0, 0.0};
                int info = 0;
                const int entry = (idx < nact) ? cl[idx] : -1;
                const bool mine = (entry >= 0) && ((entry >> 16) == it);
                const int n_mine = __popc(__ballot_sync(0xffffffffu, mine));     // a prefix of the batch (sorted list)
                pos += n_mine;
                more = (n_mine == 32);
                if (mine) {
                    const int m = entry & 0xFFFF;
                    const double lT = tcell[m];
                    double tt;
                    axis_linear(TAX, A.nT, lT, tt);
                    const double phi_p = phase_of_cell(phi_out, cell_azimuth(A.mesh, row, sp, m), phi_off, po0);   // Eq 45
                    double zp, mup;
                    template_interp(F, Z, PO, MU, A.n_fp, A.phase_order, phi_p, Fp, zp, mup);                  // Eq 46
                    if (!(Fp > 0.0)) Fp = 0.0;
                    if (Fp != 0.0) {
                        int flags;
                        pair_table_record(Fp, zp, mup, log10kB + lT, 3.0 * lT * kLog2_10 - (double)n_ref, MUAX, A.nmu, A.mu_rule, nx,
                                          A.inv_h, A.x0_over_h, uef_first, uef_last, s_top, 0.0, 0.0, pq, pb, ww, info, flags);
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4) ww[q4] *= 1.0 / kLog2_10;     // the FP32 slices are already scaled by log2(10)
                        if (flags & (PAIR_CLAMP_LO | PAIR_CLAMP_HI)) info |= 0x8000;
                        tw = tt;
                    }
                }
                const unsigned valid = __ballot_sync(0xffffffffu, Fp != 0.0);
                const int cnt = __popc(valid);
                npairs += cnt;
                __syncwarp();
                if (Fp != 0.0) {
                    const int slot = __popc(valid & ((1u << lane) - 1u));
                    const double tl = 1.0 - tw;
                    R0[slot] = make_double2(__longlong_as_double(pq), pb);
                    R1a[slot] = make_float4((float)(tl * ww[0]), (float)(tl * ww[1]), (float)(tl * ww[2]), (float)(tl * ww[3]));
                    R1b[slot] = make_float4((float)(tw * ww[0]), (float)(tw * ww[1]), (float)(tw * ww[2]), (float)(tw * ww[3]));
                    RI[slot] = info;
                }
                __syncwarp();
                // ---- step B (FP32): walk the valid pairs ----
                for (int pj = 0; pj < cnt; ++pj) {
                    const double2 r0 = R0[pj];
                    const float4 wa = R1a[pj], wb = R1b[pj];
                    const int inf = RI[pj];
                    const long long q = __double_as_longlong(r0.x);
                    const float qb = (float)r0.y;
                    const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                    const int n0 = jlo - 1 + NPL * lane;
                    const float* pl0 = Slo + (inf & 0x7FFF) + n0;
                    const float* ph0 = Shi + (inf & 0x7FFF) + n0;
                    float f[NPL + 3];
#pragma unroll
                    for (int jn = 0; jn < NPL; ++jn)
                        f[1 + jn] = contract4f(ph0 + jn, nx, wb.x, wb.y, wb.z, wb.w, contract4f(pl0 + jn, nx, wa.x, wa.y, wa.z, wa.w, qb));
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
                    if (jlo == 0 || jhi == nx - 2) {      // strategy d: linear in the first / last interval of the axis
#pragma unroll
                        for (int jn = 0; jn < NPL; ++jn) {
                            const int c = n0 + jn;
                            if (c != 0 && c != nx - 2) continue;
                            kc[jn] = make_float4(0.5f * (f[jn + 1] + f[jn + 2]), f[jn + 2] - f[jn + 1], 0.0f, 0.0f);
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
                            s = s < 0 ? 0 : (s > s_top ? s_top : s);             // clamp to the table (reading R13b)
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
                    acc[i] += scale_pow2(acc32[i], n_ref + (int)yoff[i]);
                    acc32[i] = 0.0f;
                }
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
