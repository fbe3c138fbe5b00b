// ppm_cells_map.cuh -- S4 + S5 for a per-cell effective-temperature map T_eff(theta, phi) (the paper's
// "full surface temperature map"; reading R24).  Strategy d only (emission = 2: linear in log T and log g).
// Product path (sm_100a).
//
// With one temperature per spot the 4-D table collapses per row to ONE (mu x logx) slice (k_slice).  With a map every
// cell has its own log T, so a pair needs the slices of the two log T nodes that bracket its cell:
//   v = (1 - t) v[iT] + t v[iT+1],   f_node = log2(10) sum_mu w_mu [(1 - t) S_iT + t S_iT+1][mu][c] + log2(F_p T^3).
// k_rows records, per row, which log T intervals its active cells fall in (RowD::tmask).  The block walks those
// intervals in ascending order; for interval iT it stages the node slices iT and iT+1 -- blended over the row's two
// log g nodes on the fly from the L2-resident 4-D table -- into two shared-memory buffers (the upper node of one
// interval is the lower node of the next: ping-pong, one new slice per step), and processes the row's cells of that
// interval.  Two full-width FP64 slices take 178 KB (room for 8 warps only); the WIN variant cuts the slices to the
// logx columns the interval's pairs can reach (map_window) and keeps 16 warps.
// Everything per pair and per triple is k_cells_tab's scheme (fixed-point logx coordinate, fused shuffle pass to
// per-interval monomial coefficients, Horner + degree-8 exp2), with T, kT and T^3 taken per cell.
#pragma once
#include "ppm_cells.cuh"

namespace ppm {

__device__ __forceinline__ double contract4(const double* __restrict__ sp0, int nx, double v0, double v1, double v2, double v3)
{
    return fma(v3, sp0[3 * nx], fma(v2, sp0[2 * nx], fma(v1, sp0[nx], v0 * sp0[0])));
}

// logx node window [c_lo, c_hi] that bounds every pair of log T interval `it` of a row: u = (log10(z E / kT) - x0) / h
// over z in [zlo, zhi] (template), E in [E_first, E_last] (energy tile, as fixed-point uef) and log T in the part of the
// row's range [tmin, tmax] that lies in the interval (temperatures outside the axis fall in the first / last interval).
// One node of slack on each side beyond the stencil's reach (c - 1 .. c + 2).
__device__ inline void map_window(const RowD& row, const double* __restrict__ axT, int nT, int it, double inv_h,
                                  double x0_over_h, double ue_first, double ue_last, int nx, int& c_lo, int& c_hi)
{
    const int first = __ffsll((long long)row.tmask) - 1, last = 63 - __clzll((long long)row.tmask);
    const double t_lo = (it == first) ? fmin(row.tmin, axT[it]) : axT[it];
    const double t_hi = (it == last) ? fmax(row.tmax, axT[imin_(it + 1, nT - 1)]) : axT[it + 1];
    const double log10kB = log10(kKB_keV_K);
    const double u_lo = (log10(row.zlo) - (log10kB + t_hi)) * inv_h - x0_over_h + ue_first;
    const double u_hi = (log10(row.zhi) - (log10kB + t_lo)) * inv_h - x0_over_h + ue_last;
    c_lo = imin_(imax_((int)floor(fmax(u_lo, -4.0)) - 2, 0), nx - 1);
    c_hi = imin_(imax_((int)floor(fmin(u_hi, (double)nx + 4.0)) + 3, 0), nx - 1);
}

// does every interval of the row fit a window of `wst` columns?  (rows that do not are left to the full-width kernel)
__device__ inline bool map_row_fits(const RowD& row, const double* __restrict__ axT, int nT, double inv_h, double x0_over_h,
                                    double ue_first, double ue_last, int nx, int wst)
{
    for (unsigned long long tm = row.tmask; tm; tm &= tm - 1) {
        int c_lo, c_hi;
        map_window(row, axT, nT, __ffsll((long long)tm) - 1, inv_h, x0_over_h, ue_first, ue_last, nx, c_lo, c_hi);
        if (c_hi - c_lo + 1 > wst) return false;
    }
    return true;
}

// WIN = true: 16 warps, the two node slices hold only the window's columns (row stride A.wst); rows whose windows do not
// fit are skipped (the WIN = false launch takes them).  WIN = false: 8 warps, full-width slices (row stride nx).
template <int EPL, int NPL, bool WIN>
__global__ void __launch_bounds__(WIN ? 512 : 256, 1) k_cells_map(CellArgs A)
{
    extern __shared__ __align__(16) double sm[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int chunk = blockIdx.x, pg = blockIdx.y;
    const int b = blockIdx.z / A.n_etile, et = blockIdx.z % A.n_etile;
    const int k = pg * A.nw + w;
    const bool kvalid = k < A.n_phase;
    const int e0 = et * 32 * EPL;
    const int n1 = A.n_fp + 1;
    const int nx = A.nx;
    const int wst = WIN ? A.wst : nx;                                           // row stride of the slice buffers
    const int plane = A.nmu * wst;
    // shared layout (doubles): per warp { KA [KW], KB [KW], R0 (q, qb), R1 (v0, v1), R2 (v2, v3), R3 (1-t, t) [32] as
    // double2, RI [32] int } | S0 [nmu][nx] | S1 [nmu][nx] | T [4][n1] | MUAX [nmu] | TAX [nT]
    constexpr int KW = 32 * NPL;
    constexpr int WARP_DBL = 4 * KW + 4 * 64 + 16;
    double* wbase = sm + (size_t)w * WARP_DBL;
    double2* KA = reinterpret_cast<double2*>(wbase);
    double2* R0 = KA + 2 * KW;
    double2* R1 = R0 + 32;
    double2* R2 = R1 + 32;
    double2* R3 = R2 + 32;
    int* RI = reinterpret_cast<int*>(R3 + 32);
    double* Sb0 = sm + (size_t)A.nw * WARP_DBL;
    double* Sb1 = Sb0 + plane;
    double* T = Sb1 + plane;
    double* MUAX = T + 4 * n1;
    double* TAX = MUAX + A.nmu;

    long long uef[EPL];
    double acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) {
        const int e = e0 + lane + 32 * i;
        uef[i] = A.uef[e < A.nE ? e : A.nE - 1];
        acc[i] = 0.0;
    }
    const long long uef_first = A.uef[imin_(e0, A.nE - 1)];
    const long long uef_last = A.uef[imin_(e0 + 32 * EPL, A.nE) - 1];
    const long long s_top = ((long long)(nx - 1) << 52) - 1;
    const double ue_first = (double)uef_first / kTwo52, ue_last = (double)uef_last / kTwo52;
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
        if (A.map_split) {                                                       // each row belongs to exactly one launch
            const bool fits = map_row_fits(row, A.axT, A.nT, A.inv_h, A.x0_over_h, ue_first, ue_last, nx, A.wst);
            if (fits != WIN) continue;
        }
        const SpotD& sp = A.spots[rid / A.n_theta];
        __syncthreads();
        {
            const double* ts = A.tmpl + (size_t)rid * 4 * n1;
            for (int i = threadIdx.x; i < 4 * n1; i += blockDim.x) T[i] = ts[i];
        }
        const double* F = T;
        const double* Z = T + n1;
        const double* PO = T + 2 * n1;
        const double* MU = T + 3 * n1;
        const int* cl = A.cells + (size_t)rid * A.n_phi;
        const double* tcell = A.tmap + (size_t)rid * A.n_phi;
        int pos = 0;                                                             // next unprocessed entry of the sorted cell list
        int node0 = -1, node1 = -1;                                              // log T node held by slice buffer 0 / 1
        for (unsigned long long tm = row.tmask; tm; tm &= tm - 1) {
            const int it = __ffsll((long long)tm) - 1;                           // log T interval [it, it+1]
            int c_lo = 0, c_hi = nx - 1;
            if (WIN) map_window(row, A.axT, A.nT, it, A.inv_h, A.x0_over_h, ue_first, ue_last, nx, c_lo, c_hi);
            const int pl = (!WIN && node1 == it) ? 1 : 0;                        // windowed buffers are interval-specific: no reuse
            __syncthreads();                                                     // readers of the previous interval are done
#pragma unroll
            for (int h = 0; h < 2; ++h) {                                        // h = 0: lower node -> buffer pl; 1: upper -> 1 - pl
                const int buf = h ? 1 - pl : pl, node = it + h;
                if (!WIN && (buf ? node1 : node0) == node) continue;
                if (buf) node1 = node; else node0 = node;
                double* dst = buf ? Sb1 : Sb0;
                const double* src = A.values + ((size_t)node * A.ng + row.bg) * ((size_t)A.nmu * nx);
                const int wcols = WIN ? c_hi - c_lo + 1 : nx;
                for (int i = threadIdx.x; i < A.nmu * wcols; i += blockDim.x) {
                    const int mu_i = i / wcols, col = i - mu_i * wcols;
                    const size_t gi = (size_t)mu_i * nx + (WIN ? c_lo : 0) + col;
                    double v = 0.0;
#pragma unroll
                    for (int gq = 0; gq < 4; ++gq)
                        if (row.wg[gq] != 0.0) v = fma(row.wg[gq], __ldg(src + (size_t)gq * A.nmu * nx + gi), v);
                    dst[mu_i * wst + col] = v;
                }
            }
            __syncthreads();
            if (!kvalid) continue;
            const double* Slo = pl ? Sb1 : Sb0;
            const double* Shi = pl ? Sb0 : Sb1;
            const double po0 = PO[0];
            // the row's list is sorted by log T interval (k_rows): the cells of interval `it` start at `pos`
            for (bool more = true; more;) {
                // ---- step A: lane <-> cell of this interval ----
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
                        int flags;                                                  // T, kT, T^3 of this cell
                        pair_table_record(Fp, zp, mup, log10kB + lT, 3.0 * lT * kLog2_10, MUAX, A.nmu, A.mu_rule, 1, A.inv_h,
                                          A.x0_over_h, uef_first, uef_last, s_top, 0.0, 0.0, pq, pb, ww, info, flags);
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
                    R0[slot] = make_double2(__longlong_as_double(pq), pb);
                    R1[slot] = make_double2(ww[0], ww[1]);
                    R2[slot] = make_double2(ww[2], ww[3]);
                    R3[slot] = make_double2(1.0 - tw, tw);
                    RI[slot] = info;
                }
                __syncwarp();
                // ---- step B: walk the valid pairs ----
                for (int pj = 0; pj < cnt; ++pj) {
                    const double2 r0 = R0[pj], r1 = R1[pj], r2 = R2[pj], r3 = R3[pj];
                    const int inf = RI[pj];
                    const long long q = __double_as_longlong(r0.x);
                    const double qb = r0.y, v0 = r1.x, v1 = r1.y, v2 = r2.x, v3 = r2.y;
                    const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                    const int soff = (inf & 0x7FFF) * wst - c_lo + jlo - 1 + NPL * lane;
                    const int n0 = jlo - 1 + NPL * lane;
                    double f[NPL + 3];
#pragma unroll
                    for (int jn = 0; jn < NPL; ++jn)
                        f[1 + jn] = fma(r3.y, contract4(Shi + soff + jn, wst, v0, v1, v2, v3),
                                        fma(r3.x, contract4(Slo + soff + jn, wst, v0, v1, v2, v3), qb));
                    f[0] = __shfl_up_sync(0xffffffffu, f[NPL], 1);
                    if (NPL == 1) {
                        f[2] = __shfl_down_sync(0xffffffffu, f[1], 1);
                        f[3] = __shfl_down_sync(0xffffffffu, f[1], 2);
                    } else {
                        f[NPL + 1] = __shfl_down_sync(0xffffffffu, f[1], 1);
                        f[NPL + 2] = __shfl_down_sync(0xffffffffu, f[2], 1);
                    }
                    double2 ka[NPL], kb[NPL];
#pragma unroll
                    for (int jn = 0; jn < NPL; ++jn)
                        cubic_coeffs(f[jn], f[jn + 1], f[jn + 2], f[jn + 3], ka[jn].x, ka[jn].y, kb[jn].x, kb[jn].y);
                    if (jlo == 0 || jhi == nx - 2) {      // strategy d: linear in the first / last interval of the axis
#pragma unroll
                        for (int jn = 0; jn < NPL; ++jn) {
                            const int c = n0 + jn;
                            if (c != 0 && c != nx - 2) continue;
                            const double d = f[jn + 2] - f[jn + 1];             // y = f1 + d (t - 1)
                            ka[jn] = make_double2(f[jn + 1] - d, d);
                            kb[jn] = make_double2(0.0, 0.0);
                        }
                    }
                    __syncwarp();
#pragma unroll
                    for (int jn = 0; jn < NPL; ++jn) {
                        KA[NPL * lane + jn] = ka[jn];
                        KA[NPL * lane + jn + KW] = kb[jn];
                    }
                    __syncwarp();
                    const double2* KAq = KA + (1 - jlo);
                    if (!(inf & 0x8000)) {
#pragma unroll
                        for (int i = 0; i < EPL; ++i) {
                            const long long s = q + uef[i];
                            const int shi = (int)(s >> 32);
                            const double2* kp = KAq + (shi >> 20);
                            const double tau = __hiloint2double(one_plus_frac_hi(shi), (int)s);   // t = 1 + fraction (see cubic_coeffs)
                            const double2 c01 = kp[0], c23 = kp[KW];
                            const double y = fma(fma(fma(c23.y, tau, c23.x), tau, c01.y), tau, c01.x);
                            const double r = y + kMagic;
                            const int n = __double2loint(r);
                            const double val = exp2_frac_scaled(y - (r - kMagic), n);
                            if (n >= -1000) acc[i] += val;
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < EPL; ++i) {
                            long long s = q + uef[i];
                            s = s < 0 ? 0 : (s > s_top ? s_top : s);             // clamp to the table (reading R13b)
                            const int shi = (int)(s >> 32);
                            const double2* kp = KAq + (shi >> 20);
                            const double tau = __hiloint2double(one_plus_frac_hi(shi), (int)s);   // t = 1 + fraction (see cubic_coeffs)
                            const double2 c01 = kp[0], c23 = kp[KW];
                            const double y = fma(fma(fma(c23.y, tau, c23.x), tau, c01.y), tau, c01.x);
                            const double r = y + kMagic;
                            const int n = __double2loint(r);
                            const double val = exp2_frac_scaled(y - (r - kMagic), n);
                            if (n >= -1000) acc[i] += val;
                        }
                    }
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
            if (e < A.nE) {                                                      // the 1/E_e of Eq 47
                const double v = acc[i] / A.en[e];
                out[e] = (!WIN && A.map_split) ? out[e] + v : v;                   // the full-width launch runs second and adds
            }
        }
    }
}

}  // namespace ppm
