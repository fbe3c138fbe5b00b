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
// Everything per pair and per triple is k_cells_tab's own code (pair_table_record, fused_pass with a node functor that
// blends the two slices, pair_energies with the stepped coordinate and the deferred clamped groups), with T, kT and T^3
// taken per cell.
#pragma once
#include "ppm_cells.cuh"

namespace ppm {

__device__ __forceinline__ double contract4(const double* __restrict__ sp0, int nx, double v0, double v1, double v2, double v3)
{
    return fma(v3, sp0[3 * nx], fma(v2, sp0[2 * nx], fma(v1, sp0[nx], v0 * sp0[0])));
}

// Node value of a pair in temperature-map mode: the (log T, mu) stencil -- 2 x 4 weights (1 - t) v_mu, t v_mu, formed once
// per pair in step A -- on the slices of the two log T nodes that bracket the cell's temperature, plus log2(F_p T^3).
// `lo` / `hi` point at the stencil's first mu row of the two slice buffers, each shifted by its own first column so that
// column n of the table is element n.
struct MapNode {
    const double* lo;
    const double* hi;
    int stride;
    double a0, a1, a2, a3, b0, b1, b2, b3, qb;   // (1 - t) v_mu and t v_mu: the (log T, mu) stencil's eight weights
    __device__ __forceinline__ double operator()(int n) const
    {
        const double* pl = lo + n;
        const double* ph = hi + n;
        double f = fma(a0, pl[0], qb);
        f = fma(b0, ph[0], f);
        f = fma(a1, pl[stride], f);
        f = fma(b1, ph[stride], f);
        f = fma(a2, pl[2 * stride], f);
        f = fma(b2, ph[2 * stride], f);
        f = fma(a3, pl[3 * stride], f);
        return fma(b3, ph[3 * stride], f);
    }
    __device__ __forceinline__ void check(int, int, const double*) const {}
};

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

// Columns held by the slice of log T node it + 1 when it is staged as the UPPER node of interval `it`: the interval's
// window, widened to the next interval's window when the row also has cells there -- that interval then finds its lower
// node already in shared memory (one new slice per step instead of two).  [c_lo, c_hi] = the window of interval `it`.
__device__ inline void map_upper_window(const RowD& row, const double* __restrict__ axT, int nT, int it, double inv_h,
                                        double x0_over_h, double ue_first, double ue_last, int nx, int c_lo, int c_hi,
                                        int& n_lo, int& n_hi)
{
    n_lo = c_lo; n_hi = c_hi;
    if ((row.tmask >> (it + 1)) & 1ull) {
        int a_lo, a_hi;
        map_window(row, axT, nT, it + 1, inv_h, x0_over_h, ue_first, ue_last, nx, a_lo, a_hi);
        n_lo = imin_(n_lo, a_lo); n_hi = imax_(n_hi, a_hi);
    }
}

// does every node slice of the row fit a window of `wst` columns?  (rows that do not are left to the full-width kernel)
__device__ inline bool map_row_fits(const RowD& row, const double* __restrict__ axT, int nT, double inv_h, double x0_over_h,
                                    double ue_first, double ue_last, int nx, int wst)
{
    for (unsigned long long tm = row.tmask; tm; tm &= tm - 1) {
        const int it = __ffsll((long long)tm) - 1;
        int c_lo, c_hi, n_lo, n_hi;
        map_window(row, axT, nT, it, inv_h, x0_over_h, ue_first, ue_last, nx, c_lo, c_hi);
        map_upper_window(row, axT, nT, it, inv_h, x0_over_h, ue_first, ue_last, nx, c_lo, c_hi, n_lo, n_hi);
        if (n_hi - n_lo + 1 > wst) return false;
    }
    return true;
}

// WIN = true: 16 warps, the two node slices hold only the window's columns (row stride A.wst); rows whose windows do not
// fit are skipped and counted in A.pairs[1] (the WIN = false launch takes them, and returns at once when there are none).
// WIN = false: 8 warps, full-width slices (row stride nx).
template <int EPL, int NPL, bool WIN, bool UNI>
__global__ void __launch_bounds__(WIN ? 512 : 256, 1) k_cells_map(CellArgs A)
{
    extern __shared__ __align__(16) double sm[];
    if (!WIN && A.map_split && A.pairs[1] == 0ull) return;                      // every row was taken by the windowed launch
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
    // shared layout (doubles): per warp { KA [KW], KB [KW], R0 (q, qb), R1 (a0, a1), R2 (a2, a3), R3 (b0, b1), R4 (b2, b3) [32]
    // as double2, RI [32] int2 (info, flags) } | S0 [nmu][wst] | S1 [nmu][wst] | T [4][n1] | MUAX [nmu] | TAX [nT] | UG [16]
    constexpr int KW = 32 * NPL;
    constexpr int WARP_DBL = 4 * KW + 5 * 64 + 32;
    double* wbase = sm + (size_t)w * WARP_DBL;
    double2* KA = reinterpret_cast<double2*>(wbase);
    double2* R0 = KA + 2 * KW;
    double2* R1 = R0 + 32;
    double2* R2 = R1 + 32;
    double2* R3 = R2 + 32;
    double2* R4 = R3 + 32;
    int2* RI = reinterpret_cast<int2*>(R4 + 32);
    double* Sb0 = sm + (size_t)A.nw * WARP_DBL;
    double* Sb1 = Sb0 + plane;
    double* T = Sb1 + plane;
    double* MUAX = T + 4 * n1;
    double* TAX = MUAX + A.nmu;
    long long* UG = reinterpret_cast<long long*>(TAX + A.nT);
    constexpr int NG = EPL;

    EnergyCoord<EPL, UNI> ec;
    ec.init(A.uef, A.uef_step, e0, lane, A.nE);
    double acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) acc[i] = 0.0;
    double hdef = 0.0;
    const long long uef_first = A.uef[imin_(e0, A.nE - 1)];
    const int e_last = imin_(e0 + 32 * EPL, A.nE) - 1;
    const long long uef_last = UNI ? A.uef[e0 + ((e_last - e0) & 31)] + (long long)((e_last - e0) >> 5) * A.uef_step
                                   : A.uef[e_last];
    const long long s_top = ((long long)(nx - 1) << 52) - 1;
    const double ue_first = (double)uef_first / kTwo52, ue_last = (double)uef_last / kTwo52;
    for (int i = threadIdx.x; i < A.nmu; i += blockDim.x) MUAX[i] = A.axmu[i];
    for (int i = threadIdx.x; i < A.nT; i += blockDim.x) TAX[i] = A.axT[i];
    if (threadIdx.x < NG) {
        const int ef = e0 + 32 * (int)threadIdx.x;
        UG[threadIdx.x] = (ef < A.nE) ? (UNI ? A.uef[e0] + (long long)threadIdx.x * A.uef_step : A.uef[ef]) : (1ll << 62);
    }

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
            if (fits != WIN) {
                if (WIN && pg == 0 && et == 0 && threadIdx.x == 0) atomicAdd(A.pairs + 1, 1ull);
                continue;
            }
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
        // the row's two log g nodes (strategy d: linear; axis_w4 puts the weights at stencil offsets o, o + 1)
        int go = 0;
        while (go < 2 && row.wg[go] == 0.0) ++go;
        const double wga = row.wg[go], wgb = row.wg[go + 1];
        const size_t gplane = (size_t)A.nmu * nx;
        int pos = 0;                                                             // next unprocessed entry of the sorted cell list
        int node0 = -1, node1 = -1;                                              // log T node held by slice buffer 0 / 1
        int off0 = 0, off1 = 0;                                                  // first table column held by buffer 0 / 1
        for (unsigned long long tm = row.tmask; tm; tm &= tm - 1) {
            const int it = __ffsll((long long)tm) - 1;                           // log T interval [it, it+1]
            int c_lo = 0, c_hi = nx - 1;
            if (WIN) map_window(row, A.axT, A.nT, it, A.inv_h, A.x0_over_h, ue_first, ue_last, nx, c_lo, c_hi);
            // the previous interval's upper node is this interval's lower node when the intervals are adjacent; its slice
            // was staged wide enough for both (map_upper_window): ping-pong, one new slice per step
            const int pl = (node1 == it) ? 1 : 0;
            __syncthreads();                                                     // readers of the previous interval are done
#pragma unroll
            for (int h = 0; h < 2; ++h) {                                        // h = 0: lower node -> buffer pl; 1: upper -> 1 - pl
                const int buf = h ? 1 - pl : pl, node = it + h;
                if ((buf ? node1 : node0) == node) continue;
                int n_lo = c_lo, n_hi = c_hi;
                if (WIN && h) map_upper_window(row, A.axT, A.nT, it, A.inv_h, A.x0_over_h, ue_first, ue_last, nx, c_lo, c_hi, n_lo, n_hi);
                if (buf) { node1 = node; off1 = n_lo; } else { node0 = node; off0 = n_lo; }
                double* dst = buf ? Sb1 : Sb0;
                const double* src = A.values + ((size_t)node * A.ng + row.bg + go) * gplane + n_lo;
                const int wcols = n_hi - n_lo + 1;
                // 128 consecutive threads walk the columns of one mu row (coalesced), blockDim / 128 rows per pass; kDepth
                // passes' loads are issued before their blends (2 kDepth independent L2 loads in flight per thread: the
                // staging is latency-bound, and with one pass at a time it cost as much as the interval's arithmetic)
                constexpr int kDepth = 6;
                const int rstep = (int)(blockDim.x >> 7);
                for (int col = threadIdx.x & 127; col < wcols; col += 128) {
                    for (int mu_0 = threadIdx.x >> 7; mu_0 < A.nmu; mu_0 += kDepth * rstep) {
                        double va[kDepth], vb[kDepth];
#pragma unroll
                        for (int u = 0; u < kDepth; ++u) {
                            const int mu_i = imin_(mu_0 + u * rstep, A.nmu - 1);
                            const double* s0 = src + (size_t)mu_i * nx + col;
                            va[u] = __ldg(s0);
                            vb[u] = __ldg(s0 + gplane);
                        }
#pragma unroll
                        for (int u = 0; u < kDepth; ++u) {
                            const int mu_i = mu_0 + u * rstep;
                            if (mu_i < A.nmu) dst[mu_i * wst + col] = fma(wgb, vb[u], wga * va[u]);
                        }
                    }
                }
            }
            __syncthreads();
            if (!kvalid) continue;
            const double* Slo = pl ? Sb1 - off1 : Sb0 - off0;                    // column n of the table is element n
            const double* Shi = pl ? Sb0 - off0 : Sb1 - off1;
            const double po0 = PO[0];
            // the row's list is sorted by log T interval (k_rows): the cells of interval `it` start at `pos`
            for (bool more = true; more;) {
                // ---- step A: lane <-> cell of this interval ----
                const int idx = pos + lane;
                double Fp = 0.0, pb = 0.0, tw = 0.0;
                long long pq = 0;
                double ww[4] = {0.0, 0.0, 0.0, 0.0};
                int info = 0, flags = 0;
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
                    if (Fp != 0.0) {                                                 // T, kT, T^3 of this cell
                        pair_table_record(Fp, zp, mup, log10kB + lT, 3.0 * lT * kLog2_10, MUAX, A.nmu, A.mu_rule, wst, A.inv_h,
                                          A.x0_over_h, uef_first, uef_last, s_top, A.y_lo, A.y_hi, pq, pb, ww, info, flags);
                        if (flags == PAIR_CLAMP_HI) flags |= clamped_groups<NG>(pq, UG, s_top) << 8;
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
                    const double tl = 1.0 - tw;
                    R1[slot] = make_double2(tl * ww[0], tl * ww[1]);
                    R2[slot] = make_double2(tl * ww[2], tl * ww[3]);
                    R3[slot] = make_double2(tw * ww[0], tw * ww[1]);
                    R4[slot] = make_double2(tw * ww[2], tw * ww[3]);
                    RI[slot] = make_int2(info, flags);
                }
                __syncwarp();
                // ---- step B: walk the valid pairs ----
                for (int pj = 0; pj < cnt; ++pj) {
                    const double2 r0 = R0[pj], r1 = R1[pj], r2 = R2[pj], r3 = R3[pj], r4 = R4[pj];
                    const int2 ri2 = RI[pj];
                    const int inf = ri2.x;
                    const long long q = __double_as_longlong(r0.x);
                    const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                    const MapNode node{Slo + (inf & 0xFFFF), Shi + (inf & 0xFFFF), wst, r1.x, r1.y, r2.x, r2.y, r3.x, r3.y, r4.x, r4.y, r0.y};
                    fused_pass<NPL>(node, nx, jlo, jhi, lane, 1, KA, sm);           // strategy d: linear first / last interval
                    pair_energies<KW, EPL, UNI>(acc, hdef, ec, KA + (1 - jlo), q, ri2.y, s_top, lane, sm);
                }
            }
        }
    }
    if (kvalid && et == 0 && lane == 0 && npairs) atomicAdd(A.pairs, (unsigned long long)npairs);
    spread_deferred<EPL>(acc, hdef, lane);
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
