// ppm_cells_map4.cuh -- S4 + S5 for a per-cell effective-temperature map (reading R24) under the
// interpolation strategies that are CUBIC in log T: a, b (cubic on all four axes, stencil shifted inward at the table's
// edges) and c (cubic, linear in the first / last interval of log T, log g, log x) -- PAPER.md:504, 551; readings R13c-e.
// Product path (sm_100a).
//
// A pair needs the (mu x logx) slices of the FOUR log T nodes s .. s+3 around its cell's interval `it`
// (s = clamp(it - 1, 0, nT - 4): the placement of axis_w4):
//   f_node = log2(10) sum_a wT_a sum_mu w_mu S_{s+a}[mu][c] + log2(F_p T^3).
// Four slices only fit shared memory when they are cut to the logx columns the interval's pairs can reach AND the
// energy grid is cut into tiles (the host picks the tiling: at 300 energies two tiles of 150, 8 warps).  The block walks
// the row's intervals in ascending order (the cell list is sorted by interval, k_rows); the slice of node n lives in
// buffer n & 3, so consecutive intervals reuse three of their four slices; a slice is staged wide enough for every later
// interval of the row that uses it when that fits (map4_node_window).  The slices are blended over the row's log g
// stencil (up to 4 nodes) on the fly from the L2-resident table.  Per pair and per triple everything is k_cells_tab's
// code (pair_table_record, fused_pass with the Map4Node functor, pair_energies).
// A row whose single-interval window exceeds the buffers (cell temperatures far outside the table's axis) cannot be
// evaluated in this mode: its vector gets PPM_STATUS_MAP_WINDOW and a NaN flux.
#pragma once
#include "ppm_cells_map.cuh"

namespace ppm {

constexpr int kStatusMapWindow = 8;      // = PPM_STATUS_MAP_WINDOW of include/ppm.h

struct Map4Node {
    const double* s0;                    // the stencil's first mu row in the buffers of nodes s, s+1, s+2, s+3, each shifted
    const double* s1;                    // by its own first column so that column n of the table is element n
    const double* s2;
    const double* s3;
    int stride;
    double v0, v1, v2, v3;               // mu weights (pre-scaled by log2(10))
    double t0, t1, t2, t3;               // log T weights
    double qb;                           // log2(F_p T^3)
    __device__ __forceinline__ double operator()(int n) const
    {
        double f = fma(t0, contract4(s0 + n, stride, v0, v1, v2, v3), qb);
        f = fma(t1, contract4(s1 + n, stride, v0, v1, v2, v3), f);
        f = fma(t2, contract4(s2 + n, stride, v0, v1, v2, v3), f);
        return fma(t3, contract4(s3 + n, stride, v0, v1, v2, v3), f);
    }
    __device__ __forceinline__ void check(int, int, const double*) const {}
};

__device__ __forceinline__ int map4_base(int it, int nT) { return imin_(imax_(it - 1, 0), nT - 4); }

// Columns to hold for log T node `node` when it is staged at interval `it` (whose own window is [c_lo, c_hi]): the union
// with the windows of the row's later intervals whose stencil still contains the node, as long as that fits `wst`.
__device__ inline void map4_node_window(const RowD& row, const double* __restrict__ axT, int nT, int it, int node, double inv_h,
                                        double x0_over_h, double ue_first, double ue_last, int nx, int wst, int c_lo, int c_hi,
                                        int& n_lo, int& n_hi)
{
    n_lo = c_lo; n_hi = c_hi;
    unsigned long long later = (it >= 63) ? 0ull : (row.tmask >> (it + 1)) << (it + 1);
    for (; later; later &= later - 1) {
        const int it2 = __ffsll((long long)later) - 1;
        if (map4_base(it2, nT) > node) break;
        int a_lo, a_hi;
        map_window(row, axT, nT, it2, inv_h, x0_over_h, ue_first, ue_last, nx, a_lo, a_hi);
        const int u_lo = imin_(n_lo, a_lo), u_hi = imax_(n_hi, a_hi);
        if (u_hi - u_lo + 1 > wst) break;
        n_lo = u_lo; n_hi = u_hi;
    }
}

// does every interval of the row fit a window of `wst` columns on its own?
__device__ inline bool map4_row_fits(const RowD& row, const double* __restrict__ axT, int nT, double inv_h, double x0_over_h,
                                     double ue_first, double ue_last, int nx, int wst)
{
    for (unsigned long long tm = row.tmask; tm; tm &= tm - 1) {
        int c_lo, c_hi;
        map_window(row, axT, nT, __ffsll((long long)tm) - 1, inv_h, x0_over_h, ue_first, ue_last, nx, c_lo, c_hi);
        if (c_hi - c_lo + 1 > wst) return false;
    }
    return true;
}

template <int EPL, int NPL>
__global__ void __launch_bounds__(512, 1) k_cells_map4(CellArgs A, StarD* stars_rw)
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
    const int wst = A.wst;                                                      // row stride of the four slice buffers
    const int plane = A.nmu * wst;
    // shared layout (doubles): per warp { KA [KW], KB [KW], R0 (q, qb), R1 (v0, v1), R2 (v2, v3), R3 (t0, t1), R4 (t2, t3) [32]
    // as double2, RI [32] int2 (info, flags) } | S [4][nmu][wst] | T [4][n1] | MUAX [nmu] | TAX [nT] | UG [16]
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
    double* Sb = sm + (size_t)A.nw * WARP_DBL;
    double* T = Sb + 4 * (size_t)plane;
    double* MUAX = T + 4 * n1;
    double* TAX = MUAX + A.nmu;
    long long* UG = reinterpret_cast<long long*>(TAX + A.nT);
    constexpr int NG = EPL;

    EnergyCoord<EPL, false> ec;
    ec.init(A.uef, 0, e0, lane, A.nE);
    double acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) acc[i] = 0.0;
    double hdef = 0.0;
    const long long uef_first = A.uef[imin_(e0, A.nE - 1)];
    const long long uef_last = A.uef[imin_(e0 + 32 * EPL, A.nE) - 1];
    const long long s_top = ((long long)(nx - 1) << 52) - 1;
    const double ue_first = (double)uef_first / kTwo52, ue_last = (double)uef_last / kTwo52;
    for (int i = threadIdx.x; i < A.nmu; i += blockDim.x) MUAX[i] = A.axmu[i];
    for (int i = threadIdx.x; i < A.nT; i += blockDim.x) TAX[i] = A.axT[i];
    if (threadIdx.x < NG) {
        const int ef = e0 + 32 * (int)threadIdx.x;
        UG[threadIdx.x] = (ef < A.nE) ? A.uef[ef] : (1ll << 62);
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
        if (!map4_row_fits(row, A.axT, A.nT, A.inv_h, A.x0_over_h, ue_first, ue_last, nx, wst)) {
            if (threadIdx.x == 0) atomicOr(&stars_rw[b].status, kStatusMapWindow);   // k_reduce fills the vector's flux with NaN
            continue;
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
        const size_t gplane = (size_t)A.nmu * nx;
        int pos = 0;                                                             // next unprocessed entry of the sorted cell list
        int bn0 = -1, bn1 = -1, bn2 = -1, bn3 = -1;                              // log T node held by buffer 0..3
        int lo0 = 0, lo1 = 0, lo2 = 0, lo3 = 0, hi0 = -1, hi1 = -1, hi2 = -1, hi3 = -1;   // its table columns [lo, hi]
        for (unsigned long long tm = row.tmask; tm; tm &= tm - 1) {
            const int it = __ffsll((long long)tm) - 1;                           // log T interval [it, it+1]
            const int sT = map4_base(it, A.nT);                                  // its stencil: nodes sT .. sT+3
            int c_lo, c_hi;
            map_window(row, A.axT, A.nT, it, A.inv_h, A.x0_over_h, ue_first, ue_last, nx, c_lo, c_hi);
            __syncthreads();                                                     // readers of the previous interval are done
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int node = sT + j, bq = node & 3;
                const int held = bq == 0 ? bn0 : bq == 1 ? bn1 : bq == 2 ? bn2 : bn3;
                const int hlo = bq == 0 ? lo0 : bq == 1 ? lo1 : bq == 2 ? lo2 : lo3;
                const int hhi = bq == 0 ? hi0 : bq == 1 ? hi1 : bq == 2 ? hi2 : hi3;
                if (held == node && hlo <= c_lo && hhi >= c_hi) continue;         // staged earlier, wide enough
                int n_lo, n_hi;
                map4_node_window(row, A.axT, A.nT, it, node, A.inv_h, A.x0_over_h, ue_first, ue_last, nx, wst, c_lo, c_hi,
                                 n_lo, n_hi);
                if (bq == 0) { bn0 = node; lo0 = n_lo; hi0 = n_hi; } else if (bq == 1) { bn1 = node; lo1 = n_lo; hi1 = n_hi; }
                else if (bq == 2) { bn2 = node; lo2 = n_lo; hi2 = n_hi; } else { bn3 = node; lo3 = n_lo; hi3 = n_hi; }
                double* dst = Sb + (size_t)bq * plane;
                const double* src = A.values + ((size_t)node * A.ng + row.bg) * gplane + n_lo;
                const int wcols = n_hi - n_lo + 1;
                // three (mu row, column) passes' loads -- up to 12 independent L2 loads per thread -- are issued before their
                // blends: the staging is bound by L2 latency (see k_cells_map)
                constexpr int kDepth = 3;
                const int rstep = (int)(blockDim.x >> 7);
                const double wg0 = row.wg[0], wg1 = row.wg[1], wg2 = row.wg[2], wg3 = row.wg[3];
                for (int col = threadIdx.x & 127; col < wcols; col += 128) {
                    for (int mu_0 = threadIdx.x >> 7; mu_0 < A.nmu; mu_0 += kDepth * rstep) {
                        double x[kDepth][4];
#pragma unroll
                        for (int u = 0; u < kDepth; ++u) {
                            const double* s0 = src + (size_t)imin_(mu_0 + u * rstep, A.nmu - 1) * nx + col;
                            x[u][0] = (wg0 != 0.0) ? __ldg(s0) : 0.0;
                            x[u][1] = (wg1 != 0.0) ? __ldg(s0 + gplane) : 0.0;
                            x[u][2] = (wg2 != 0.0) ? __ldg(s0 + 2 * gplane) : 0.0;
                            x[u][3] = (wg3 != 0.0) ? __ldg(s0 + 3 * gplane) : 0.0;
                        }
#pragma unroll
                        for (int u = 0; u < kDepth; ++u) {
                            const int mu_i = mu_0 + u * rstep;
                            double v = 0.0;                                      // zero weights are skipped, as in k_slice
                            if (wg0 != 0.0) v = fma(wg0, x[u][0], v);
                            if (wg1 != 0.0) v = fma(wg1, x[u][1], v);
                            if (wg2 != 0.0) v = fma(wg2, x[u][2], v);
                            if (wg3 != 0.0) v = fma(wg3, x[u][3], v);
                            if (mu_i < A.nmu) dst[mu_i * wst + col] = v;
                        }
                    }
                }
            }
            __syncthreads();
            if (!kvalid) continue;
            // buffer of stencil node j (node sT + j): ((sT + j) & 3); column n of the table is element n
            const double* P[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int bq = (sT + j) & 3;
                const int blo = bq == 0 ? lo0 : bq == 1 ? lo1 : bq == 2 ? lo2 : lo3;
                P[j] = Sb + (size_t)bq * plane - blo;
            }
            const double po0 = PO[0];
            // the row's list is sorted by log T interval (k_rows): the cells of interval `it` start at `pos`
            for (bool more = true; more;) {
                // ---- step A: lane <-> cell of this interval ----
                const int idx = pos + lane;
                double Fp = 0.0, pb = 0.0;
                long long pq = 0;
                double ww[4] = {0.0, 0.0, 0.0, 0.0}, wt[4] = {0.0, 0.0, 0.0, 0.0};
                int info = 0, flags = 0;
                const int entry = (idx < nact) ? cl[idx] : -1;
                const bool mine = (entry >= 0) && ((entry >> 16) == it);
                const int n_mine = __popc(__ballot_sync(0xffffffffu, mine));     // a prefix of the batch (sorted list)
                pos += n_mine;
                more = (n_mine == 32);
                if (mine) {
                    const int m = entry & 0xFFFF;
                    const double lT = tcell[m];
                    const double phi_p = phase_of_cell(phi_out, cell_azimuth(A.mesh, row, sp, m), phi_off, po0);   // Eq 45
                    double zp, mup;
                    template_interp(F, Z, PO, MU, A.n_fp, A.phase_order, phi_p, Fp, zp, mup);                  // Eq 46
                    if (!(Fp > 0.0)) Fp = 0.0;
                    if (Fp != 0.0) {                                                 // T, kT, T^3 of this cell
                        int bT;
                        axis_w4(TAX, A.nT, lT, A.t_rule, bT, wt);                    // bT == sT (same interval, same placement)
                        pair_table_record(Fp, zp, mup, log10kB + lT, 3.0 * lT * kLog2_10, MUAX, A.nmu, A.mu_rule, wst, A.inv_h,
                                          A.x0_over_h, uef_first, uef_last, s_top, A.y_lo, A.y_hi, pq, pb, ww, info, flags);
                        if (flags == PAIR_CLAMP_HI) flags |= clamped_groups<NG>(pq, UG, s_top) << 8;
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
                    R3[slot] = make_double2(wt[0], wt[1]);
                    R4[slot] = make_double2(wt[2], wt[3]);
                    RI[slot] = make_int2(info, flags);
                }
                __syncwarp();
                // ---- step B: walk the valid pairs ----
                for (int pj = 0; pj < cnt; ++pj) {
                    const double2 r0 = R0[pj], r1 = R1[pj], r2 = R2[pj], r3 = R3[pj], r4 = R4[pj];
                    const int2 ri2 = RI[pj];
                    const int inf = ri2.x, mo = inf & 0xFFFF;
                    const long long q = __double_as_longlong(r0.x);
                    const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                    const Map4Node node{P[0] + mo, P[1] + mo, P[2] + mo, P[3] + mo, wst, r1.x, r1.y, r2.x, r2.y,
                                        r3.x, r3.y, r4.x, r4.y, r0.y};
                    fused_pass<NPL>(node, nx, jlo, jhi, lane, A.x_linedge, KA, sm);
                    pair_energies<KW, EPL, false>(acc, hdef, ec, KA + (1 - jlo), q, ri2.y, s_top, lane, sm);
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
            if (e < A.nE) out[e] = acc[i] / A.en[e];                            // the 1/E_e of Eq 47
        }
    }
}

}  // namespace ppm
