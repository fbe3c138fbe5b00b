// ppm_cells_yx.cuh -- S4 + S5, table emission on a log-uniform energy grid: the "y-exchange" form of the cell kernel.
// Product path (sm_100a).  Same block / warp / lane ownership of the OUTPUT as k_cells_tab (warp = output phase, lane l
// owns energies e0 + l + 32 i, accumulators in registers, no atomics) and the same step A, node contraction and
// per-interval cubics (ppm_cells.cuh).  What differs is who evaluates the cubic:
//   k_cells_tab:  the lane that owns the interval writes its coefficient record (32 B) to shared memory; every energy's
//                 lane fetches the record of its interval (2 x LDS.128 per triple).  On sm_100a a 128-bit load costs 4
//                 shared-memory wavefronts unless both lanes of every aligned lane pair read the same address, so the
//                 warp pays 8 wavefronts per energy group for about 11 distinct records: the kernel sits at 88 % of the
//                 shared-memory wavefront peak with the FP64 pipe at 59 % (profiles/r2c_k_cells_tab.md).
//   k_cells_yx:   the lane that owns the interval keeps the coefficients in REGISTERS and evaluates the cubic itself at
//                 the energies that fall into its intervals (log-uniform grid: energy index e <-> coordinate
//                 base + e * step, so a lane finds its first energy by one division and walks on by additions), and
//                 writes y = log2(term) -- 8 bytes per energy -- to a per-warp array; after one __syncwarp the energy's
//                 own lane reads its y (LDS.64, conflict-free) and does 2^y and the accumulation.  32 -> 16 bytes of
//                 shared-memory traffic per triple, no 128-bit loads, and the per-triple 64-bit coordinate arithmetic of
//                 the energy lanes disappears.
// Energies beyond the table (reading R13b: the coordinate clamps, the term is the pair's constant): the y of the axis' end
// is filled in for the straddling energy group; whole groups beyond the top are deferred exactly as in k_cells_tab.
// Taken by the host when ppm_uniform_energy() holds and an interval holds at most 4 energies; otherwise k_cells_tab.
#pragma once
#include "ppm_cells.cuh"

namespace ppm {

// 2^y with y = n + f split by the 1.5 * 2^52 constant (see exp2_frac_scaled)
__device__ __forceinline__ double exp2_of(double y)
{
    const double r = y + kMagic;
    return exp2_frac_scaled(y - (r - kMagic), __double2loint(r));
}

// range-checked form: below 2^-1000 the term is 0, above 2^1000 it is +inf
__device__ __forceinline__ double exp2_of_checked(double y)
{
    const double r = y + kMagic;
    const double v = exp2_frac_scaled(y - (r - kMagic), __double2loint(r));
    return !(y > -1000.0) ? 0.0 : (y > 1000.0 ? INFINITY : v);
}

template <int EPL, int G>
__device__ __forceinline__ void yx_groups(int g, double (&acc)[EPL], const double* __restrict__ Yl)
{
    if (g == G) {
#pragma unroll
        for (int i = 0; i < G; ++i) acc[i] += exp2_of(Yl[32 * i]);
    } else if constexpr (G > 1) yx_groups<EPL, G - 1>(g, acc, Yl);
}

template <int EPL, int NPL>
__global__ void __launch_bounds__(512, 1) k_cells_yx(CellArgs A)
{
    extern __shared__ __align__(16) double sm[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int chunk = blockIdx.x, pg = blockIdx.y;
    const int b = blockIdx.z / A.n_etile, et = blockIdx.z % A.n_etile;
    const int k = pg * A.nw + w;
    const bool kvalid = k < A.n_phase;
    const int e0 = et * 32 * EPL;
    const int ne = imin_(32 * EPL, A.nE - e0);                                  // energies of this tile
    const int n1 = A.n_fp + 1;
    const int nx = A.nx;
    const int plane = A.nmu * nx;
    // shared layout (doubles): per warp { Y [2][32 EPL] (two buffers: one __syncwarp per pair), R0 [32] (q, qb), R1 [32]
    // (v0, v1), R2 [32] (v2, v3) as double2, RI [32] int2 (info, flags) } | S [nmu][nx] | T [4][n1] | MUAX [nmu] | UG [16]
    constexpr int NY = 32 * EPL;
    constexpr int WARP_DBL = 2 * NY + 3 * 64 + 32;
    double* wbase = sm + (size_t)w * WARP_DBL;
    double* Y = wbase;
    double2* R0 = reinterpret_cast<double2*>(wbase + 2 * NY);
    double2* R1 = R0 + 32;
    double2* R2 = R1 + 32;
    int2* RI = reinterpret_cast<int2*>(R2 + 32);
    double* S = sm + (size_t)A.nw * WARP_DBL;
    double* T = S + plane;
    double* MUAX = T + 4 * n1;
    long long* UG = reinterpret_cast<long long*>(MUAX + A.nmu);                 // [NG]: coordinate part of each group's first energy
    constexpr int NG = EPL;

    double acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) acc[i] = 0.0;
    double hdef = 0.0;                           // lane g: sum of the constants 2^y(s_top) of the pairs whose groups >= g are clamped
    const long long step1 = A.uef_step1;
    const long long U0 = A.uef[e0];                                             // energy k of the tile: U0 + k step1 (R27)
    const long long uef_first = U0, uef_last = U0 + (long long)(ne - 1) * step1;
    const long long s_top = ((long long)(nx - 1) << 52) - 1;                     // largest in-table coordinate
    const int kmax = A.kmax;
    for (int i = threadIdx.x; i < A.nmu; i += blockDim.x) MUAX[i] = A.axmu[i];
    if (threadIdx.x < NG)                        // a group without any energy (ragged tail) counts as beyond the table
        UG[threadIdx.x] = (32 * (int)threadIdx.x < ne) ? U0 + 32ll * threadIdx.x * step1 : (1ll << 62);

    const StarD& st = A.stars[b];
    const double phi_off = st.phi_off;
    const double phi_out = (double)k / A.n_phase;                               // reading R3
    unsigned npairs = 0;
    int ybuf = 0;

    for (int ri = 0; ri < A.rows_per_chunk; ++ri) {
        const int rl = chunk + ri * A.nchunk;                                   // strided chunks balance row sizes
        if (rl >= A.RT) break;
        const int rid = b * A.RT + rl;
        const RowD& row = A.rows[rid];
        const int nact = row.n_active;
        if (nact == 0 || !row.visible) continue;
        const SpotD& sp = A.spots[rid / A.n_theta];
        __syncthreads();
        {   // stage slice + template (16-byte loads)
            if ((plane & 1) == 0) {
                const double2* src = reinterpret_cast<const double2*>(A.slices + (size_t)rid * plane);
                double2* dst = reinterpret_cast<double2*>(S);
                for (int i = threadIdx.x; i < plane / 2; i += blockDim.x) dst[i] = src[i];
            } else {
                const double* src = A.slices + (size_t)rid * plane;
                for (int i = threadIdx.x; i < plane; i += blockDim.x) S[i] = src[i];
            }
            const double* ts = A.tmpl + (size_t)rid * 4 * n1;
            for (int i = threadIdx.x; i < 4 * n1; i += blockDim.x) T[i] = ts[i];
        }
        __syncthreads();
        if (!kvalid) continue;
        const double* F = T;
        const double* Z = T + n1;
        const double* PO = T + 2 * n1;
        const double* MU = T + 3 * n1;
        const int* cl = A.cells + (size_t)rid * A.n_phi;
        const double po0 = PO[0];
        for (int base = 0; base < nact; base += 32) {
            // ---- step A: lane <-> cell; Eq 45-46 and the per-pair record, compacted over the pairs with F_p != 0 ----
            const int idx = base + lane;
            double Fp = 0.0, pb = 0.0;                // pb = log2(F_p T^3)
            long long pq = 0;                         // u_pair in units of 2^-52 intervals
            double ww[4] = {0.0, 0.0, 0.0, 0.0};
            int info = 0, flags = 0;
            if (idx < nact) {
                const double phi_p = phase_of_cell(phi_out, cell_azimuth(A.mesh, row, sp, cl[idx]), phi_off, po0);   // Eq 45
                double zp, mup;
                template_interp(F, Z, PO, MU, A.n_fp, A.phase_order, phi_p, Fp, zp, mup);                            // Eq 46
                if (!(Fp > 0.0)) Fp = 0.0;
                if (Fp != 0.0) {
                    pair_table_record(Fp, zp, mup, sp.log10kT, sp.log2T3, MUAX, A.nmu, A.mu_rule, nx, A.inv_h, A.x0_over_h,
                                      uef_first, uef_last, s_top, A.y_lo, A.y_hi, pq, pb, ww, info, flags);
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
                RI[slot] = make_int2(info, flags);
            }
            __syncwarp();
            // ---- step B: walk the valid pairs ----
            for (int pj = 0; pj < cnt; ++pj) {
                const double2 r0 = R0[pj], r1 = R1[pj], r2 = R2[pj];
                const int2 ri2 = RI[pj];
                const int inf = ri2.x, flg = ri2.y;
                const long long q = __double_as_longlong(r0.x);
                const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                const SliceNode node{S + (inf & 0xFFFF), nx, r1.x, r1.y, r2.x, r2.y, r0.y};
                double2 ka[NPL], kb[NPL];
                interval_coeffs<NPL>(node, nx, jlo, jhi, lane, A.x_linedge, ka, kb, sm);
                // ---- phase 1: the interval's lane evaluates y at the energies inside its intervals ----
                double* Yb = Y + ybuf * NY;
                ybuf ^= 1;
                const int n0 = jlo - 1 + NPL * lane;
                const long long sbase = q + U0;                                  // coordinate of the tile's energy 0
                // first energy at or beyond the lane's first real interval: estimate by one FP64 division, settle exactly
                const long long lo52 = (long long)imax_(n0, 0) << 52;
                const long long target = lo52 - sbase;
                int e = (target > 0) ? __double2int_ru((double)target * A.inv_step1) : 0;
                long long s = sbase + (long long)e * step1;
                if (s < lo52) { s += step1; ++e; }
                else if (e > 0 && s - step1 >= lo52) { s -= step1; --e; }
                const int e_first = e;                                           // lane 0: energies below it lie under the axis
                int e_top = ne;                                                  // first energy beyond the top of the axis
                // Slots: interval c = n0 + jn takes up to kmax energies.  Straight-line code (the store is predicated, the
                // walk advances by a masked add): a branch per slot would serialise the independent Horner chains.
                const unsigned ybase = (unsigned)__cvta_generic_to_shared(Yb);
#pragma unroll
                for (int jn = 0; jn < NPL; ++jn) {
                    const int c = n0 + jn;
                    const int real = ((c >= 0) && (c <= nx - 2)) ? 1 : 0;
#pragma unroll
                    for (int kk = 0; kk < 4; ++kk) {
                        if (kk < kmax) {
                            const int shi = (int)(s >> 32);
                            const int ok = real & (((shi >> 20) == c) ? 1 : 0) & ((e < ne) ? 1 : 0);
                            const double t = __hiloint2double(one_plus_frac_hi(shi), (int)s);
                            const double y = fma(fma(fma(kb[jn].y, t, kb[jn].x), t, ka[jn].y), t, ka[jn].x);
                            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %2, 0;\n\t@p st.shared.f64 [%0], %1;\n\t}"
                                         :: "r"(ybase + 8u * (unsigned)e), "d"(y), "r"(ok) : "memory");
                            s += step1 & -(long long)ok;
                            e += ok;
                        }
                    }
                    e_top = (c == nx - 2) ? e : e_top;
                }
                if (flg != 0) {
                    // ends of the axis (reading R13b): y of the clamped coordinate, from the lane that owns the end interval
                    if (flg & PAIR_CLAMP_HI) {
                        const int off = nx - 2 - (jlo - 1), lo_ = off / NPL, jo = off - lo_ * NPL;
                        double yt = 0.0;
                        if (lane == lo_) {
                            const double tt = __longlong_as_double(0x3FFFFFFFFFFFFFFFll);      // t of s_top: 2 - 2^-52
#pragma unroll
                            for (int jn = 0; jn < NPL; ++jn)
                                if (jn == jo) yt = fma(fma(fma(kb[jn].y, tt, kb[jn].x), tt, ka[jn].y), tt, ka[jn].x);
                        }
                        yt = __shfl_sync(0xffffffffu, yt, lo_);
                        const int et_ = __shfl_sync(0xffffffffu, e_top, lo_);
                        if ((flg & 7) == PAIR_CLAMP_HI) {
                            // groups >= g lie beyond the top for every lane: deferred (hdef); only group g - 1 straddles the end
                            const int g = flg >> 8;
                            if (g < EPL && lane == g) hdef += exp2_of(yt);
                            const int ei = lane + 32 * (g - 1);
                            if (g >= 1 && ei >= et_ && ei < ne) Yb[ei] = yt;
                        } else {
#pragma unroll
                            for (int i = 0; i < EPL; ++i)
                                if (lane + 32 * i >= et_ && lane + 32 * i < ne) Yb[lane + 32 * i] = yt;
                        }
                    }
                    if (flg & PAIR_CLAMP_LO) {
                        const int off = 0 - (jlo - 1), lo_ = off / NPL, jo = off - lo_ * NPL;       // jlo == 0 here
                        double yb = 0.0;
                        if (lane == lo_) {
#pragma unroll
                            for (int jn = 0; jn < NPL; ++jn)
                                if (jn == jo) yb = (kb[jn].y + kb[jn].x) + (ka[jn].y + ka[jn].x);       // t = 1
                        }
                        yb = __shfl_sync(0xffffffffu, yb, lo_);
                        const int eb_ = __shfl_sync(0xffffffffu, e_first, 0);
#pragma unroll
                        for (int i = 0; i < EPL; ++i)
                            if (lane + 32 * i < eb_) Yb[lane + 32 * i] = yb;
                    }
                }
                __syncwarp();
                // ---- phase 2: the energy's lane: 2^y and the accumulation ----
                const double* Yl = Yb + lane;
                if (flg == 0) {
#pragma unroll
                    for (int i = 0; i < EPL; ++i) acc[i] += exp2_of(Yl[32 * i]);
                } else if ((flg & 7) == PAIR_CLAMP_HI) {
                    yx_groups<EPL, EPL>(flg >> 8, acc, Yl);                       // groups >= g are deferred (hdef)
                } else {
#pragma unroll
                    for (int i = 0; i < EPL; ++i) acc[i] += exp2_of_checked(Yl[32 * i]);
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
