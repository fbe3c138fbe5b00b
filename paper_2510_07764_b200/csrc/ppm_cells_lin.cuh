// ppm_cells_lin.cuh -- S4 + S5 with the table interpolation applied to the INTENSITY I/T^3 = 10^table (interp_domain = 1,
// reading R13g) instead of its logarithm: the form in which the paper's interpolation-strategy study observes negative
// intensities under uniform cubic interpolation (strategy a), zero "holes" after clipping (strategy b) and clean
// profiles with boundary linearisation (strategies c, d) -- PAPER.md:492-561, SURVEY.md 8(f)2.  Product path (sm_100a).
//
// Same ownership, step A, fixed-point logx coordinate and fused pass as k_cells_tab (ppm_cells.cuh).  What differs:
//   * the row slice holds sum_T sum_g w_T w_g 10^table (k_slice with domain = 1);
//   * the mu stencil weights carry F_p T^3 (everything is linear in the node values), no logarithm, no exponential;
//   * a triple is the cubic in tau itself (3 DFMA), clipped at 0 for strategy b, with the coordinate clamped to the
//     table (reading R13b).
#pragma once
#include "ppm_cells.cuh"

namespace ppm {

template <int EPL, int NPL>
__global__ void __launch_bounds__(512, 1) k_cells_lin(CellArgs A)
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
    const int plane = A.nmu * nx;
    constexpr int KW = 32 * NPL;
    constexpr int WARP_DBL = 4 * KW + 3 * 64 + 32;                              // k_cells_tab's layout
    double* wbase = sm + (size_t)w * WARP_DBL;
    double2* KA = reinterpret_cast<double2*>(wbase);
    double2* R0 = KA + 2 * KW;
    double2* R1 = R0 + 32;
    double2* R2 = R1 + 32;
    int2* RI = reinterpret_cast<int2*>(R2 + 32);
    double* S = sm + (size_t)A.nw * WARP_DBL;
    double* T = S + plane;
    double* MUAX = T + 4 * n1;

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
    for (int i = threadIdx.x; i < A.nmu; i += blockDim.x) MUAX[i] = A.axmu[i];

    const StarD& st = A.stars[b];
    const double phi_off = st.phi_off;
    const double phi_out = (double)k / A.n_phase;                               // reading R3
    const bool clip = A.clip != 0;
    unsigned npairs = 0;

    for (int ri = 0; ri < A.rows_per_chunk; ++ri) {
        const int rl = chunk + ri * A.nchunk;
        if (rl >= A.RT) break;
        const int rid = b * A.RT + rl;
        const RowD& row = A.rows[rid];
        const int nact = row.n_active;
        if (nact == 0 || !row.visible) continue;
        const SpotD& sp = A.spots[rid / A.n_theta];
        const double Tt = exp10(sp.log10T), T3 = Tt * Tt * Tt;
        __syncthreads();
        {
            const double* src = A.slices + (size_t)rid * plane;
            for (int i = threadIdx.x; i < plane; i += blockDim.x) S[i] = src[i];
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
            // ---- step A ----
            const int idx = base + lane;
            double Fp = 0.0, pb = 0.0;
            long long pq = 0;
            double ww[4] = {0.0, 0.0, 0.0, 0.0};
            int info = 0, flags = 0;
            if (idx < nact) {
                const double phi_p = phase_of_cell(phi_out, cell_azimuth(A.mesh, row, sp, cl[idx]), phi_off, po0);   // Eq 45
                double zp, mup;
                template_interp(F, Z, PO, MU, A.n_fp, A.phase_order, phi_p, Fp, zp, mup);                            // Eq 46
                if (!(Fp > 0.0)) Fp = 0.0;
                if (Fp != 0.0) {
                    pair_table_record(Fp, zp, mup, sp.log10kT, 0.0, MUAX, A.nmu, A.mu_rule, nx, A.inv_h, A.x0_over_h, uef_first,
                                      uef_last, s_top, 0.0, 0.0, pq, pb, ww, info, flags);
                    const double scale = Fp * T3 * (1.0 / kLog2_10);             // F_p T^3 (the record's weights carry log2(10))
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) ww[q4] *= scale;
                }
            }
            const unsigned valid = __ballot_sync(0xffffffffu, Fp != 0.0);
            const int cnt = __popc(valid);
            npairs += cnt;
            __syncwarp();
            if (Fp != 0.0) {
                const int slot = __popc(valid & ((1u << lane) - 1u));
                R0[slot] = make_double2(__longlong_as_double(pq), 0.0);
                R1[slot] = make_double2(ww[0], ww[1]);
                R2[slot] = make_double2(ww[2], ww[3]);
                RI[slot] = make_int2(info, flags);
            }
            __syncwarp();
            // ---- step B ----
            for (int pj = 0; pj < cnt; ++pj) {
                const double2 r0 = R0[pj], r1 = R1[pj], r2 = R2[pj];
                const int inf = RI[pj].x;
                const long long q = __double_as_longlong(r0.x);
                const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                const double* srow = S + (inf & 0xFFFF);
                const SliceNode node{srow, nx, r1.x, r1.y, r2.x, r2.y, 0.0};
                fused_pass<NPL>(node, nx, jlo, jhi, lane, A.x_linedge, KA, sm);
                const double2* KAq = KA + (1 - jlo);
#pragma unroll
                for (int i = 0; i < EPL; ++i) {
                    long long s = q + uef[i];
                    s = s < 0 ? 0 : (s > s_top ? s_top : s);                     // clamp to the table (reading R13b)
                    const int shi = (int)(s >> 32);
                    const double2* kp = KAq + (shi >> 20);
                    const double tau = __hiloint2double(one_plus_frac_hi(shi), (int)s);   // t = 1 + fraction (see cubic_coeffs)
                    const double2 c01 = kp[0], c23 = kp[KW];
                    double v = fma(fma(fma(c23.y, tau, c23.x), tau, c01.y), tau, c01.x);   // F_p T^3 * (I/T^3)
                    if (clip) v = fmax(v, 0.0);                                  // strategy b
                    acc[i] += v;
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
