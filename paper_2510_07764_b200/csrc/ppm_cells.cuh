// ppm_cells.cuh -- S4 + S5 of DESIGN.md: the per-(cell, phase, energy) shift-and-add kernel
// (Eq 45-47) with the atmosphere interpolation, plus the
// per-row table-slice build and the deterministic cross-chunk reduction.  Product path (sm_100a).
#pragma once
#include "ppm_common.cuh"

namespace ppm {

constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52: (x + kMagic) rounds x to the nearest integer

struct CellArgs {
    const StarD* stars; const SpotD* spots; const RowD* rows; const int* cells;
    const double* tmpl;      // [rows][4][n_fp+1]
    const double* slices;    // [rows][nmu][nx]  (table emission)
    const double* axmu;      // [nmu]
    const double* ue;        // [nE]: log10(E_e) / h   (h = logx spacing)
    const double* le2;       // [nE]: -log2(E_e)
    const double* en;        // [nE]: E_e (keV)
    double* partial;         // [nb][nchunk][n_phase][nE]
    unsigned long long* pairs;   // counter: (cell, phase) pairs with F_p != 0 (energy tile 0 only)
    double x0_over_h, inv_h;
    int nb, RT, n_spots, n_theta, n_phi, n_phase, n_fp, nE;
    int nmu, nx, mu_rule, x_linedge;
    int nchunk, rows_per_chunk, nw, n_etile;
};

// ---- K4: collapse the 4-D table to the row's (mu x logx) slice: T is per spot, g per row -------
struct SliceArgs {
    const SpotD* spots; const RowD* rows; const double* values; double* slices;
    int n_theta, nT, ng, nmu, nx;
};

__global__ void __launch_bounds__(256) k_slice(SliceArgs A)
{
    const int rid = blockIdx.y;
    const RowD& r = A.rows[rid];
    if (r.n_active == 0 || !r.visible) return;
    const SpotD& sp = A.spots[rid / A.n_theta];
    const int plane = A.nmu * A.nx;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= plane) return;
    double v = 0.0;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const double wa = sp.wT[a];
        if (wa == 0.0) continue;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double wb = r.wg[b];
            if (wb == 0.0) continue;
            v = fma(wa * wb, __ldg(A.values + ((size_t)(sp.bT + a) * A.ng + (r.bg + b)) * plane + i), v);
        }
    }
    A.slices[(size_t)rid * plane + i] = v;
}

// 2^f on [-0.5, 0.5]: Taylor series of exp(f ln 2) to degree 12 (truncation < 2e-16 relative)
__device__ __forceinline__ double exp2_poly(double f)
{
    // c_n = (ln 2)^n / n!
    double p = 2.567843599348820514199e-11;                 // n = 12
    p = fma(p, f, 4.445538271870811497596e-10);             // 11
    p = fma(p, f, 7.054911620801123329875e-9);              // 10
    p = fma(p, f, 1.017808600923969972749e-7);              // 9
    p = fma(p, f, 1.321548679014430948840e-6);              // 8
    p = fma(p, f, 1.525273380405984028003e-5);              // 7
    p = fma(p, f, 1.540353039338160995443e-4);              // 6
    p = fma(p, f, 1.333355814642844342341e-3);              // 5
    p = fma(p, f, 9.618129107628477161980e-3);              // 4
    p = fma(p, f, 5.550410866482157995314e-2);              // 3
    p = fma(p, f, 2.402265069591007123336e-1);              // 2
    p = fma(p, f, 6.931471805599453094172e-1);              // 1
    p = fma(p, f, 1.0);
    return p;
}

// 2^y for any y: round, polynomial, exponent add (integer pipe).  y < -1000 -> 0.
__device__ __forceinline__ double exp2_fast(double y)
{
    const double r = y + kMagic;
    const int n = __double2loint(r);
    const double f = y - (r - kMagic);
    const double p = exp2_poly(f);
    const int hi = __double2hiint(p) + n * 1048576;
    const int lo = __double2loint(p);
    return (n < -1000) ? 0.0 : __hiloint2double(hi, lo);
}

// ------------------------------------------------------------------------------------------------
// K5: shift-and-add.  Block = (row chunk, group of `nw` consecutive output phases, vector x energy
// tile); warp w owns output phase k and the 32*EPL energies of the tile (lane owns energies
// e0+lane+32 i): the (k, e) accumulators live in registers for the whole chunk -- output-stationary,
// no atomics.  Per row the (mu x logx) slice and the ring template sit in shared memory.  Lanes first
// prepare 32 (cell, k) pairs in parallel (Eq 45-46, mu stencil), then the warp walks the valid pairs:
// contract the mu stencil into a 1-D vector over logx (shared by all energies of the pair), then each
// lane interpolates in logx and accumulates F_p I / E (Eq 47) as one exp2.
// MODE 0: closed-form isotropic blackbody (Eq C.5); MODE 1: table.
// ------------------------------------------------------------------------------------------------
template <int EPL, int MODE>
__global__ void __launch_bounds__(512, 1) k_cells(CellArgs A)
{
    extern __shared__ __align__(16) double sm[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int chunk = blockIdx.x, pg = blockIdx.y;
    const int b = blockIdx.z / A.n_etile, et = blockIdx.z % A.n_etile;
    const int k = pg * A.nw + w;
    const bool kvalid = k < A.n_phase;
    const int e0 = et * 32 * EPL;
    const int n1 = A.n_fp + 1;
    const int plane = (MODE == 1) ? A.nmu * A.nx : 0;
    double* S = sm;                                  // [nmu][nx]
    double* T = sm + plane;                          // F, z, phi_o, mu: [4][n1]
    double* MUAX = T + 4 * n1;                       // [nmu]
    double* CV = MUAX + ((MODE == 1) ? A.nmu : 0) + (size_t)w * A.nx;   // per-warp contracted vector [nx]

    double ue[EPL], c2[EPL], acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) {
        const int e = e0 + lane + 32 * i;
        const bool ok = e < A.nE;
        if (MODE == 1) {
            ue[i] = A.ue[ok ? e : A.nE - 1];
            c2[i] = ok ? A.le2[e] : -5000.0;
        } else {
            ue[i] = ok ? A.en[e] : 1.0;              // E_e
            c2[i] = ok ? 1.0 : 0.0;
        }
        acc[i] = 0.0;
    }
    const int e_last = imin_(e0 + 32 * EPL, A.nE) - 1;
    const double ue_first = (MODE == 1) ? A.ue[imin_(e0, A.nE - 1)] : 0.0;
    const double ue_last = (MODE == 1) ? A.ue[e_last] : 0.0;
    if (MODE == 1) for (int i = threadIdx.x; i < A.nmu; i += blockDim.x) MUAX[i] = A.axmu[i];

    const StarD& st = A.stars[b];
    const double phi_off = st.phi_off;
    const double phi_out = (double)k / A.n_phase;                               // reading R3
    unsigned npairs = 0;

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
            // ---- step A: lane <-> cell; Eq 45-46 and the per-pair constants ----
            const int idx = base + lane;
            double Fp = 0.0, pa = 0.0, pb = 0.0;      // MODE 1: pa = uz, pb = lf;  MODE 0: pa = z_p, pb = F_p z_p^3 K
            double w0 = 0.0, w1 = 0.0, w2 = 0.0, w3 = 0.0;
            int mb = 0;
            if (idx < nact) {
                const int m = cl[idx];
                const double dphi_m = -sp.W + ((double)m + 0.5) * sp.dphi;
                const double phi_m = sp.phi_c + dphi_m;
                const double s0 = phi_out + phi_m / (2.0 * kPi) + phi_off + 1.0 - po0;
                const double phi_p = (s0 - floor(s0)) + po0;                    // Eq 45
                int lo = 0, hi = A.n_fp;
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (PO[mid] <= phi_p) lo = mid; else hi = mid;
                }
                const double t = (phi_p - PO[lo]) / (PO[lo + 1] - PO[lo]);
                Fp = F[lo] + (F[lo + 1] - F[lo]) * t;                           // Eq 46, linear (reading R11)
                const double zp = Z[lo] + (Z[lo + 1] - Z[lo]) * t;
                const double mup = MU[lo] + (MU[lo + 1] - MU[lo]) * t;
                if (Fp != 0.0) {
                    if (MODE == 1) {
                        pa = (log10(zp) - sp.log10kT) * A.inv_h - A.x0_over_h - 0.5;   // u - 0.5 = (x - x0)/h - 0.5, less the energy part
                        pb = log2(Fp) + sp.log2T3;
                        double ww[4];
                        axis_w4(MUAX, A.nmu, mup, A.mu_rule, mb, ww);
                        w0 = ww[0]; w1 = ww[1]; w2 = ww[2]; w3 = ww[3];
                    } else {
                        pa = zp / sp.kT;
                        pb = Fp * (2.0 / (kH_keV_s * kH_keV_s * kH_keV_s * kC_cm_s * kC_cm_s)) * zp * zp * zp;
                    }
                }
            }
            unsigned todo = __ballot_sync(0xffffffffu, Fp != 0.0);
            npairs += __popc(todo);
            // ---- step B: walk the valid pairs ----
            while (todo) {
                const int j = __ffs(todo) - 1;
                todo &= todo - 1;
                const double qa = __shfl_sync(0xffffffffu, pa, j);
                const double qb = __shfl_sync(0xffffffffu, pb, j);
                if (MODE == 0) {
#pragma unroll
                    for (int i = 0; i < EPL; ++i) {
                        const double E = ue[i];
                        acc[i] += c2[i] * (qb * E * E / expm1(qa * E));         // F_p I(z_p E)/E, Eq 47 with Eq C.5
                    }
                    continue;
                }
                const double v0 = __shfl_sync(0xffffffffu, w0, j);
                const double v1 = __shfl_sync(0xffffffffu, w1, j);
                const double v2 = __shfl_sync(0xffffffffu, w2, j);
                const double v3 = __shfl_sync(0xffffffffu, w3, j);
                const int sb = __shfl_sync(0xffffffffu, mb, j);
                // column range of logx touched by this pair's energies
                const double ulo = qa + ue_first + 0.5, uhi = qa + ue_last + 0.5;
                const bool fast = (ulo >= 1.5) && (uhi < (double)A.nx - 2.5);
                const int jlo = imin_(imax_((int)floor(fmin(fmax(ulo, 0.0), (double)A.nx)) - 2, 0), A.nx - 4);
                const int jhi = imin_(imax_((int)floor(fmin(fmax(uhi, 0.0), (double)A.nx)) + 2, 3), A.nx - 1);
                const double* s0p = S + (size_t)sb * A.nx;
                __syncwarp();
                for (int c = jlo + lane; c <= jhi; c += 32)
                    CV[c] = fma(v3, s0p[3 * A.nx + c], fma(v2, s0p[2 * A.nx + c], fma(v1, s0p[A.nx + c], v0 * s0p[c])));
                __syncwarp();
                if (fast) {
#pragma unroll
                    for (int i = 0; i < EPL; ++i) {
                        const double uu = qa + ue[i];                           // (x - x0)/h - 0.5
                        const double r = uu + kMagic;
                        const int ii = __double2loint(r);                       // interval index, x in [x_ii, x_ii+1]
                        const double tau = uu - (r - kMagic);                   // offset from the interval midpoint
                        const double c0 = CV[ii - 1], c1 = CV[ii], c2v = CV[ii + 1], c3 = CV[ii + 2];
                        // cubic Lagrange on nodes at -1.5, -0.5, 0.5, 1.5 (uniform logx axis)
                        const double a = tau * tau;
                        const double A6 = fma(a, 1.0 / 6.0, -1.0 / 24.0);
                        const double B2 = fma(a, 0.5, -1.125);
                        const double e1 = fma(tau, c3 - c0, 1.5 * (c3 + c0));
                        const double e2 = fma(tau, c1 - c2v, -0.5 * (c1 + c2v));
                        const double p = fma(A6, e1, B2 * e2);
                        acc[i] += exp2_fast(fma(p, kLog2_10, qb) + c2[i]);      // F_p T^3 10^v / E
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < EPL; ++i) {
                        double uq = qa + ue[i] + 0.5;                           // (x - x0)/h, clamped (reading R13b)
                        uq = fmin(fmax(uq, 0.0), (double)(A.nx - 1));
                        const int ii = imin_((int)uq, A.nx - 2);
                        double p;
                        if (A.x_linedge && (ii == 0 || ii == A.nx - 2)) {      // strategy d: linear edge intervals
                            const double t = uq - (double)ii;
                            p = (1.0 - t) * CV[ii] + t * CV[ii + 1];
                        } else {                                                // interior, or shifted stencil (strategy a)
                            const int s = imin_(imax_(ii - 1, 0), A.nx - 4);
                            const double g = uq - (double)s;                    // in [0, 3]
                            const double g1 = g - 1.0, g2 = g - 2.0, g3 = g - 3.0;
                            p = (-1.0 / 6.0) * (g1 * g2 * g3) * CV[s] + 0.5 * (g * g2 * g3) * CV[s + 1]
                              - 0.5 * (g * g1 * g3) * CV[s + 2] + (1.0 / 6.0) * (g * g1 * g2) * CV[s + 3];
                        }
                        acc[i] += exp2_fast(fma(p, kLog2_10, qb) + c2[i]);
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
            if (e < A.nE) out[e] = acc[i];
        }
    }
}

// ---- K6: F_t[b][k][e] = sum over chunks, fixed order (deterministic); NaN for rejected vectors ----
__global__ void __launch_bounds__(256) k_reduce(const double* __restrict__ partial, const StarD* __restrict__ stars,
                                                int nchunk, int n_out, double* __restrict__ flux, int* status)
{
    const int b = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int stt = stars[b].status;
    if (i == 0 && status) status[b] = stt;
    if (i >= n_out) return;
    double s = 0.0;
    if (stt) s = nan("");
    else {
        const double* p = partial + (size_t)b * nchunk * n_out + i;
        for (int c = 0; c < nchunk; ++c) s += p[(size_t)c * n_out];
    }
    flux[(size_t)b * n_out + i] = s;
}

}  // namespace ppm
