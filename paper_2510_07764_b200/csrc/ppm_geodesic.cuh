// ppm_geodesic.cuh -- S0..S3 of DESIGN.md: star / spot / row scalars, cell mask, the device-built
// psi / lag lookup (per-row Chebyshev series in the emission angle alpha at the row's compactness u)
// and the ring templates.  Product path (CUDA, sm_100a).
#pragma once
#include "ppm_common.cuh"

namespace ppm {

__constant__ double c_glx[kNGL];   // Gauss-Legendre nodes on [-1, 1]
__constant__ double c_glw[kNGL];   // weights

// ------------------------------------------------------------------------------------------------
// Schwarzschild integrals in the regularised variable x = sqrt(1 - R/r) (Eq 32-35;
// the garbled Eq 32 is read with D = cos^2(alpha) + x^2 q, reading R5):
//   I1 = Int_0^1 x dx / sqrt(D)                 psi = 2 sin(a)/sqrt(1-u) I1          (Eq 12 / 32)
//   I2 = Int_0^1 x dx / (sqrt(D) (1+sqrt(D)))   c dt_p/R = 2 sin^2(a)/(1-u) I2       (Eq 15 / 35)
//   q  = [2 - x^2 - u (1-x^2)^2/(1-u)] sin^2(a)                                      (Eq 33)
// The integrand has a layer of width |cos a|/sqrt(q(0)) at x = 0, so [0,1] is cut dyadically
// (1/2, 1/4, ...) down to that width and every piece gets one 16-point Gauss-Legendre panel: on each
// panel the nearest complex singularity is >= one panel width away, which makes the rule converge to
// round-off (S2).
// ------------------------------------------------------------------------------------------------
// Cooperative form: a group of kNGL = 16 adjacent lanes integrates one (u, alpha); lane g of the group owns
// Gauss-Legendre point g of every panel, the group sums by xor-shuffles after the panel loop (all 32 lanes of
// the warp must call these functions together; the two groups of a warp may run different panel counts).
__device__ inline void geo_integrals(double u, double sa, double cabs, int g, double& I1, double& I2)
{
    const double k = u / (1.0 - u), sa2 = sa * sa, ca2 = cabs * cabs;
    const double q0 = (2.0 - k) * sa2;
    // width of the layer at x = 0 where D turns from cos^2(alpha) into x^2 q.  At the periastron call (cos(alpha) = 0
    // exactly) there is no layer: x / sqrt(D) = 1 / sqrt(q) is smooth on [0, 1] (nearest zero of q at |x| >= 0.6 i for
    // u <= 0.56) and four dyadic panels resolve it to round-off.
    const double layer = (cabs == 0.0) ? 0.0625 : ((q0 > 0.0) ? cabs / sqrt(q0) : 1.0);
    const double gx = c_glx[g], gw = c_glw[g];
    double s1 = 0.0, s2 = 0.0;
    double hi = 1.0;
    bool last = false;
    for (int p = 0; p <= kMaxPanels && !last; ++p) {
        last = (p == kMaxPanels) || !(hi > layer);
        const double lo = last ? 0.0 : 0.5 * hi;                 // dyadic panels [hi/2, hi], then [0, hi]
        const double hm = 0.5 * (hi - lo), c = 0.5 * (lo + hi);
        const double x = fma(hm, gx, c);
        const double x2 = x * x, om = 1.0 - x2;
        const double q = (2.0 - x2 - k * om * om) * sa2;
        const double sD = sqrt(fma(x2, q, ca2));
        const double t = hm * gw * x / sD;
        s1 += t;
        s2 += t / (1.0 + sD);
        hi = lo;
    }
#pragma unroll
    for (int m = kNGL / 2; m > 0; m >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, m);
        s2 += __shfl_xor_sync(0xffffffffu, s2, m);
    }
    I1 = s1; I2 = s2;
}

// psi(u, alpha) and lag(u, alpha) = (c Delta t - c delta t(R)) / R for 0 < alpha < pi.
// Outgoing rays: Eq 12 / 15.  Inward rays (alpha > pi/2): Eq 13-14 and Eq 17
// read dimensionally (reading R6), everything divided by R:
//   psi = 2 psi(u/rho, pi/2) - psi(u, pi - alpha)
//   lag = 2 rho G(u/rho, pi/2) - G(u, pi - alpha) + 2 [1 - rho + u ln((1-u)/(rho-u))]
__device__ inline void geo_psi_lag(double u, double alpha, int g, double& psi, double& lag)
{
    double sa, ca;
    sincos(alpha, &sa, &ca);
    double I1, I2;
    geo_integrals(u, sa, fabs(ca), g, I1, I2);
    const double psi_o = 2.0 * sa / sqrt(1.0 - u) * I1;
    const double G_o = 2.0 * sa * sa / (1.0 - u) * I2;
    const bool inward = alpha > 0.5 * kPi;
    // the periastron integrals are needed by inward rays only; the call is warp-uniform (outgoing groups of a warp
    // that holds an inward ray discard theirs)
    const double s3 = sqrt(3.0 * (1.0 - u));
    const double arg = fmin(3.0 * u * s3 / (2.0 * sa), 1.0);
    const double rho = inward ? -2.0 * sa / s3 * cos((acos(arg) + 2.0 * kPi) / 3.0) : 1.0;      // Eq 14
    const double up = u / rho;
    double J1 = 0.0, J2 = 0.0;
    if (__any_sync(0xffffffffu, inward)) geo_integrals(up, 1.0, 0.0, g, J1, J2);
    if (!inward) { psi = psi_o; lag = G_o; return; }
    const double psi_p = 2.0 / sqrt(1.0 - up) * J1;
    const double G_p = 2.0 / (1.0 - up) * J2;
    psi = 2.0 * psi_p - psi_o;
    lag = 2.0 * rho * G_p - G_o + 2.0 * (1.0 - rho + u * log((1.0 - u) / (rho - u)));
}

// Chebyshev series f(s) = c0/2 + sum_{n>=1} c_n T_n(s): value and derivative by Clenshaw.
__device__ inline void cheb_eval(const double* __restrict__ c, double s, double& f, double& df)
{
    double b1 = 0.0, b2 = 0.0, d1 = 0.0, d2 = 0.0;
    const double s2 = 2.0 * s;
#pragma unroll 4
    for (int n = kNCheb - 1; n >= 1; --n) {
        const double d0 = fma(s2, d1, 2.0 * b1) - d2;
        const double b0 = fma(s2, b1, c[n]) - b2;
        d2 = d1; d1 = d0;
        b2 = b1; b1 = b0;
    }
    f = fma(s, b1, 0.5 * c[0]) - b2;
    df = fma(s, d1, b1) - d2;
}

// ------------------------------------------------------------------------------------------------
// K0: per vector -- star scalars (Eq 7-8, 11), domain check (reading R4), per-spot box and T stencil.
// ------------------------------------------------------------------------------------------------
// rule of the log T and log g axes per emission mode (strategies a, d, c; readings R13c, R13e)
__host__ __device__ inline int tg_rule(int emission)
{
    return (emission == PPM_EMISSION_TABLE_CUBIC || emission == PPM_EMISSION_TABLE_CUBIC_CLIP) ? AX_CUBIC_SHIFT
         : emission == PPM_EMISSION_TABLE_CUBIC_LINEDGE ? AX_CUBIC_LINEDGE : AX_LINEAR;
}

struct GeoArgs {
    const double* params;   // [nb][P]
    int nb, P, n_spots, n_theta, n_phi, n_phase, n_fp, oblate, emission, mesh;
    StarD* stars; SpotD* spots; RowD* rows; int* cells;
    double* lookup;         // [rows][2][kNCheb]: H = psi/alpha, lag
    double* tmpl;           // [rows][4][n_fp+1]
    const double* axT; int nT; const double* axg; int ng;
    const double* tmap;     // [rows][n_phi] log10 T per cell, NaN = not emitting (temperature-map mode), or nullptr
};

__global__ void k_star(GeoArgs A)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= A.nb) return;
    const double* p = A.params + (size_t)b * A.P;
    StarD s;
    int status = 0;
    for (int i = 0; i < A.P; ++i) if (!isfinite(p[i])) status |= PPM_STATUS_INPUT;
    const double M = p[0], Re_km = p[1], nu = p[2], cosi = p[3], Dkpc = p[4];
    if (!status && !(M > 0.0 && Re_km > 0.0 && nu >= 0.0 && cosi >= -1.0 && cosi <= 1.0 && Dkpc > 0.0))
        status |= PPM_STATUS_INPUT;
    const double GM = M * kGMsun, Re_m = Re_km * 1.0e3;
    s.Rs = 2.0 * GM / (kC_m_s * kC_m_s) * 100.0;
    s.Re = Re_m * 100.0;
    s.x = GM / (kC_m_s * kC_m_s * Re_m);
    const double Om = 2.0 * kPi * nu;
    s.Ob2 = Om * Om * Re_m * Re_m * Re_m / GM;
    s.o2 = A.oblate ? s.Ob2 * (-0.788 + 1.030 * s.x) : 0.0;
    s.g0 = GM / (Re_m * Re_m) / sqrt(1.0 - s.Rs / s.Re) * 100.0;
    s.nu = nu; s.cosi = cosi; s.sini = sqrt(fmax(1.0 - cosi * cosi, 0.0));
    s.D = Dkpc * 1.0e3 * kPc_cm;
    s.phi_off = p[6];
    if (!status) {
        const double Rpole = s.Re * (1.0 + s.o2);
        const double u_pole = s.Rs / Rpole, u_eq = s.Rs / s.Re;
        const double um = fmax(u_pole, u_eq);
        if (!(um > 0.0 && um <= kUmax) || !(Rpole > 0.0)) status |= PPM_STATUS_COMPACTNESS;
        else {
            const double beq = 2.0 * kPi * nu * s.Re / (kC_cm_s * sqrt(1.0 - u_eq));
            if (!(beq < 1.0)) status |= PPM_STATUS_INPUT;
        }
        for (int j = 0; j < A.n_spots; ++j) {
            const double* q = p + 8 + 8 * j;
            if (!(q[2] > 0.0 && q[2] <= kPi && q[0] >= 0.0 && q[0] <= kPi && q[6] >= 0.0 && q[6] <= kPi &&
                  q[4] >= 0.0 && q[4] <= kPi))
                status |= PPM_STATUS_SPOT;
        }
    }
    s.status = status; s.pad = 0;
    A.stars[b] = s;
    for (int j = 0; j < A.n_spots; ++j) {
        const double* q = p + 8 + 8 * j;
        SpotD sp;
        sp.theta_c = q[0]; sp.phi_c = q[1]; sp.zeta = q[2]; sp.log10T = q[3];
        sp.theta_m = q[4]; sp.phi_m = q[5]; sp.zeta_m = q[6];
        sp.theta_lo = fmax(0.0, sp.theta_c - sp.zeta);
        sp.theta_hi = fmin(kPi, sp.theta_c + sp.zeta);
        const bool polar = (sp.theta_c <= sp.zeta) || (sp.theta_c >= kPi - sp.zeta) || (sp.zeta >= 0.5 * kPi);
        sp.W = polar ? kPi : asin(sin(sp.zeta) / sin(sp.theta_c));
        sp.dphi = 2.0 * sp.W / A.n_phi;
        sp.cos_tc = cos(sp.theta_c); sp.sin_tc = sin(sp.theta_c); sp.cos_z = cos(sp.zeta);
        sp.cos_tm = cos(sp.theta_m); sp.sin_tm = sin(sp.theta_m); sp.cos_zm = cos(sp.zeta_m);
        sp.log10kT = log10(kKB_keV_K) + sp.log10T;
        sp.kT = kKB_keV_K * pow(10.0, sp.log10T);
        sp.log2T3 = 3.0 * sp.log10T * kLog2_10;
        sp.bT = 0; sp.pad = 0;
        sp.wT[0] = sp.wT[1] = sp.wT[2] = sp.wT[3] = 0.0;
        if (A.emission != PPM_EMISSION_BLACKBODY && !status)
            axis_w4(A.axT, A.nT, sp.log10T, tg_rule(A.emission),
                    sp.bT, sp.wT);
        A.spots[(size_t)b * A.n_spots + j] = sp;
    }
}

// ------------------------------------------------------------------------------------------------
// K1: one block per (vector, spot, row): row scalars (S0; Eq 2-3, 7, 10, 16, 18) and the compacted
// list of active azimuth cells (S1; PAPER.md:259 centre within zeta, PAPER.md:571 omitted region).
// The mask test uses separately rounded multiplies and adds (no FMA contraction) so that the
// inequality is decided in the same arithmetic as a plain C evaluation of the same expression.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_rows(GeoArgs A)
{
    __shared__ RowD row;
    __shared__ int warp_cnt[4];
    __shared__ int base_s;
    __shared__ unsigned long long tmask_s;
    __shared__ double tlo_s[4], thi_s[4];
    const int rid = blockIdx.x;                          // (b * n_spots + s) * n_theta + j
    const int j = rid % A.n_theta, bs = rid / A.n_theta, b = bs / A.n_spots;
    const StarD st = A.stars[b];
    const SpotD sp = A.spots[bs];
    if (threadIdx.x == 0) {
        RowD r;
        double th;
        r.npix = A.n_phi; r.phi0 = 0.0; r.dphi = sp.dphi;
        if (A.mesh == 1) {
            // HEALPix ring i = j + 1 of N_side = n_phi / 4 (Eq 24-29); pixel area pi / (3 N_side^2)
            const int nside = A.n_phi / 4, i = j + 1;
            const bool south = i > 2 * nside;
            const int in = south ? 4 * nside - i : i;
            double z;
            if (in < nside) {                                                      // Eq 24-25
                z = 1.0 - (double)in * (double)in / (3.0 * (double)nside * (double)nside);
                r.npix = 4 * in;
                r.dphi = kPi / (2.0 * (double)in);
                r.phi0 = r.dphi * 0.5;
            } else {                                                               // Eq 26-27
                z = 4.0 / 3.0 - 2.0 * (double)in / (3.0 * (double)nside);
                r.npix = 4 * nside;
                r.dphi = kPi / (2.0 * (double)nside);
                r.phi0 = r.dphi * (1.0 - 0.5 * (double)((in - nside + 1) % 2));
            }
            th = acos(south ? -z : z);                                             // Eq 28
            r.dOmega = kPi / (3.0 * (double)nside * (double)nside);
            r.dcos = r.dOmega / r.dphi;
        } else {
            const double e0 = sp.theta_lo + (sp.theta_hi - sp.theta_lo) * (double)j / A.n_theta;
            const double e1 = sp.theta_lo + (sp.theta_hi - sp.theta_lo) * (double)(j + 1) / A.n_theta;
            th = 0.5 * (e0 + e1);
            r.dcos = cos(e0) - cos(e1);
            r.dOmega = r.dcos * sp.dphi;
        }
        r.theta = th;
        const double ct = cos(th), sth = sin(th);
        const double R = st.Re * (1.0 + st.o2 * ct * ct);                         // Eq 7
        const double u = st.Rs / R;
        const double dR = -2.0 * st.Re * st.o2 * sth * ct;
        const double f = dR / (R * sqrt(1.0 - u));                                 // Eq 2
        r.R = R; r.u = u; r.f = f;
        r.coseta = 1.0 / sqrt(1.0 + f * f);                                        // Eq 3
        r.sineta = f / sqrt(1.0 + f * f);
        r.beta = 2.0 * kPi * st.nu * R * sth / (kC_cm_s * sqrt(1.0 - u));          // Eq 18
        r.gamma = 1.0 / sqrt(1.0 - r.beta * r.beta);
        double gr = 1.0;                                                           // Eq 10 (sphere: 1, reading R20)
        if (A.oblate) {
            const double O2 = st.Ob2, O4 = O2 * O2, O6 = O4 * O2, x = st.x;
            const double e = O4 * (13.47 * x - 27.13 * x * x);
            gr = 1.0 + sth * sth * (O2 * (-0.791 + 0.776 * x) + O4 * (-1.315 * x + 2.431 * x * x) + O6 * (-1.172 * x))
               + ct * ct * (O2 * (1.138 - 1.431 * x) + O4 * (0.653 * x - 2.864 * x * x) + O6 * (0.975 * x) - e)
               + fabs(ct) * e;
        }
        r.log10g = log10(st.g0 * gr);
        r.c_dt = st.Re - R + st.Rs * log((st.Re - st.Rs) / (R - st.Rs));           // Eq 16
        r.alpha_max = 0.5 * kPi + fabs(atan(f));                                   // visible rays: alpha <= pi/2 + |eta|
        r.psi_max = 0.0;
        r.bg = 0; r.wg[0] = r.wg[1] = r.wg[2] = r.wg[3] = 0.0;
        if (A.emission != PPM_EMISSION_BLACKBODY && !st.status)
            axis_w4(A.axg, A.ng, r.log10g, tg_rule(A.emission),
                    r.bg, r.wg);
        r.n_active = 0; r.visible = 0; r.tmask = 0ull; r.tmin = r.tmax = r.zlo = r.zhi = 0.0;
        row = r;
        base_s = 0;
        tmask_s = 0ull;
    }
    __syncthreads();
    int* cl = A.cells + (size_t)rid * A.n_phi;
    const double ct = cos(row.theta), sth = sin(row.theta);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double tlo = INFINITY, thi = -INFINITY;
    for (int m0 = 0; m0 < A.n_phi; m0 += blockDim.x) {
        const int m = m0 + threadIdx.x;
        bool act = false;
        int entry = m;                                            // temperature-map mode: m | (log T interval << 16)
        if (m < row.npix && !st.status) {
            const double dphi_m = (A.mesh == 1) ? __dadd_rn(__dadd_rn(row.phi0, __dmul_rn((double)m, row.dphi)), -sp.phi_c)
                                                : __dadd_rn(-sp.W, __dmul_rn((double)m + 0.5, sp.dphi));
            const double cd = __dadd_rn(__dmul_rn(ct, sp.cos_tc), __dmul_rn(__dmul_rn(sth, sp.sin_tc), cos(dphi_m)));
            act = (cd >= sp.cos_z);
            if (act && sp.zeta_m > 0.0) {
                const double phi_m = __dadd_rn(sp.phi_c, dphi_m);
                const double cm = __dadd_rn(__dmul_rn(ct, sp.cos_tm),
                                            __dmul_rn(__dmul_rn(sth, sp.sin_tm), cos(__dadd_rn(phi_m, -sp.phi_m))));
                if (cm >= sp.cos_zm) act = false;
            }
            if (act && A.tmap) {                                  // temperature map: NaN cells do not emit (reading R24)
                const double lT = A.tmap[(size_t)rid * A.n_phi + m];
                act = isfinite(lT);
                if (act) {
                    double t;
                    const int iT = axis_linear(A.axT, A.nT, lT, t);
                    atomicOr(&tmask_s, 1ull << iT);
                    entry = m | (iT << 16);
                    tlo = fmin(tlo, lT); thi = fmax(thi, lT);
                }
            }
        }
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (lane == 0) warp_cnt[w] = __popc(bal);
        __syncthreads();
        int off = base_s;
        for (int ww = 0; ww < w; ++ww) off += warp_cnt[ww];
        if (act) cl[off + __popc(bal & ((1u << lane) - 1u))] = entry;
        __syncthreads();
        if (threadIdx.x == 0) base_s += warp_cnt[0] + warp_cnt[1] + warp_cnt[2] + warp_cnt[3];
        __syncthreads();
    }
#pragma unroll
    for (int q = 16; q > 0; q >>= 1) {
        tlo = fmin(tlo, __shfl_xor_sync(0xffffffffu, tlo, q));
        thi = fmax(thi, __shfl_xor_sync(0xffffffffu, thi, q));
    }
    if (lane == 0) { tlo_s[w] = tlo; thi_s[w] = thi; }
    __syncthreads();
    if (A.tmap && tmask_s) {
        // temperature-map mode: stable sort of the row's list by log T interval (ordered compaction per interval through
        // a shared-memory copy), so that k_cells_map finds the cells of each interval in one contiguous, ordered range
        extern __shared__ int tmp_cells[];
        const int n = base_s;
        for (int i = threadIdx.x; i < n; i += blockDim.x) tmp_cells[i] = cl[i];
        if (threadIdx.x == 0) base_s = 0;
        __syncthreads();
        for (unsigned long long tm = tmask_s; tm; tm &= tm - 1) {
            const int it = __ffsll((long long)tm) - 1;
            for (int i0 = 0; i0 < n; i0 += blockDim.x) {
                const int i = i0 + threadIdx.x;
                const bool take = (i < n) && ((tmp_cells[i] >> 16) == it);
                const unsigned bal = __ballot_sync(0xffffffffu, take);
                if (lane == 0) warp_cnt[w] = __popc(bal);
                __syncthreads();
                int off = base_s;
                for (int ww = 0; ww < w; ++ww) off += warp_cnt[ww];
                if (take) cl[off + __popc(bal & ((1u << lane) - 1u))] = tmp_cells[i];
                __syncthreads();
                if (threadIdx.x == 0) base_s += warp_cnt[0] + warp_cnt[1] + warp_cnt[2] + warp_cnt[3];
                __syncthreads();
            }
        }
    }
    if (threadIdx.x == 0) {
        row.n_active = base_s;
        row.tmask = tmask_s;
        row.tmin = fmin(fmin(tlo_s[0], tlo_s[1]), fmin(tlo_s[2], tlo_s[3]));
        row.tmax = fmax(fmax(thi_s[0], thi_s[1]), fmax(thi_s[2], thi_s[3]));
        A.rows[rid] = row;
    }
}

// ------------------------------------------------------------------------------------------------
// K2 (S2): device-built lookup.  One block of kNCheb threads per row; thread j integrates psi and the
// lag at the Chebyshev-Gauss node alpha_j of [0, alpha_max]; the block then turns the samples of
// H(alpha) = psi/alpha (even and smooth, keeps relative accuracy as alpha -> 0) and of the lag into
// Chebyshev coefficients.  u is constant along a row, so the table is 1-D in the emission angle and
// indexed by the row (= compactness).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kNCheb * kNGL) k_lookup(GeoArgs A)
{
    __shared__ double fH[kNCheb], fG[kNCheb], ctab[4 * kNCheb];
    const int rid = blockIdx.x;
    const RowD r = A.rows[rid];
    if (r.n_active == 0) return;
    const int j = threadIdx.x / kNGL, g = threadIdx.x % kNGL;    // Chebyshev node, Gauss-Legendre point
    const double s = cospi((2.0 * j + 1.0) / (2.0 * kNCheb));
    const double alpha = 0.5 * r.alpha_max * (1.0 + s);
    double psi, lag;
    geo_psi_lag(r.u, alpha, g, psi, lag);
    if (g == 0) { fH[j] = psi / alpha; fG[j] = lag; }
    if (threadIdx.x >= kNCheb * kNGL - 32) {                     // last warp (its own nodes, alpha -> 0, are the cheapest):
                                                                 // psi at the largest visible emission angle
        double pm, lm;
        geo_psi_lag(r.u, r.alpha_max, g, pm, lm);
        if (threadIdx.x == kNCheb * kNGL - 32) A.rows[rid].psi_max = pm;
    }
    if (threadIdx.x < 4 * kNCheb) ctab[threadIdx.x] = cospi((double)threadIdx.x / (2.0 * kNCheb));   // cos(pi m / 128), m < 256
    __syncthreads();
    if (threadIdx.x < 2 * kNCheb) {                              // DCT: 64 coefficients of H and of the lag
        const int jj = threadIdx.x % kNCheb;
        const double* fv = (threadIdx.x < kNCheb) ? fH : fG;
        double cc = 0.0;
        for (int i = 0; i < kNCheb; ++i) cc = fma(fv[i], ctab[(jj * (2 * i + 1)) & (4 * kNCheb - 1)], cc);
        A.lookup[(size_t)rid * 2 * kNCheb + threadIdx.x] = cc * (2.0 / kNCheb);
    }
}

// evaluate a row's lookup at given emission angles (ppm_debug_lookup)
__global__ void k_lookup_eval(const double* __restrict__ L, double alpha_max, const double* __restrict__ alpha, int n,
                              double* psi, double* dpsi, double* lag)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double a = alpha[i], s = 2.0 * a / alpha_max - 1.0;
    double h, dh, g, dg;
    cheb_eval(L, s, h, dh);
    cheb_eval(L + kNCheb, s, g, dg);
    psi[i] = a * h;
    dpsi[i] = fma(a * dh, 2.0 / alpha_max, h);
    lag[i] = g;
}

// ------------------------------------------------------------------------------------------------
// K3 (S3): ring template of one row (Eq 38-44), one block per row.
// Dynamic shared memory: 2*kNCheb coefficients + 4*(n_fp+1) template entries.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_template(GeoArgs A)
{
    extern __shared__ double sm[];
    __shared__ int inv_min, inv_max, vis0;
    const int rid = blockIdx.x;
    const RowD r = A.rows[rid];
    if (r.n_active == 0) return;
    const int bs = rid / A.n_theta, b = bs / A.n_spots;
    const StarD st = A.stars[b];
    const int nfp = A.n_fp, n1 = nfp + 1;
    double* cH = sm;
    double* cG = sm + kNCheb;
    double* F = sm + 2 * kNCheb;
    double* Z = F + n1;
    double* PO = Z + n1;
    double* MU = PO + n1;
    for (int i = threadIdx.x; i < 2 * kNCheb; i += blockDim.x) sm[i] = A.lookup[(size_t)rid * 2 * kNCheb + i];
    if (threadIdx.x == 0) { inv_min = nfp; inv_max = 0; vis0 = 0; }   // step 1, once per ring (reading R9)
    __syncthreads();
    const double u = r.u, sq1mu = sqrt(1.0 - u);
    const double sth = sin(r.theta), ct = cos(r.theta);
    const double inv_amax2 = 2.0 / r.alpha_max;
    for (int i = threadIdx.x; i < nfp; i += blockDim.x) {
        const double phi = 2.0 * kPi * (double)i / nfp;
        double sphi, cphi;
        sincos(phi, &sphi, &cphi);
        double cpsi = st.sini * sth * cphi + st.cosi * ct;                      // step 2
        cpsi = fmin(fmax(cpsi, -1.0), 1.0);
        const double psi = acos(cpsi), spsi = sin(psi);
        bool visible = (psi <= r.psi_max);                                       // alpha <= pi/2 + |eta| (Eq 4)
        double Fv = 0.0, zv = 0.0, pov = 0.0, muv = 0.0;
        if (visible) {
            // step 3: invert psi = alpha H(alpha) on the row's lookup by Newton from Beloborodov's guess
            double al = acos(fmin(fmax(1.0 - (1.0 - cpsi) * (1.0 - u), -1.0), 1.0));
            al = fmin(al, r.alpha_max);
            double h = 0.0, dh = 0.0, dpsi = 1.0;
            for (int it = 0; it < 12; ++it) {
                cheb_eval(cH, al * inv_amax2 - 1.0, h, dh);
                dpsi = fma(al * dh, inv_amax2, h);
                const double step = (al * h - psi) / dpsi;
                al = fmin(fmax(al - step, 0.0), r.alpha_max);
                if (fabs(step) <= 4.0e-16 * al) break;
            }
            cheb_eval(cH, al * inv_amax2 - 1.0, h, dh);
            dpsi = fma(al * dh, inv_amax2, h);
            double sa, ca;
            sincos(al, &sa, &ca);
            double LF, cossig, cosxi;
            if (spsi < 1.0e-14) {                                                // sub-observer point (reading R7)
                LF = 1.0 - u; cossig = ca * r.coseta; cosxi = 0.0;
            } else {
                LF = sa / (spsi * dpsi);                                         // d cos(alpha) / d cos(psi)
                cossig = ca * r.coseta + sa * r.sineta / spsi * (st.cosi * sth - st.sini * ct * cphi);   // Eq 39
                cosxi = -sa * st.sini * sphi / spsi;                             // Table 2
            }
            if (cossig < 0.0) visible = false;                                   // step 5
            else {
                const double delta = 1.0 / (r.gamma * (1.0 - r.beta * cosxi));   // Eq 19
                double g, dg;
                cheb_eval(cG, al * inv_amax2 - 1.0, g, dg);
                const double dt = (r.R * g + r.c_dt) / kC_cm_s;                  // PAPER.md:201, Eq 17
                Fv = sq1mu * delta * delta * delta * (delta * cossig) * LF * r.gamma * r.R * r.R *
                     sqrt(1.0 + r.f * r.f) * r.dOmega / (st.D * st.D);           // Eq 40
                zv = 1.0 / (delta * sq1mu);
                pov = phi / (2.0 * kPi) + st.nu * dt;
                muv = delta * cossig;
            }
        }
        if (!visible) { atomicMin(&inv_min, i); atomicMax(&inv_max, i); }
        else if (i == 0) vis0 = 1;
        F[i] = Fv; Z[i] = zv; PO[i] = pov; MU[i] = muv;
    }
    __syncthreads();
    const int visible_ring = vis0;
    if (visible_ring) {
        if (threadIdx.x == 0) { F[nfp] = F[0]; Z[nfp] = Z[0]; MU[nfp] = MU[0]; PO[nfp] = PO[0] + 1.0; }   // reading R2
        __syncthreads();
        if (inv_min <= inv_max) {                                                // Eq 41-44
            const int a = inv_min - 1, bb = inv_max + 1;
            const double za = Z[a], zb = Z[bb], pa = PO[a], pb = PO[bb];
            __syncthreads();
            for (int i = inv_min + threadIdx.x; i <= inv_max; i += blockDim.x) {
                const double t = ((double)i - a) / ((double)bb - a);
                F[i] = 0.0; MU[i] = 0.0;
                Z[i] = za + (zb - za) * t;
                PO[i] = pa + (pb - pa) * t;
            }
        }
    } else {
        for (int i = threadIdx.x; i < 4 * n1; i += blockDim.x) F[i] = 0.0;
    }
    __syncthreads();
    double* out = A.tmpl + (size_t)rid * 4 * n1;
    for (int i = threadIdx.x; i < 4 * n1; i += blockDim.x) out[i] = F[i];
    // range of z over the fine phases (after the fill): bounds every z_p of Eq 46; used to size logx windows
    __shared__ double zlo_s[4], zhi_s[4];
    double zlo = INFINITY, zhi = -INFINITY;
    if (visible_ring)
        for (int i = threadIdx.x; i < n1; i += blockDim.x) { zlo = fmin(zlo, Z[i]); zhi = fmax(zhi, Z[i]); }
#pragma unroll
    for (int q = 16; q > 0; q >>= 1) {
        zlo = fmin(zlo, __shfl_xor_sync(0xffffffffu, zlo, q));
        zhi = fmax(zhi, __shfl_xor_sync(0xffffffffu, zhi, q));
    }
    if ((threadIdx.x & 31) == 0) { zlo_s[threadIdx.x >> 5] = zlo; zhi_s[threadIdx.x >> 5] = zhi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        A.rows[rid].visible = visible_ring;
        A.rows[rid].zlo = fmin(fmin(zlo_s[0], zlo_s[1]), fmin(zlo_s[2], zlo_s[3]));
        A.rows[rid].zhi = fmax(fmax(zhi_s[0], zhi_s[1]), fmax(zhi_s[2], zhi_s[3]));
    }
}

}  // namespace ppm
