// ppm_common.cuh -- constants, device-side records and small helpers shared by the PPM kernels.
// Product path (CUDA, sm_100a).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>

namespace ppm {

// ---- reading R0: CODATA-2019 exact SI values, IAU nominal GM_sun; work in cm, s, keV ----------
constexpr double kC_m_s    = 299792458.0;
constexpr double kC_cm_s   = 29979245800.0;
constexpr double kH_keV_s  = 6.62607015e-34 / 1.602176634e-19 / 1.0e3;
constexpr double kKB_keV_K = 1.380649e-23 / 1.602176634e-19 / 1.0e3;
constexpr double kGMsun    = 1.32712440018e20;      // m^3 s^-2
constexpr double kPc_cm    = 3.0856775814913673e18;
constexpr double kPi       = 3.14159265358979323846;
constexpr double kUmax     = 0.560;                 // supported compactness domain (reading R4)
constexpr double kLog2_10  = 3.32192809488736234787;

constexpr int kNCheb = 64;     // Chebyshev nodes per row of the psi / lag lookup (S2)
constexpr int kNGL   = 16;     // Gauss-Legendre points per quadrature panel
constexpr int kMaxPanels = 48; // dyadic panels towards x = 0

// per-axis interpolation rules (readings R13b-d)
enum AxisRule { AX_LINEAR = 0, AX_CUBIC_SHIFT = 1, AX_CUBIC_LINEDGE = 2, AX_MU_PROTECTED = 3 };

struct StarD {
    double Rs, Re;        // Schwarzschild / equatorial radius [cm]
    double x, Ob2, o2;    // Eq 7-8
    double g0;            // Eq 11 [cm s^-2]
    double nu, cosi, sini, D, phi_off;
    int status, pad;
};

struct SpotD {
    double theta_c, phi_c, zeta, log10T, theta_m, phi_m, zeta_m;
    double theta_lo, theta_hi, W, dphi;           // bounding box (reading R1)
    double cos_tc, sin_tc, cos_z, cos_tm, sin_tm, cos_zm;
    double log10kT, log2T3, kT;
    double wT[4];                                 // log T axis stencil weights (zeros when linear)
    int bT, pad;
};

struct RowD {
    double theta, dcos, R, u, f, coseta, sineta, beta, gamma, log10g, c_dt, dOmega;
    double alpha_max, psi_max;
    double wg[4];                                 // log g axis stencil
    int bg, n_active, visible, npix;              // npix: azimuth cells of this row (HEALPix rings differ)
    double phi0, dphi;                            // azimuth of cell m: phi0 + m dphi (HEALPix mesh only)
    unsigned long long tmask;                     // temperature-map mode: bit i set iff an active cell lies in log T interval i
    double tmin, tmax;                            // temperature-map mode: range of log10 T over the row's emitting cells
    double zlo, zhi;                              // range of the template's redshift factor z over the fine phases
};

__host__ __device__ inline int imin_(int a, int b) { return a < b ? a : b; }
__host__ __device__ inline int imax_(int a, int b) { return a > b ? a : b; }

// Stencil of up to four consecutive nodes ax[base..base+3] with Lagrange weights on the actual
// abscissae (reading R13d); linear rules put their two weights inside the same 4-wide window.
// x is clamped to the axis range first (reading R13b).  Requires n >= 4.
__device__ inline void axis_w4(const double* __restrict__ ax, int n, double x, int rule, int& base, double w[4])
{
    x = fmin(fmax(x, ax[0]), ax[n - 1]);
    int lo = 0, hi = n - 1;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (ax[mid] <= x) lo = mid; else hi = mid;
    }
    const int i = imin_(lo, n - 2);
    bool linear;
    switch (rule) {
    case AX_LINEAR:        linear = true; break;
    case AX_CUBIC_SHIFT:   linear = false; break;
    case AX_CUBIC_LINEDGE: linear = (i == 0 || i == n - 2); break;
    default:               linear = (i < 3 || i == n - 2); break;   // protected small-mu zone
    }
    const int s = imin_(imax_(i - 1, 0), n - 4);
    base = s;
    if (linear) {
        const double t = (x - ax[i]) / (ax[i + 1] - ax[i]);
        const int o = i - s;                                   // 0, 1 or 2
        const double a = 1.0 - t;
        w[0] = (o == 0) ? a : 0.0;
        w[1] = (o == 0) ? t : ((o == 1) ? a : 0.0);
        w[2] = (o == 1) ? t : ((o == 2) ? a : 0.0);
        w[3] = (o == 2) ? t : 0.0;
        return;
    }
    const double x0 = ax[s], x1 = ax[s + 1], x2 = ax[s + 2], x3 = ax[s + 3];
    const double d0 = x - x0, d1 = x - x1, d2 = x - x2, d3 = x - x3;
    w[0] = (d1 * d2 * d3) / ((x0 - x1) * (x0 - x2) * (x0 - x3));
    w[1] = (d0 * d2 * d3) / ((x1 - x0) * (x1 - x2) * (x1 - x3));
    w[2] = (d0 * d1 * d3) / ((x2 - x0) * (x2 - x1) * (x2 - x3));
    w[3] = (d0 * d1 * d2) / ((x3 - x0) * (x3 - x1) * (x3 - x2));
}

// Linear rule on one axis (the log T axis of a temperature map): x clamped to the axis (reading R13b), interval i with
// ax[i] <= x <= ax[i+1], t = (x - ax[i]) / (ax[i+1] - ax[i]) -- the arithmetic of axis_w4's AX_LINEAR branch.
__device__ inline int axis_linear(const double* __restrict__ ax, int n, double x, double& t)
{
    x = fmin(fmax(x, ax[0]), ax[n - 1]);
    int lo = 0, hi = n - 1;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (ax[mid] <= x) lo = mid; else hi = mid;
    }
    const int i = imin_(lo, n - 2);
    t = (x - ax[i]) / (ax[i + 1] - ax[i]);
    return i;
}

}  // namespace ppm
