/*
 * ppm_oracle.c -- CPU ORACLE for the OS+D pulse-profile forward model of
 * arxiv/paper_2510_07764 (Zhou & Huang, "GPU-accelerated X-ray pulse profile modeling").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may build, link or call it.  It
 * shares no code, header, table or constant generator with the CUDA path under
 * paper_2510_07764_b200/csrc/ and neither includes the other.
 *
 * It is a plain, slow, step-by-step restatement of the paper's "computation recipe"
 * (section 2.8) with ONE deliberate difference fixed by the task's
 * north_star: the light-bending angle psi(u,alpha), the lensing factor
 * d cos(alpha)/d cos(psi) and the time lag are obtained by DIRECT NUMERICAL QUADRATURE
 * of the Schwarzschild integrals at every template point (no lookup table).
 * Everything else follows the paper in the paper's order and notation; the places
 * where the paper is silent / garbled follow the readings R0..R22 of DESIGN.md.
 *
 * Arithmetic: IEEE double everywhere, long double inside the quadrature / root solve.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1..P20 of DESIGN.md (P17-P20, tests/test_oracle_rotation.py: the
 * rotation / aberration terms of the template against a moving blackbody in flat space and against unit vectors,
 * the Eq 41-44 fill, Eq 10's Obar^6 terms).  Parts that have
 * no pin other than internal consistency are listed under "parity unpinned" there:
 *   - absolute agreement with the external NICER-grade benchmarks (OS1a-l, Ring/Crescent)
 *     -- PARITY UNPINNED (reference data not available).
 *
 * Units: lengths in cm, time in s, photon energy in keV, T in K.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

/* ------------------------------------------------------------------------------------
 * O0  Constants (paper silent -> reading R0: CODATA-2019 exact SI values, IAU GM_sun).
 * ---------------------------------------------------------------------------------- */
#define ORC_C_M_S      299792458.0            /* m/s  */
#define ORC_H_J_S      6.62607015e-34         /* J s  */
#define ORC_KB_J_K     1.380649e-23           /* J/K  */
#define ORC_E_C        1.602176634e-19        /* C    */
#define ORC_GMSUN      1.32712440018e20       /* m^3/s^2 */
#define ORC_PC_M       3.0856775814913673e16  /* m    */

static const ld ORC_PIl = 3.14159265358979323846264338327950288L;

double orc_const(int which)
{
    switch (which) {
    case 0: return ORC_C_M_S * 100.0;                       /* c  [cm/s]      */
    case 1: return ORC_H_J_S / ORC_E_C / 1.0e3;             /* h  [keV s]     */
    case 2: return ORC_KB_J_K / ORC_E_C / 1.0e3;            /* k_B [keV/K]    */
    case 3: return ORC_GMSUN;                               /* GM_sun [m^3/s^2] */
    case 4: return ORC_PC_M * 100.0;                        /* pc [cm]        */
    case 5: {                                               /* 2/(h^3 c^2) [keV^-3 cm^-2 s^-1] */
        double h = ORC_H_J_S / ORC_E_C / 1.0e3, c = ORC_C_M_S * 100.0;
        return 2.0 / (h * h * h * c * c);
    }
    default: return NAN;
    }
}

/* ------------------------------------------------------------------------------------
 * Quadrature: n-point Gauss-Legendre panels (nodes from Newton iteration on P_n) with
 * plain recursive bisection until |whole - (left+right)| is below tolerance.
 * ---------------------------------------------------------------------------------- */
#define ORC_NGL 15
static ld gl_x[ORC_NGL], gl_w[ORC_NGL];

__attribute__((constructor)) static void gl_init(void)
{
    const int n = ORC_NGL;
    for (int i = 0; i < n; ++i) {
        ld x = cosl(ORC_PIl * ((ld)i + 0.75L) / ((ld)n + 0.5L));
        ld dp = 1.0L;
        for (int it = 0; it < 100; ++it) {
            ld p0 = 1.0L, p1 = x;                 /* Legendre recurrence */
            for (int k = 2; k <= n; ++k) {
                ld p2 = (((ld)(2 * k - 1)) * x * p1 - ((ld)(k - 1)) * p0) / (ld)k;
                p0 = p1; p1 = p2;
            }
            dp = (ld)n * (x * p1 - p0) / (x * x - 1.0L);
            ld dx = p1 / dp;
            x -= dx;
            if (fabsl(dx) < 1e-20L) break;
        }
        /* recompute derivative at the converged node */
        ld p0 = 1.0L, p1 = x;
        for (int k = 2; k <= n; ++k) {
            ld p2 = (((ld)(2 * k - 1)) * x * p1 - ((ld)(k - 1)) * p0) / (ld)k;
            p0 = p1; p1 = p2;
        }
        dp = (ld)n * (x * p1 - p0) / (x * x - 1.0L);
        gl_x[i] = x;
        gl_w[i] = 2.0L / ((1.0L - x * x) * dp * dp);
    }
}

/* exposed so a test can check the rule itself (weights sum to 2, exact on polynomials) */
void orc_gl_rule(int* n, double* x, double* w)
{
    *n = ORC_NGL;
    for (int i = 0; i < ORC_NGL; ++i) { x[i] = (double)gl_x[i]; w[i] = (double)gl_w[i]; }
}

typedef ld (*orc_fn)(ld x, const void* ctx);

static ld gl_panel(orc_fn f, const void* ctx, ld a, ld b)
{
    ld hm = 0.5L * (b - a), c = 0.5L * (a + b), s = 0.0L;
    for (int i = 0; i < ORC_NGL; ++i) s += gl_w[i] * f(c + hm * gl_x[i], ctx);
    return s * hm;
}

static ld adapt_rec(orc_fn f, const void* ctx, ld a, ld b, ld whole, ld tol, int depth)
{
    ld m = 0.5L * (a + b);
    ld L = gl_panel(f, ctx, a, m), R = gl_panel(f, ctx, m, b);
    if (depth >= 80 || fabsl(L + R - whole) <= tol) return L + R;
    return adapt_rec(f, ctx, a, m, L, tol, depth + 1) + adapt_rec(f, ctx, m, b, R, tol, depth + 1);
}

static ld integrate_panel(orc_fn f, const void* ctx, ld a, ld b)
{
    ld whole = gl_panel(f, ctx, a, b);
    ld tol = 1e-17L * fabsl(whole) + 1e-300L;
    return adapt_rec(f, ctx, a, b, whole, tol, 0);
}

/* Integral over [0,1] of an integrand that has a boundary layer of width `layer` at x = 0
 * (the Eq 32/35 integrands vary on the scale x ~ cos(alpha)/sqrt(q(0)) there).  The interval is
 * first cut at x = 1/2, 1/4, ... down to `layer`, and every piece is integrated adaptively:
 * a single top-level panel cannot see a layer narrower than its first node and would accept
 * the layer-free value (an O(cos alpha) error for |alpha - pi/2| < ~1e-8). */
static ld integrate01(orc_fn f, const void* ctx, ld layer)
{
    ld sum = 0.0L, hi = 1.0L;
    for (int j = 0; j < 70 && hi > layer; ++j) {
        ld lo = 0.5L * hi;
        sum += integrate_panel(f, ctx, lo, hi);
        hi = lo;
    }
    return sum + integrate_panel(f, ctx, 0.0L, hi);
}

/* ------------------------------------------------------------------------------------
 * Light bending, Eq 12 in the regularised form Eq 32-33 (the garbled
 * "sqrt(cos^2 a + x^2) a" is read as sqrt(cos^2 a + x^2 q), reading R5):
 *   psi(u,alpha) = 2 sin(alpha)/sqrt(1-u) * Int_0^1 x dx / sqrt(cos^2 alpha + x^2 q)
 *   q = [2 - x^2 - u (1-x^2)^2/(1-u)] sin^2 alpha                                (alpha <= pi/2)
 * ---------------------------------------------------------------------------------- */
typedef struct { ld u, sa2, ca2, layer; } bend_ctx;

static inline ld q_of_x(ld x, const bend_ctx* c)
{
    ld x2 = x * x, om = 1.0L - x2;
    return (2.0L - x2 - c->u * om * om / (1.0L - c->u)) * c->sa2;
}
static ld f_psi(ld x, const void* p)
{
    const bend_ctx* c = (const bend_ctx*)p;
    return x / sqrtl(c->ca2 + x * x * q_of_x(x, c));
}
/* d psi / d alpha integrand (derived from Eq 32 by differentiating under the integral,
 * reading R12; valid for alpha < pi/2):  2 cos(alpha)/sqrt(1-u) Int_0^1 x dx/(cos^2 a + x^2 q)^{3/2} */
static ld f_dpsi(ld x, const void* p)
{
    const bend_ctx* c = (const bend_ctx*)p;
    ld D = c->ca2 + x * x * q_of_x(x, c);
    return x / (D * sqrtl(D));
}
/* time delay Eq 15 in the form Eq 35:
 *   c dt_p / R = 2 sin^2 a/(1-u) Int_0^1 x dx / ( sqrt(D) (1+sqrt(D)) ),  D = cos^2 a + x^2 q */
static ld f_lag(ld x, const void* p)
{
    const bend_ctx* c = (const bend_ctx*)p;
    ld sD = sqrtl(c->ca2 + x * x * q_of_x(x, c));
    return x / (sD * (1.0L + sD));
}

static void bend_ctx_set(bend_ctx* c, ld u, ld alpha)
{
    ld sa = sinl(alpha), ca = cosl(alpha);
    c->u = u; c->sa2 = sa * sa; c->ca2 = ca * ca;
    /* width of the x -> 0 layer of D = cos^2 a + x^2 q:  |cos a| / sqrt(q(0)),  q(0) = (2 - u/(1-u)) sin^2 a */
    ld q0 = (2.0L - u / (1.0L - u)) * c->sa2;
    c->layer = (q0 > 0.0L) ? fabsl(ca) / sqrtl(q0) : 1.0L;
}

static ld psi_out(ld u, ld alpha)          /* 0 <= alpha <= pi/2 */
{
    bend_ctx c; bend_ctx_set(&c, u, alpha);
    return 2.0L * sinl(alpha) / sqrtl(1.0L - u) * integrate01(f_psi, &c, c.layer);
}
static ld dpsi_out_analytic(ld u, ld alpha) /* 0 <= alpha < pi/2 */
{
    bend_ctx c; bend_ctx_set(&c, u, alpha);
    return 2.0L * cosl(alpha) / sqrtl(1.0L - u) * integrate01(f_dpsi, &c, c.layer);
}
static ld lag_out(ld u, ld alpha)          /* G(u,alpha) = c dt_p / R, 0 <= alpha <= pi/2 */
{
    bend_ctx c; bend_ctx_set(&c, u, alpha);
    return 2.0L * c.sa2 / (1.0L - u) * integrate01(f_lag, &c, c.layer);
}

/* periastron ratio rho = R_p / R for an inward ray, Eq 14 */
static ld rho_of(ld u, ld alpha)
{
    ld s3 = sqrtl(3.0L * (1.0L - u));
    ld arg = 3.0L * u * s3 / (2.0L * sinl(alpha));
    if (arg > 1.0L) arg = 1.0L;
    return -2.0L * sinl(alpha) / s3 * cosl((acosl(arg) + 2.0L * ORC_PIl) / 3.0L);
}

/* psi for any 0 <= alpha < pi:  Eq 12/32 for alpha <= pi/2, Eq 13/34 beyond */
static ld psi_any(ld u, ld alpha)
{
    const ld half_pi = 0.5L * ORC_PIl;
    if (alpha <= half_pi) return psi_out(u, alpha);
    ld rho = rho_of(u, alpha);
    return 2.0L * psi_out(u / rho, half_pi) - psi_out(u, ORC_PIl - alpha);
}

/* d psi/d alpha: analytic integral for alpha < pi/2 - 0.05; 6th-order central differences of
 * psi_any (step 1e-3) near and beyond pi/2 where the analytic form is 0 x inf (reading R12). */
static ld dpsi_any(ld u, ld alpha)
{
    const ld half_pi = 0.5L * ORC_PIl;
    if (alpha < half_pi - 0.05L) return dpsi_out_analytic(u, alpha);
    const ld h = 1.0e-3L;
    ld f1 = psi_any(u, alpha + h) - psi_any(u, alpha - h);
    ld f2 = psi_any(u, alpha + 2 * h) - psi_any(u, alpha - 2 * h);
    ld f3 = psi_any(u, alpha + 3 * h) - psi_any(u, alpha - 3 * h);
    return (45.0L * f1 - 9.0L * f2 + f3) / (60.0L * h);
}

/* c delta t(R') = R_e - R' + R_S ln((R_e-R_S)/(R'-R_S)), Eq 16; lengths in any one unit */
static ld c_delta_t(ld Re, ld Rs, ld Rp)
{
    return Re - Rp + Rs * logl((Re - Rs) / (Rp - Rs));
}

/* total c*Delta t (same length unit as R) for emission at radius R (u = Rs/R) at angle alpha,
 * relative to a radial photon from R_e:
 *   alpha <= pi/2 : R G(u,alpha) + c dt(R)
 *   alpha >  pi/2 : Eq 17 read dimensionally (reading R6):
 *                   2 R_p G(u/rho, pi/2) - R G(u, pi-alpha) + 2 c dt(R_p) - c dt(R),  R_p = rho R */
static ld c_lag_total(ld Re, ld Rs, ld R, ld alpha)
{
    const ld half_pi = 0.5L * ORC_PIl;
    ld u = Rs / R;
    if (alpha <= half_pi) return R * lag_out(u, alpha) + c_delta_t(Re, Rs, R);
    ld rho = rho_of(u, alpha), Rp = rho * R;
    return 2.0L * Rp * lag_out(u / rho, half_pi) - R * lag_out(u, ORC_PIl - alpha)
         + 2.0L * c_delta_t(Re, Rs, Rp) - c_delta_t(Re, Rs, R);
}

/* ---- thin double-precision entry points for the pins ---- */
double orc_psi(double u, double alpha)          { return (double)psi_any((ld)u, (ld)alpha); }
double orc_dpsi_dalpha(double u, double alpha)  { return (double)dpsi_any((ld)u, (ld)alpha); }
double orc_dpsi_dalpha_analytic(double u, double alpha) { return (double)dpsi_out_analytic((ld)u, (ld)alpha); }
double orc_lag(double u, double alpha)          { return (double)lag_out((ld)u, (ld)alpha); }
double orc_rho(double u, double alpha)          { return (double)rho_of((ld)u, (ld)alpha); }
/* c*Delta t / R with R_e := R (no oblate offset): what pins P6 quote */
double orc_lag_total_over_R(double u, double alpha)
{
    return (double)c_lag_total(1.0L, (ld)u, 1.0L, (ld)alpha);
}
double orc_lag_total(double Re, double Rs, double R, double alpha)
{
    return (double)c_lag_total((ld)Re, (ld)Rs, (ld)R, (ld)alpha);
}

/* Solve psi(u,alpha) = psi_t for alpha in [0, alpha_max] (psi is increasing in alpha).
 * Brent's method in long double.  Returns 0 on success, 1 if psi_t > psi(u,alpha_max). */
static int alpha_of_psi_l(ld u, ld psi_t, ld alpha_max, ld* alpha_out)
{
    if (psi_t <= 0.0L) { *alpha_out = 0.0L; return 0; }
    ld a = 0.0L, b = alpha_max;
    ld fa = -psi_t, fb = psi_any(u, b) - psi_t;
    if (fb < 0.0L) return 1;
    if (fb == 0.0L) { *alpha_out = b; return 0; }
    ld c = a, fc = fa, d = b - a, e = d;
    for (int it = 0; it < 200; ++it) {
        if ((fb > 0 && fc > 0) || (fb < 0 && fc < 0)) { c = a; fc = fa; d = e = b - a; }
        if (fabsl(fc) < fabsl(fb)) { a = b; b = c; c = a; fa = fb; fb = fc; fc = fa; }
        ld tol1 = 2.0L * 1.0e-19L * fabsl(b) + 0.5e-17L;
        ld xm = 0.5L * (c - b);
        if (fabsl(xm) <= tol1 || fb == 0.0L) break;
        if (fabsl(e) >= tol1 && fabsl(fa) > fabsl(fb)) {
            ld s = fb / fa, p, q;
            if (a == c) { p = 2.0L * xm * s; q = 1.0L - s; }
            else {
                ld qq = fa / fc, r = fb / fc;
                p = s * (2.0L * xm * qq * (qq - r) - (b - a) * (r - 1.0L));
                q = (qq - 1.0L) * (r - 1.0L) * (s - 1.0L);
            }
            if (p > 0) q = -q;
            p = fabsl(p);
            ld min1 = 3.0L * xm * q - fabsl(tol1 * q), min2 = fabsl(e * q);
            if (2.0L * p < (min1 < min2 ? min1 : min2)) { e = d; d = p / q; }
            else { d = xm; e = d; }
        } else { d = xm; e = d; }
        a = b; fa = fb;
        if (fabsl(d) > tol1) b += d; else b += (xm > 0 ? tol1 : -tol1);
        fb = psi_any(u, b) - psi_t;
    }
    *alpha_out = b;
    return 0;
}
int orc_alpha_of_psi(double u, double psi_t, double alpha_max, double* alpha)
{
    ld a; int rc = alpha_of_psi_l((ld)u, (ld)psi_t, (ld)alpha_max, &a);
    *alpha = rc ? NAN : (double)a;
    return rc;
}

/* ------------------------------------------------------------------------------------
 * O1  Star scalars  (Eq 7-8, Eq 11)
 * ---------------------------------------------------------------------------------- */
typedef struct {
    double GM;      /* m^3/s^2 */
    double Rs_cm;   /* Schwarzschild radius 2GM/c^2 */
    double Re_cm;   /* equatorial radius */
    double x;       /* GM/(c^2 R_e) */
    double Obar2;   /* (2 pi nu)^2 R_e^3 / GM */
    double o2;      /* Obar2 (-0.788 + 1.030 x); 0 in sphere mode */
    double g0_cgs;  /* GM/R_e^2 / sqrt(1 - R_S/R_e) */
    double nu;      /* Hz */
    int    oblate;
} orc_star;

void orc_star_init(double M_msun, double Re_km, double nu_hz, int oblate, orc_star* s)
{
    double GM = M_msun * ORC_GMSUN, c = ORC_C_M_S, Re_m = Re_km * 1.0e3;
    s->GM = GM;
    s->Rs_cm = 2.0 * GM / (c * c) * 100.0;
    s->Re_cm = Re_m * 100.0;
    s->x = GM / (c * c * Re_m);
    double Om = 2.0 * M_PI * nu_hz;
    s->Obar2 = Om * Om * Re_m * Re_m * Re_m / GM;
    s->o2 = oblate ? s->Obar2 * (-0.788 + 1.030 * s->x) : 0.0;
    s->g0_cgs = GM / (Re_m * Re_m) / sqrt(1.0 - s->Rs_cm / s->Re_cm) * 100.0;
    s->nu = nu_hz;
    s->oblate = oblate;
}

/* Effective gravity g(theta)/g0, Eq 10, as printed. Sphere mode: 1 (reading R20). */
static double g_ratio(const orc_star* s, double theta)
{
    if (!s->oblate) return 1.0;
    double O2 = s->Obar2, O4 = O2 * O2, O6 = O4 * O2, x = s->x;
    double st = sin(theta), ct = cos(theta);
    double e = O4 * (13.47 * x - 27.13 * x * x);
    return 1.0
        + st * st * (O2 * (-0.791 + 0.776 * x) + O4 * (-1.315 * x + 2.431 * x * x) + O6 * (-1.172 * x))
        + ct * ct * (O2 * (1.138 - 1.431 * x) + O4 * (0.653 * x - 2.864 * x * x) + O6 * (0.975 * x) - e)
        + fabs(ct) * e;
}

/* ------------------------------------------------------------------------------------
 * O2  Rows of one spot (reading R1: per-spot bounding-box grid in (theta, phi)).
 * ---------------------------------------------------------------------------------- */
typedef struct {
    double theta;     /* row-centre colatitude */
    double dcos;      /* cos(edge_j) - cos(edge_{j+1}) */
    double R_cm, u, f, coseta, sineta, beta, gamma, log10g;
    double c_dt_cm;   /* c * delta t(R), Eq 16 */
} orc_row;

typedef struct {
    double theta_c, phi_c, zeta, log10T, theta_m, phi_m, zeta_m;
} orc_spot;

typedef struct {
    double theta_lo, theta_hi, W, dphi;
} orc_box;

void orc_spot_box(const orc_spot* sp, int n_theta, int n_phi, orc_box* bx)
{
    (void)n_theta;
    bx->theta_lo = fmax(0.0, sp->theta_c - sp->zeta);
    bx->theta_hi = fmin(M_PI, sp->theta_c + sp->zeta);
    int polar = (sp->theta_c <= sp->zeta) || (sp->theta_c >= M_PI - sp->zeta) || (sp->zeta >= 0.5 * M_PI);
    bx->W = polar ? M_PI : asin(sin(sp->zeta) / sin(sp->theta_c));
    bx->dphi = 2.0 * bx->W / n_phi;
}

static void row_from_theta(const orc_star* s, double th, double dcos, orc_row* r);

void orc_row_init(const orc_star* s, const orc_box* bx, int n_theta, int j, orc_row* r)
{
    double e0 = bx->theta_lo + (bx->theta_hi - bx->theta_lo) * (double)j / n_theta;
    double e1 = bx->theta_lo + (bx->theta_hi - bx->theta_lo) * (double)(j + 1) / n_theta;
    row_from_theta(s, 0.5 * (e0 + e1), cos(e0) - cos(e1), r);
}

/* row scalars at colatitude th (Eq 2-3, 7, 10-11, 16, 18) */
static void row_from_theta(const orc_star* s, double th, double dcos, orc_row* r)
{
    r->theta = th;
    r->dcos = dcos;
    double ct = cos(th), st = sin(th);
    double R = s->Re_cm * (1.0 + s->o2 * ct * ct);               /* Eq 7 */
    double u = s->Rs_cm / R;
    double dR = -2.0 * s->Re_cm * s->o2 * st * ct;               /* dR/dtheta */
    double f = dR / (R * sqrt(1.0 - u));                         /* Eq 2 */
    r->R_cm = R; r->u = u; r->f = f;
    r->coseta = 1.0 / sqrt(1.0 + f * f);                         /* Eq 3 */
    r->sineta = f / sqrt(1.0 + f * f);
    r->beta = 2.0 * M_PI * s->nu * R * st / (ORC_C_M_S * 100.0 * sqrt(1.0 - u));  /* Eq 18 */
    r->gamma = 1.0 / sqrt(1.0 - r->beta * r->beta);
    r->log10g = log10(s->g0_cgs * g_ratio(s, th));               /* Eq 10-11 */
    r->c_dt_cm = (double)c_delta_t((ld)s->Re_cm, (ld)s->Rs_cm, (ld)R);    /* Eq 16 */
}

/* HEALPix ring scheme (Eq 24-29): ring i = 1 .. 4 N_side - 1 -> cos(theta) of its pixel centres,
 * number of pixels, azimuth of pixel i_phi = 1 and azimuth step; every pixel covers pi / (3 N_side^2) sr. */
void orc_healpix_ring(int nside, int i, double* costheta, int* npix, double* phi0, double* dphi)
{
    int south = i > 2 * nside;
    int in = south ? 4 * nside - i : i;                           /* Eq 28-29: mirror of the northern ring */
    double z;
    if (in < nside) {                                             /* Eq 24-25 */
        z = 1.0 - (double)in * (double)in / (3.0 * (double)nside * (double)nside);
        *npix = 4 * in;
        *dphi = M_PI / (2.0 * (double)in);
        *phi0 = *dphi * 0.5;
    } else {                                                      /* Eq 26-27 */
        z = 4.0 / 3.0 - 2.0 * (double)in / (3.0 * (double)nside);
        *npix = 4 * nside;
        *dphi = M_PI / (2.0 * (double)nside);
        *phi0 = *dphi * (1.0 - 0.5 * (double)((in - nside + 1) % 2));
    }
    *costheta = south ? -z : z;
}

void orc_row_init_healpix(const orc_star* s, int nside, int j, orc_row* r)
{
    double z, phi0, dphi; int npix;
    orc_healpix_ring(nside, j + 1, &z, &npix, &phi0, &dphi);
    row_from_theta(s, acos(z), M_PI / (3.0 * (double)nside * (double)nside) / dphi, r);   /* dcos := dOmega / dphi */
}

/* cell (j,m) active?  centre-in test for the cap, minus the omitted (masking) cap
 * ("angular separation <= zeta"; PAPER.md:571 masks hide the region they cover). */
static int cell_active(const orc_spot* sp, double theta_j, double dphi_m /* phi_m - phi_c */)
{
    double ct = cos(theta_j), st = sin(theta_j);
    double cd = ct * cos(sp->theta_c) + st * sin(sp->theta_c) * cos(dphi_m);
    if (!(cd >= cos(sp->zeta))) return 0;
    if (sp->zeta_m > 0.0) {
        double phi_m = sp->phi_c + dphi_m;
        double cm = ct * cos(sp->theta_m) + st * sin(sp->theta_m) * cos(phi_m - sp->phi_m);
        if (cm >= cos(sp->zeta_m)) return 0;
    }
    return 1;
}

static inline double cell_dphi(const orc_box* bx, int m)      /* phi_m - phi_c */
{
    return -bx->W + ((double)m + 0.5) * bx->dphi;
}

/* mask[n_theta][n_phi] (1 = active) for one spot; returns number of active cells */
int orc_spot_mask(const orc_spot* sp, int n_theta, int n_phi, uint8_t* mask)
{
    orc_box bx; orc_spot_box(sp, n_theta, n_phi, &bx);
    int n = 0;
    for (int j = 0; j < n_theta; ++j) {
        double e0 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * (double)j / n_theta;
        double e1 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * (double)(j + 1) / n_theta;
        double th = 0.5 * (e0 + e1);
        for (int m = 0; m < n_phi; ++m) {
            int a = cell_active(sp, th, cell_dphi(&bx, m));
            mask[(size_t)j * n_phi + m] = (uint8_t)a; n += a;
        }
    }
    return n;
}

/* Smallest distance of any cell of the spot's box grid from a mask decision boundary, min |cos(sep) - cos(zeta)| (and the
 * same for the omitted cap): a cell closer than a few ulp to a boundary is decided by the last bit of cos(), which
 * differs between math libraries -- parity tests compare such cells' masks only when this margin is comfortably large. */
double orc_spot_mask_margin(const orc_spot* sp, int n_theta, int n_phi)
{
    orc_box bx; orc_spot_box(sp, n_theta, n_phi, &bx);
    double mg = INFINITY;
    for (int j = 0; j < n_theta; ++j) {
        double e0 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * (double)j / n_theta;
        double e1 = bx.theta_lo + (bx.theta_hi - bx.theta_lo) * (double)(j + 1) / n_theta;
        double th = 0.5 * (e0 + e1), ct = cos(th), st = sin(th);
        for (int m = 0; m < n_phi; ++m) {
            double dphi_m = cell_dphi(&bx, m);
            double cd = ct * cos(sp->theta_c) + st * sin(sp->theta_c) * cos(dphi_m);
            if (fabs(cd - cos(sp->zeta)) < mg) mg = fabs(cd - cos(sp->zeta));
            if (sp->zeta_m > 0.0) {
                double cm = ct * cos(sp->theta_m) + st * sin(sp->theta_m) * cos(sp->phi_c + dphi_m - sp->phi_m);
                if (fabs(cm - cos(sp->zeta_m)) < mg) mg = fabs(cm - cos(sp->zeta_m));
            }
        }
    }
    return mg;
}

/* HEALPix mask[4 nside - 1][4 nside] (1 = active; entries beyond a ring's pixel count are 0) */
int orc_spot_mask_healpix(const orc_spot* sp, int nside, uint8_t* mask)
{
    int n = 0;
    const int n_phi = 4 * nside;
    memset(mask, 0, (size_t)(4 * nside - 1) * n_phi);
    for (int j = 0; j < 4 * nside - 1; ++j) {
        double z, phi0, dphi; int npix;
        orc_healpix_ring(nside, j + 1, &z, &npix, &phi0, &dphi);
        double th = acos(z);
        for (int m = 0; m < npix; ++m) {
            int a = cell_active(sp, th, (phi0 + (double)m * dphi) - sp->phi_c);
            mask[(size_t)j * n_phi + m] = (uint8_t)a; n += a;
        }
    }
    return n;
}

/* ------------------------------------------------------------------------------------
 * O3 + O4  Ring template of one row (Eq 38-44).
 * Arrays have n_fp+1 entries.  vis[i] (optional) = 1 visible / 0 invisible before the fill.
 * margin (optional): min over template nodes of the distance to a visibility flip,
 * min(|cos sigma|, |psi - psi_max|)  (used by generators to re-draw, reading R22).
 * Returns 1 if the ring is visible somewhere (entry 0 visible), else 0 (ring contributes 0).
 * ---------------------------------------------------------------------------------- */
int orc_template(const orc_star* s, const orc_row* r, double cosi, double D_cm, double dOmega,
                 int n_fp, double* F, double* z, double* phio, double* mu,
                 uint8_t* vis_out, double* margin_out, double* alpha_out, double* lf_out)
{
    const double u = r->u, sini = sqrt(1.0 - cosi * cosi);
    const double st = sin(r->theta), ct = cos(r->theta);
    const double sq1mu = sqrt(1.0 - u);
    const ld alpha_max = 0.5L * ORC_PIl + (ld)fabs(atan(r->f));        /* pi/2 + |eta| */
    const double psi_max = (double)psi_any((ld)u, alpha_max);
    double margin = INFINITY;
    int i_inv_min = n_fp, i_inv_max = 0;                               /* step 1 (reading R9) */
    uint8_t* vis = (uint8_t*)malloc((size_t)n_fp + 1);

    for (int i = 0; i < n_fp; ++i) {
        double phi = 2.0 * M_PI * (double)i / n_fp;
        double cphi = cos(phi), sphi = sin(phi);
        double cpsi = sini * st * cphi + cosi * ct;                    /* step 2 */
        if (cpsi > 1.0) cpsi = 1.0;
        if (cpsi < -1.0) cpsi = -1.0;
        double psi = acos(cpsi), spsi = sin(psi);
        int visible = 1;
        double alpha = 0.0, LF = 0.0, cossig = 0.0, cosxi = 0.0;
        if (fabs(psi - psi_max) < margin) margin = fabs(psi - psi_max);
        if (psi > psi_max) visible = 0;                                /* implied by Eq 4: alpha <= pi/2+|eta| */
        else {
            ld al;
            alpha_of_psi_l((ld)u, (ld)psi, alpha_max, &al);            /* step 3 by quadrature + root solve */
            alpha = (double)al;
            double sa = sin(alpha), ca = cos(alpha);
            if (spsi < 1.0e-14) {                                      /* sub-observer point (reading R7) */
                LF = 1.0 - u; cossig = ca * r->coseta; cosxi = 0.0;
            } else {
                LF = sa / (spsi * (double)dpsi_any((ld)u, al));        /* dcos(alpha)/dcos(psi) */
                cossig = ca * r->coseta + sa * r->sineta / spsi * (cosi * st - sini * ct * cphi);  /* Eq 39 */
                cosxi = -sa * sini * sphi / spsi;                      /* Table 2 */
            }
            if (fabs(cossig) < margin) margin = fabs(cossig);
            if (cossig < 0.0) visible = 0;                             /* step 5 */
        }
        vis[i] = (uint8_t)visible;
        if (alpha_out) alpha_out[i] = visible ? alpha : NAN;
        if (lf_out) lf_out[i] = visible ? LF : NAN;
        if (!visible) {
            if (i < i_inv_min) i_inv_min = i;
            if (i > i_inv_max) i_inv_max = i;
            F[i] = 0.0; z[i] = 0.0; phio[i] = 0.0; mu[i] = 0.0;
            continue;
        }
        double delta = 1.0 / (r->gamma * (1.0 - r->beta * cosxi));     /* Eq 19 */
        double c_dt = (double)c_lag_total((ld)s->Re_cm, (ld)s->Rs_cm, (ld)r->R_cm, (ld)alpha);
        double dt = c_dt / (ORC_C_M_S * 100.0);
        /* Eq 40 (cos sigma' == mu = delta cos sigma, reading R8) */
        F[i] = sq1mu * delta * delta * delta * (delta * cossig) * LF * r->gamma
             * r->R_cm * r->R_cm * sqrt(1.0 + r->f * r->f) * dOmega / (D_cm * D_cm);
        z[i] = 1.0 / (delta * sq1mu);
        phio[i] = phi / (2.0 * M_PI) + s->nu * dt;
        mu[i] = delta * cossig;
    }
    int ring_visible = vis[0];
    if (ring_visible) {
        /* periodic closure (reading R2) */
        F[n_fp] = F[0]; z[n_fp] = z[0]; mu[n_fp] = mu[0]; phio[n_fp] = phio[0] + 1.0; vis[n_fp] = 1;
        if (i_inv_min <= i_inv_max) {                                  /* O4: Eq 41-44 */
            int a = i_inv_min - 1, b = i_inv_max + 1;
            for (int i = i_inv_min; i <= i_inv_max; ++i) {
                double t = ((double)i - a) / ((double)b - a);
                F[i] = 0.0; mu[i] = 0.0;
                z[i] = z[a] + (z[b] - z[a]) * t;
                phio[i] = phio[a] + (phio[b] - phio[a]) * t;
            }
        }
    } else {
        for (int i = 0; i <= n_fp; ++i) { F[i] = 0.0; z[i] = 0.0; phio[i] = 0.0; mu[i] = 0.0; }
        vis[n_fp] = 0;
    }
    if (vis_out) memcpy(vis_out, vis, (size_t)n_fp + 1);
    if (margin_out) *margin_out = margin;
    free(vis);
    return ring_visible;
}

/* ------------------------------------------------------------------------------------
 * O6  Intensity.
 * ---------------------------------------------------------------------------------- */
typedef struct {
    int32_t nT, ng, nmu, nx;
    const double *logT, *logg, *mu, *logx;   /* strictly increasing axes */
    const double *values;                    /* log10(I/T^3), [nT][ng][nmu][nx] C order */
} orc_atm;

/* per-axis rule codes */
enum { AX_LINEAR = 0, AX_CUBIC_SHIFT = 1, AX_CUBIC_LINEDGE = 2, AX_MU_PROTECTED = 3 };

/* Lagrange weights on the actual node abscissae.  Returns base index b and count cnt (2 or 4):
 * interpolant = sum_{k<cnt} w[k] * y[b+k].   x is clamped to the axis range first (reading R13b).
 * interval i = largest i with ax[i] <= x, capped at n-2 (reading R13d). */
static void axis_weights(const double* ax, int n, double x, int rule, int* b, int* cnt, double* w)
{
    if (x < ax[0]) x = ax[0];
    if (x > ax[n - 1]) x = ax[n - 1];
    int lo = 0, hi = n - 1;                       /* invariant ax[lo] <= x, (hi==n-1 or x < ax[hi]) */
    while (hi - lo > 1) { int mid = (lo + hi) / 2; if (ax[mid] <= x) lo = mid; else hi = mid; }
    int i = lo; if (i > n - 2) i = n - 2;
    int linear;
    switch (rule) {
    case AX_LINEAR:        linear = 1; break;
    case AX_CUBIC_SHIFT:   linear = 0; break;
    case AX_CUBIC_LINEDGE: linear = (i == 0 || i == n - 2); break;
    default:               linear = (i < 3 || i == n - 2); break;   /* AX_MU_PROTECTED: mu <= mu[3] or last interval */
    }
    if (linear) {
        double t = (x - ax[i]) / (ax[i + 1] - ax[i]);
        *b = i; *cnt = 2; w[0] = 1.0 - t; w[1] = t;
        return;
    }
    int s = i - 1; if (s < 0) s = 0; if (s > n - 4) s = n - 4;
    *b = s; *cnt = 4;
    for (int k = 0; k < 4; ++k) {
        double num = 1.0, den = 1.0;
        for (int m = 0; m < 4; ++m) if (m != k) { num *= (x - ax[s + m]); den *= (ax[s + k] - ax[s + m]); }
        w[k] = num / den;
    }
}

/* exposed for the 1-D pins */
double orc_interp1(const double* ax, const double* y, int n, double x, int rule)
{
    int b, cnt; double w[4], v = 0.0;
    axis_weights(ax, n, x, rule, &b, &cnt, w);
    for (int k = 0; k < cnt; ++k) v += w[k] * y[b + k];
    return v;
}

/* strategy: 1 = (a) cubic on all four axes; 2 = (d) mixed order (reading R13c);
 * 3 = (c) cubic on all four axes with linear interpolation at the table boundaries (Fig 4 caption PAPER.md:537)
 * and in the protected small-mu zone ("linear interpolation enforced at the mu -> 0 boundary"; R13e) */
static double interp4_domain(const orc_atm* A, int strategy, int domain, double logT, double logg, double mu, double logx);

double orc_interp4(const orc_atm* A, int strategy, double logT, double logg, double mu, double logx)
{
    return interp4_domain(A, strategy, 0, logT, logg, mu, logx);
}

/* domain 0: the weighted sum runs over the tabulated log10(I/T^3) (reading R13a); domain 1: over I/T^3 = 10^table
 * (reading R13g -- the form in which a cubic stencil can return a negative intensity).
 * strategy 4 = (b): the stencils of (a); the clipping of negative intensities is applied by the caller. */
double orc_interp4_domain(const orc_atm* A, int strategy, int domain, double logT, double logg, double mu, double logx)
{
    return interp4_domain(A, strategy, domain, logT, logg, mu, logx);
}

static double interp4_domain(const orc_atm* A, int strategy, int domain, double logT, double logg, double mu, double logx)
{
    int rT, rg, rm, rx;
    if (strategy == 1 || strategy == 4) { rT = rg = rm = rx = AX_CUBIC_SHIFT; }
    else if (strategy == 3) { rT = rg = rx = AX_CUBIC_LINEDGE; rm = AX_MU_PROTECTED; }
    else { rT = rg = AX_LINEAR; rm = AX_MU_PROTECTED; rx = AX_CUBIC_LINEDGE; }
    int bT, cT, bg, cg, bm, cm, bx, cx; double wT[4], wg[4], wm[4], wx[4];
    axis_weights(A->logT, A->nT, logT, rT, &bT, &cT, wT);
    axis_weights(A->logg, A->ng, logg, rg, &bg, &cg, wg);
    axis_weights(A->mu, A->nmu, mu, rm, &bm, &cm, wm);
    axis_weights(A->logx, A->nx, logx, rx, &bx, &cx, wx);
    double v = 0.0;
    for (int a = 0; a < cT; ++a)
        for (int b = 0; b < cg; ++b)
            for (int c = 0; c < cm; ++c)
                for (int d = 0; d < cx; ++d) {
                    size_t idx = (((size_t)(bT + a) * A->ng + (bg + b)) * A->nmu + (bm + c)) * A->nx + (bx + d);
                    double node = domain ? pow(10.0, A->values[idx]) : A->values[idx];
                    v += wT[a] * wg[b] * wm[c] * wx[d] * node;
                }
    return v;
}

/* I(E', mu): emission 0 = isotropic blackbody Eq C.5; 1,2 = table,
 * I = T^3 10^v (reading R13a).  E' in keV, returns keV^0 s^-1 cm^-2 sr^-1 (per keV, times keV). */
static int g_beaming = 0;   /* blackbody beaming law: 0 isotropic; 1 prop. to cos^2(sigma'); 2 prop. to sin^2(sigma')
                             * ("simple parametric laws"; cos(sigma') = mu, reading R23) */
static int g_domain = 0;    /* table emission: 0 interpolate log10(I/T^3) (R13a); 1 interpolate I/T^3 itself (R13g) */
static double intensity(int emission, const orc_atm* A, double log10T, double log10g, double Ep, double mu)
{
    const double kB = ORC_KB_J_K / ORC_E_C / 1.0e3;
    double T = pow(10.0, log10T), kT = kB * T;
    if (emission == 0) {
        double h = ORC_H_J_S / ORC_E_C / 1.0e3, c = ORC_C_M_S * 100.0;
        double I = 2.0 / (h * h * h * c * c) * Ep * Ep * Ep / expm1(Ep / kT);
        if (g_beaming == 1) I *= mu * mu;
        else if (g_beaming == 2) I *= 1.0 - mu * mu;
        return I;
    }
    if (g_domain == 0) {
        /* strategy b clips negative intensities; 10^v > 0, so here it is strategy a (reading R13f) */
        double v = interp4_domain(A, emission, 0, log10T, log10g, mu, log10(Ep / kT));
        return T * T * T * pow(10.0, v);
    }
    double w = interp4_domain(A, emission, 1, log10T, log10g, mu, log10(Ep / kT));   /* I/T^3, may be negative */
    if (emission == 4 && w < 0.0) w = 0.0;                                           /* strategy b: clip to zero */
    return T * T * T * w;
}
double orc_intensity(int emission, const orc_atm* A, double log10T, double log10g, double Ep, double mu)
{
    return intensity(emission, A, log10T, log10g, Ep, mu);
}
double orc_intensity_domain(int emission, int domain, const orc_atm* A, double log10T, double log10g, double Ep, double mu)
{
    int keep = g_domain;
    g_domain = domain;
    double v = intensity(emission, A, log10T, log10g, Ep, mu);
    g_domain = keep;
    return v;
}

/* ------------------------------------------------------------------------------------
 * Interp of Eq 46 on the periodic template (phio strictly increasing, phio[n_fp] = phio[0] + 1).
 * order 1 (reading R11): piecewise linear on the bracket phio[i] <= phi_p < phio[i+1].
 * order 3 (reading R11b): 4-point Lagrange on the nodes {i-1, i, i+1, i+2} with the TRUE abscissae phio, wrapped
 * periodically (node -1 = node n_fp-1 one cycle earlier, node n_fp+1 = node 1 one cycle later).  Next to the
 * visibility edge F has a kink and the filled z, phio are only continuous: if any of the four F nodes is 0
 * (an invisible or filled entry, Eq 41) the bracket reverts to the linear rule -- the same "linear at the
 * boundary" safeguard the paper applies to the atmosphere table.
 * y = one of F, z, mu.  Returns the bracket index through *i_out (optional).
 * ---------------------------------------------------------------------------------- */
double orc_phase_interp(int n_fp, const double* phio, const double* F, const double* y, double phi_p, int order, int* i_out)
{
    int lo = 0, hi = n_fp;                                                       /* phio[lo] <= phi_p < phio[hi] */
    while (hi - lo > 1) { int mid = (lo + hi) / 2; if (phio[mid] <= phi_p) lo = mid; else hi = mid; }
    if (i_out) *i_out = lo;
    if (order == 3) {
        int idx[4]; double x[4], f[4], v[4];
        for (int k = 0; k < 4; ++k) {
            int j = lo - 1 + k; double shift = 0.0;
            if (j < 0) { j += n_fp; shift = -1.0; }
            if (j > n_fp) { j -= n_fp; shift = 1.0; }
            idx[k] = j; x[k] = phio[j] + shift; f[k] = F[j]; v[k] = y[j];
        }
        (void)idx;
        if (f[0] != 0.0 && f[1] != 0.0 && f[2] != 0.0 && f[3] != 0.0) {
            double r = 0.0;
            for (int k = 0; k < 4; ++k) {
                double num = 1.0, den = 1.0;
                for (int m = 0; m < 4; ++m) if (m != k) { num *= (phi_p - x[m]); den *= (x[k] - x[m]); }
                r += num / den * v[k];
            }
            return r;
        }
    }
    double t = (phi_p - phio[lo]) / (phio[lo + 1] - phio[lo]);
    return y[lo] + (y[lo + 1] - y[lo]) * t;
}

/* ------------------------------------------------------------------------------------
 * O2..O7  One evaluation:  F_t[k][e]  (photons cm^-2 s^-1 keV^-1).
 * params: [M/Msun, R_eq/km, nu/Hz, cos i, D/kpc, N_H/1e20, phase offset/cycles, reserved]
 *         + per spot [theta_c, phi_c, zeta, log10 T, theta_m, phi_m, zeta_m, reserved].
 * phase_sel (optional, n_phase_sel entries): compute only these output-phase indices
 * (row k of flux then corresponds to phase_sel[k]); NULL -> all n_phase phases.
 * Returns 0 ok; status bits as in include/ppm.h otherwise (flux filled with NaN).
 * ---------------------------------------------------------------------------------- */
typedef struct {
    int32_t n_spots, n_theta, n_phi, n_phase, n_fp, n_energy, emission, oblate;
    int32_t mesh;    /* 0: per-spot theta x phi bounding-box grid (reading R1); 1: HEALPix rings (Eq 24-29) with
                        N_side = n_phi / 4, n_theta = 4 N_side - 1, the same mesh for every spot */
    int32_t beaming; /* emission 0 only: 0 isotropic, 1 cos^2(sigma'), 2 sin^2(sigma') */
    int32_t phase_interp;  /* Interp of Eq 46: 0 / 1 linear (reading R11); 3 four-point Lagrange (reading R11b) */
    int32_t interp_domain; /* table emission: 0 interpolate log10(I/T^3) (R13a); 1 interpolate I/T^3 (R13g) */
} orc_config;

#define ORC_U_MAX 0.560     /* supported compactness domain (reading R4) */

static int check_domain(const orc_config* cfg, const double* p, const orc_star* s)
{
    int status = 0;
    for (int k = 0; k < 8 + 8 * cfg->n_spots; ++k) if (!isfinite(p[k])) status |= 2;
    if (status) return status;
    if (!(p[0] > 0 && p[1] > 0 && p[2] >= 0 && p[3] >= -1.0 && p[3] <= 1.0 && p[4] > 0)) status |= 2;
    double R_pole = s->Re_cm * (1.0 + s->o2);
    double u_pole = s->Rs_cm / R_pole, u_eq = s->Rs_cm / s->Re_cm;
    double umax = u_pole > u_eq ? u_pole : u_eq;
    if (!(umax > 0.0 && umax <= ORC_U_MAX) || !(R_pole > 0)) status |= 1;
    else {
        double beq = 2.0 * M_PI * s->nu * s->Re_cm / (ORC_C_M_S * 100.0 * sqrt(1.0 - u_eq));
        if (!(beq < 1.0)) status |= 2;
    }
    for (int sidx = 0; sidx < cfg->n_spots; ++sidx) {
        const double* q = p + 8 + 8 * sidx;
        if (!(q[2] > 0.0 && q[2] <= M_PI && q[0] >= 0.0 && q[0] <= M_PI && q[6] >= 0.0 && q[6] <= M_PI
              && q[4] >= 0.0 && q[4] <= M_PI)) status |= 4;
    }
    return status;
}

/* tmap (optional): per-cell effective temperature map log10 T[n_spots][n_theta][n_phi] ("a full
 * surface temperature map T_eff(theta, phi)"); a cell of the mesh emits iff it passes the spot's geometric mask AND
 * its map entry is finite (NaN = not emitting); the spot's own log10 T parameter is then ignored (reading R24). */
static int evaluate_impl(const orc_config* cfg, const double* energies, const double* params, const orc_atm* atm,
                         const double* tmap, const int32_t* phase_sel, int n_phase_sel, double* flux, double* margin_out)
{
    const int nk = phase_sel ? n_phase_sel : cfg->n_phase, nE = cfg->n_energy, nfp = cfg->n_fp;
    orc_star star; orc_star_init(params[0], params[1], params[2], cfg->oblate, &star);
    int status = check_domain(cfg, params, &star);
    if (status) { for (size_t i = 0; i < (size_t)nk * nE; ++i) flux[i] = NAN; return status; }
    g_beaming = cfg->emission == 0 ? cfg->beaming : 0;   /* set before the parallel region; one evaluation at a time */
    g_domain = cfg->emission != 0 ? cfg->interp_domain : 0;
    const int porder = cfg->phase_interp == 3 ? 3 : 1;
    const double cosi = params[3], D_cm = params[4] * 1.0e3 * ORC_PC_M * 100.0, phi_off = params[6];
    const double kB = ORC_KB_J_K / ORC_E_C / 1.0e3;
    (void)kB;
    memset(flux, 0, sizeof(double) * (size_t)nk * nE);
    double margin_all = INFINITY;
    const int n_rows_total = cfg->n_spots * cfg->n_theta;

#pragma omp parallel
    {
        double* acc = (double*)calloc((size_t)nk * nE, sizeof(double));
        double* F = (double*)malloc(sizeof(double) * 4 * ((size_t)nfp + 1));
        double *z = F + (nfp + 1), *po = z + (nfp + 1), *mu = po + (nfp + 1);
        double margin_thr = INFINITY;
#pragma omp for schedule(dynamic, 1)
        for (int rr = 0; rr < n_rows_total; ++rr) {
            int sidx = rr / cfg->n_theta, j = rr % cfg->n_theta;
            const double* q = params + 8 + 8 * sidx;
            orc_spot sp = { q[0], q[1], q[2], q[3], q[4], q[5], q[6] };
            orc_box bx; orc_spot_box(&sp, cfg->n_theta, cfg->n_phi, &bx);
            orc_row row;
            int npix = cfg->n_phi;
            double hp_phi0 = 0.0, hp_dphi = 0.0, dOmega;
            if (cfg->mesh == 1) {
                const int nside = cfg->n_phi / 4;
                double zc;
                orc_healpix_ring(nside, j + 1, &zc, &npix, &hp_phi0, &hp_dphi);
                orc_row_init_healpix(&star, nside, j, &row);
                dOmega = M_PI / (3.0 * (double)nside * (double)nside);
            } else {
                orc_row_init(&star, &bx, cfg->n_theta, j, &row);
                dOmega = row.dcos * bx.dphi;
            }
#define CELL_DPHI(m) (cfg->mesh == 1 ? (hp_phi0 + (double)(m) * hp_dphi) - sp.phi_c : cell_dphi(&bx, (m)))
            /* active azimuths of this ring */
            const double* trow = tmap ? tmap + ((size_t)sidx * cfg->n_theta + j) * cfg->n_phi : NULL;
#define CELL_ON(m) (cell_active(&sp, row.theta, CELL_DPHI(m)) && (!trow || isfinite(trow[(m)])))
            int n_act = 0;
            for (int m = 0; m < npix; ++m) n_act += CELL_ON(m);
            if (n_act == 0) continue;
            double mg;
            int visible = orc_template(&star, &row, cosi, D_cm, dOmega, nfp, F, z, po, mu, NULL, &mg, NULL, NULL);
            if (mg < margin_thr) margin_thr = mg;
            if (!visible) continue;
            /* O5 shift-and-add */
            for (int m = 0; m < npix; ++m) {
                double dphi_m = CELL_DPHI(m);
                if (!CELL_ON(m)) continue;
                const double cell_log10T = trow ? trow[m] : sp.log10T;
                double phi_m = sp.phi_c + dphi_m;
                for (int kk = 0; kk < nk; ++kk) {
                    int k = phase_sel ? phase_sel[kk] : kk;
                    double phi_out = (double)k / cfg->n_phase;                               /* reading R3 */
                    double s0 = phi_out + phi_m / (2.0 * M_PI) + phi_off + 1.0 - po[0];
                    double phi_p = (s0 - floor(s0)) + po[0];                                 /* Eq 45 */
                    double Fp = orc_phase_interp(nfp, po, F, F, phi_p, porder, NULL);         /* Eq 46 (R11 / R11b) */
                    double zp = orc_phase_interp(nfp, po, F, z, phi_p, porder, NULL);
                    double mup = orc_phase_interp(nfp, po, F, mu, phi_p, porder, NULL);
                    if (Fp == 0.0) continue;
                    for (int e = 0; e < nE; ++e) {
                        double E = energies[e];
                        double I = intensity(cfg->emission, atm, cell_log10T, row.log10g, zp * E, mup);
                        acc[(size_t)kk * nE + e] += Fp * I / E;                               /* Eq 47 */
                    }
                }
            }
        }
#pragma omp critical
        {
            for (size_t i = 0; i < (size_t)nk * nE; ++i) flux[i] += acc[i];
            if (margin_thr < margin_all) margin_all = margin_thr;
        }
        free(acc); free(F);
    }
    if (margin_out) *margin_out = margin_all;
    return 0;
}

int orc_evaluate(const orc_config* cfg, const double* energies, const double* params, const orc_atm* atm,
                 const int32_t* phase_sel, int n_phase_sel, double* flux, double* margin_out)
{
    return evaluate_impl(cfg, energies, params, atm, NULL, phase_sel, n_phase_sel, flux, margin_out);
}

int orc_evaluate_map(const orc_config* cfg, const double* energies, const double* params, const orc_atm* atm,
                     const double* tmap, const int32_t* phase_sel, int n_phase_sel, double* flux, double* margin_out)
{
    return evaluate_impl(cfg, energies, params, atm, tmap, phase_sel, n_phase_sel, flux, margin_out);
}

/* ------------------------------------------------------------------------------------
 * O8  ISM attenuation + banded response fold (Eq 22-23, 51, 55)
 *   C[k][c] = sum_e F_t[k][e] exp(-N_H20 tau_ref[e]) RSP0[e][c]
 * RSP0 stored banded: row e covers channels first_chan[e] .. first_chan[e]+band_w-1.
 * ---------------------------------------------------------------------------------- */
void orc_fold(const double* flux, int n_phase, int n_energy, int n_channel, int band_w,
              const int32_t* first_chan, const double* rsp_band, const double* tau_ref, double NH20,
              double* counts)
{
    memset(counts, 0, sizeof(double) * (size_t)n_phase * n_channel);
    for (int k = 0; k < n_phase; ++k)
        for (int e = 0; e < n_energy; ++e) {
            double a = flux[(size_t)k * n_energy + e] * exp(-NH20 * tau_ref[e]);
            for (int w = 0; w < band_w; ++w) {
                int c = first_chan[e] + w;
                if (c < 0 || c >= n_channel) continue;
                counts[(size_t)k * n_channel + c] += a * rsp_band[(size_t)e * band_w + w];
            }
        }
}

/* ------------------------------------------------------------------------------------
 * O9  Poisson log-likelihood (reading R14):
 *   m[k][c] = t_exp C[k][c] / N_ph + bkg[c];  lnL = sum d ln m - m - lgamma(d+1)
 *   0 ln 0 := 0;  lnL = -inf if some m = 0 < d.
 * ---------------------------------------------------------------------------------- */
double orc_loglike(const double* counts, const double* data, const double* bkg, int n_phase, int n_channel,
                   double exposure_s)
{
    double s = 0.0;
    for (int k = 0; k < n_phase; ++k)
        for (int c = 0; c < n_channel; ++c) {
            double m = exposure_s * counts[(size_t)k * n_channel + c] / n_phase + (bkg ? bkg[c] : 0.0);
            double d = data[(size_t)k * n_channel + c];
            if (d > 0.0) {
                if (!(m > 0.0)) return -INFINITY;
                s += d * log(m);
            }
            s += -m - lgamma(d + 1.0);
        }
    return s;
}

/* chi^2 mismatch statistic, Eq 56-57: K sum (m-d)^2/m, K = 1e6/sum m */
double orc_chi2(const double* m, const double* d, size_t n)
{
    double sm = 0.0, s = 0.0;
    for (size_t i = 0; i < n; ++i) sm += m[i];
    for (size_t i = 0; i < n; ++i) if (m[i] > 0.0) s += (m[i] - d[i]) * (m[i] - d[i]) / m[i];
    return 1.0e6 / sm * s;
}

/* ------------------------------------------------------------------------------------
 * O10  Reference chain for the device-resident sampler loop (PAPER.md:716 names "a fully GPU-resident
 * parallel-tempered MCMC" without giving an algorithm -> reading R26): W walkers, walker w at inverse temperature
 * beta[w]; per step (i) Gaussian random-walk proposal p' = p + sigma * n inside a box prior [lo, hi] (outside: rejected),
 * (ii) Metropolis accept iff ln u < beta_w (lnL' - lnL), (iii) replica exchange between the neighbours (i, i+1) with
 * i = t mod 2, t mod 2 + 2, ...: swap iff ln u < (beta_i - beta_{i+1}) (lnL_{i+1} - lnL_i).
 * All random numbers come from the counter-based generator Philox4x32-10 (Salmon et al. 2011) keyed by the seed, with the
 * counter (t low, t high, walker, stream): streams 0..P/2 -> proposal normals of parameters (2 s, 2 s + 1) by Box-Muller,
 * 0x10000 -> accept uniform, 0x10001 -> swap uniform of the pair starting at `walker`.
 * ---------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 53-bit uniform in (0, 1) from two 32-bit words */
static double u01(uint32_t a, uint32_t b)
{
    uint64_t m = ((uint64_t)(a >> 5) << 26) | (uint64_t)(b >> 6);
    return ((double)m + 0.5) * (1.0 / 9007199254740992.0);
}

/* two uniforms (u0, u1) and the two Box-Muller normals (n0, n1) of counter (t, walker, stream) */
void orc_chain_random(uint64_t seed, uint64_t t, uint32_t walker, uint32_t stream, double* u0, double* u1, double* n0, double* n1)
{
    uint32_t ctr[4] = { (uint32_t)t, (uint32_t)(t >> 32), walker, stream };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, x[4];
    orc_philox4x32_10(ctr, key, x);
    double a = u01(x[0], x[1]), b = u01(x[2], x[3]);
    double r = sqrt(-2.0 * log(a));
    *u0 = a; *u1 = b; *n0 = r * cos(2.0 * M_PI * b); *n1 = r * sin(2.0 * M_PI * b);
}

/* ln L of one parameter vector: O2-O9 in sequence (evaluate, fold, Poisson likelihood); -inf outside the model's domain */
static double chain_loglike(const orc_config* cfg, const double* energies, const orc_atm* atm, const double* p,
                            int n_channel, int band_w, const int32_t* first_chan, const double* rsp_band,
                            const double* tau_ref, const double* data, const double* bkg, double exposure_s,
                            double* flux, double* counts)
{
    if (orc_evaluate(cfg, energies, p, atm, NULL, 0, flux, NULL) != 0) return -INFINITY;
    orc_fold(flux, cfg->n_phase, cfg->n_energy, n_channel, band_w, first_chan, rsp_band, tau_ref, p[5], counts);
    return orc_loglike(counts, data, bkg, cfg->n_phase, n_channel, exposure_s);
}

/* Runs n_steps of the chain in place.  params [W][P], loglike [W] (in: ln L of params; out: updated), accepted [W],
 * swapped [W] (exchanges that moved a new state into slot w).  t0 = index of the first step.  margin (optional): the
 * smallest |ln u - log acceptance ratio| met, so that a test can tell a robust decision from a coin flip. */
void orc_chain_run(const orc_config* cfg, const double* energies, const orc_atm* atm, int n_channel, int band_w,
                   const int32_t* first_chan, const double* rsp_band, const double* tau_ref, const double* data,
                   const double* bkg, double exposure_s, int W, const double* lo, const double* hi, const double* sigma,
                   const double* beta, uint64_t seed, uint64_t t0, int n_steps, double* params, double* loglike,
                   int64_t* accepted, int64_t* swapped, double* margin)
{
    const int P = 8 + 8 * cfg->n_spots;
    double* prop = (double*)malloc(sizeof(double) * P);
    double* flux = (double*)malloc(sizeof(double) * (size_t)cfg->n_phase * cfg->n_energy);
    double* counts = (double*)malloc(sizeof(double) * (size_t)cfg->n_phase * n_channel);
    double mg = INFINITY;
    for (int st = 0; st < n_steps; ++st) {
        const uint64_t t = t0 + (uint64_t)st;
        for (int w = 0; w < W; ++w) {
            double* cur = params + (size_t)w * P;
            int inside = 1;
            for (int k = 0; k < P; ++k) {
                prop[k] = cur[k];
                if (sigma[k] > 0.0) {
                    double u0, u1, n0, n1;
                    orc_chain_random(seed, t, (uint32_t)w, (uint32_t)(k / 2), &u0, &u1, &n0, &n1);
                    prop[k] = cur[k] + sigma[k] * ((k & 1) ? n1 : n0);
                    if (!(prop[k] >= lo[k] && prop[k] <= hi[k])) inside = 0;
                }
            }
            if (!inside) continue;                                       /* zero prior: rejected without evaluation */
            double lp = chain_loglike(cfg, energies, atm, prop, n_channel, band_w, first_chan, rsp_band, tau_ref, data, bkg,
                                      exposure_s, flux, counts);
            double u0, u1, n0, n1;
            orc_chain_random(seed, t, (uint32_t)w, 0x10000u, &u0, &u1, &n0, &n1);
            double ratio = beta[w] * (lp - loglike[w]);
            if (isfinite(lp) && fabs(log(u0) - ratio) < mg) mg = fabs(log(u0) - ratio);
            if (isfinite(lp) && log(u0) < ratio) {
                memcpy(cur, prop, sizeof(double) * P);
                loglike[w] = lp;
                accepted[w] += 1;
            }
        }
        for (int i = (int)(t & 1); i + 1 < W; i += 2) {                  /* replica exchange, reading R26 (iii) */
            double u0, u1, n0, n1;
            orc_chain_random(seed, t, (uint32_t)i, 0x10001u, &u0, &u1, &n0, &n1);
            double ratio = (beta[i] - beta[i + 1]) * (loglike[i + 1] - loglike[i]);
            if (beta[i] != beta[i + 1] && fabs(log(u0) - ratio) < mg) mg = fabs(log(u0) - ratio);
            if (log(u0) < ratio) {
                for (int k = 0; k < P; ++k) { double x = params[(size_t)i * P + k]; params[(size_t)i * P + k] = params[(size_t)(i + 1) * P + k]; params[(size_t)(i + 1) * P + k] = x; }
                double x = loglike[i]; loglike[i] = loglike[i + 1]; loglike[i + 1] = x;
                swapped[i] += 1; swapped[i + 1] += 1;
            }
        }
    }
    if (margin) *margin = mg;
    free(prop); free(flux); free(counts);
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
