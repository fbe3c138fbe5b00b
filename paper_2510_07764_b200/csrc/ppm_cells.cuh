// ppm_cells.cuh -- S4 + S5 of DESIGN.md: the per-(cell, phase, energy) shift-and-add kernel
// (Eq 45-47) with the atmosphere interpolation.  The per-row
// table-slice build and the deterministic cross-chunk reduction are in ppm_rowops.cuh.  Product path (sm_100a).
#pragma once
#include "ppm_common.cuh"

namespace ppm {

constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52: (x + kMagic) rounds x to the nearest integer

struct CellArgs {
    const StarD* stars; const SpotD* spots; const RowD* rows; const int* cells;
    const double* tmpl;      // [rows][4][n_fp+1]
    const double* slices;    // [rows][nmu][nx]  (table emission)
    const double* axmu;      // [nmu]
    const long long* uef;    // [nE]: round(log10(E_e) / h * 2^52): energy part of the logx coordinate in fixed point
                             //       (h = logx spacing; units of 2^-52 table intervals)
    long long uef_step;      // log-uniform energy grids (uniform_e = 1): 32 * the grid's constant step of uef (see EnergyCoord)
    int uniform_e;
    const double* en;        // [nE]: E_e (keV)
    double* partial;         // [nb][nchunk][n_phase][nE]
    const double* tmap;      // temperature-map mode: [rows][n_phi] log10 T per cell
    const double* values;    // temperature-map mode: the 4-D table [nT][ng][nmu][nx]
    const double* axT;       // temperature-map mode: log T axis [nT]
    int nT, ng;
    int wst, map_split;      // temperature-map mode: column capacity of the windowed slice buffers; 1 = rows are split
                             // between the windowed (16-warp) and the full-width (8-warp) launch
    unsigned long long* pairs;   // counter: (cell, phase) pairs with F_p != 0 (energy tile 0 only)
    double x0_over_h, inv_h;
    int nb, RT, n_spots, n_theta, n_phi, n_phase, n_fp, nE;
    int nmu, nx, mu_rule, x_linedge;
    int t_rule;              // temperature-map mode under strategies a-c (k_cells_map4): AxisRule of the log T axis
    int nchunk, rows_per_chunk, nw, n_etile, mesh;
    int beaming;             // blackbody only: 0 isotropic, 1 cos^2(sigma'), 2 sin^2(sigma')
    int clip;                // intensity-domain interpolation (k_cells_lin): 1 = strategy b, negative intensities -> 0
    int phase_order;         // Interp of Eq 46: 1 linear (reading R11), 3 four-point Lagrange (reading R11b)
    double y_lo, y_hi;       // bounds of log2(10) * (any interpolated table value): a pair whose log2(F_p T^3) + y_lo
                             // < -900 or + y_hi > 900 takes the range-checked energy loop (exponent add must not wrap)
};

// 2^y for the table path: y = n + f, n = round(y) through the 1.5*2^52 constant (done by the caller), |f| <= 1/2;
// 2^f by a degree-8 polynomial (Chebyshev-node fit on [-1/2, 1/2]; max relative error 1.1e-12 -- three orders
// below the 1e-9 per-bin parity bar; degree 10 reaches 4e-16 at +2 DFMA per triple, measured 6 % slower),
// 2^n by an integer add into the exponent field.  The caller drops terms with n < -1000.
// (Literal coefficients: measured faster than operands from the constant bank -- C5 x 8 54.3 vs 56.3 ms, maps 11.5 vs 13.0 ms.)
__device__ __forceinline__ double exp2_frac_scaled(double f, int n)      // 2^f * 2^n, |f| <= 1/2, no range check
{
    double p = 1.3255224878668817e-06;
    p = fma(p, f, 1.5310079402249296e-05);
    p = fma(p, f, 0.00015403455852453838);
    p = fma(p, f, 0.0013333450568000645);
    p = fma(p, f, 0.009618129159402558);
    p = fma(p, f, 0.05550410941205933);
    p = fma(p, f, 0.2402265069581299);
    p = fma(p, f, 0.6931471805459335);
    p = fma(p, f, 1.0);
    return __hiloint2double(__double2hiint(p) + n * 1048576, __double2loint(p));
}

// ------------------------------------------------------------------------------------------------
// Step A of every cell kernel: one lane <-> one (cell, output phase) slot.
// phase_of_cell: Eq 45.  template_interp: the bracket phi_o[i] <= phi_p < phi_o[i+1] and Interp of
// Eq 46 -- ORDER 1: piecewise linear (reading R11); ORDER 3: 4-point Lagrange on the true
// abscissae phi_o with periodic wrap, reverting to linear when one of the four F nodes is 0 (a hidden or filled
// entry, Eq 41; reading R11b).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double phase_of_cell(double phi_out, double phi_m, double phi_off, double po0)
{
    const double s0 = phi_out + phi_m / (2.0 * kPi) + phi_off + 1.0 - po0;
    return (s0 - floor(s0)) + po0;
}

__device__ __forceinline__ void template_interp(const double* __restrict__ F, const double* __restrict__ Z,
                                                const double* __restrict__ PO, const double* __restrict__ MU, int n_fp,
                                                int order, double phi_p, double& Fp, double& zp, double& mup)
{
    int lo = 0, hi = n_fp;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (PO[mid] <= phi_p) lo = mid; else hi = mid;
    }
    if (order == 3) {
        const int i0 = (lo == 0) ? n_fp - 1 : lo - 1, i3 = (lo + 2 > n_fp) ? 1 : lo + 2;
        const double f0 = F[i0], f1 = F[lo], f2 = F[lo + 1], f3 = F[i3];
        if (f0 != 0.0 && f1 != 0.0 && f2 != 0.0 && f3 != 0.0) {
            const double x0 = PO[i0] + ((lo == 0) ? -1.0 : 0.0), x1 = PO[lo], x2 = PO[lo + 1];
            const double x3 = PO[i3] + ((lo + 2 > n_fp) ? 1.0 : 0.0);
            const double d0 = phi_p - x0, d1 = phi_p - x1, d2 = phi_p - x2, d3 = phi_p - x3;
            const double w0 = (d1 * d2 * d3) / ((x0 - x1) * (x0 - x2) * (x0 - x3));
            const double w1 = (d0 * d2 * d3) / ((x1 - x0) * (x1 - x2) * (x1 - x3));
            const double w2 = (d0 * d1 * d3) / ((x2 - x0) * (x2 - x1) * (x2 - x3));
            const double w3 = (d0 * d1 * d2) / ((x3 - x0) * (x3 - x1) * (x3 - x2));
            Fp = fma(w3, f3, fma(w2, f2, fma(w1, f1, w0 * f0)));
            zp = fma(w3, Z[i3], fma(w2, Z[lo + 1], fma(w1, Z[lo], w0 * Z[i0])));
            mup = fma(w3, MU[i3], fma(w2, MU[lo + 1], fma(w1, MU[lo], w0 * MU[i0])));
            return;
        }
    }
    const double t = (phi_p - PO[lo]) / (PO[lo + 1] - PO[lo]);
    Fp = F[lo] + (F[lo + 1] - F[lo]) * t;
    zp = Z[lo] + (Z[lo + 1] - Z[lo]) * t;
    mup = MU[lo] + (MU[lo + 1] - MU[lo]) * t;
}

// azimuth of cell m of a row (box mesh, reading R1; HEALPix ring, Eq 24-27)
__device__ __forceinline__ double cell_azimuth(int mesh, const RowD& row, const SpotD& sp, int m)
{
    return mesh ? row.phi0 + (double)m * row.dphi : sp.phi_c + (-sp.W + ((double)m + 0.5) * sp.dphi);
}

// flags of a pair record (int2.y); bits 8.. hold the number of energy groups that still need per-triple work when only
// PAIR_CLAMP_HI is set (see k_cells_tab)
enum { PAIR_CLAMP_LO = 1, PAIR_CLAMP_HI = 2, PAIR_RANGE = 4 };

// The table part of a pair record: logx coordinate of the pair in fixed point (units of 2^-52 intervals; the energy
// part uef[e] is added per triple), log2(F_p T^3), the mu stencil (weights pre-scaled by log2(10)), the window of logx
// intervals [jlo, jhi] the tile's energies touch (coordinates clamped to the table, reading R13b) and the flags.
//   info = (first mu row of the stencil * row_stride) | jlo << 16 | jhi << 24
__device__ __forceinline__ void pair_table_record(double Fp, double zp, double mup, double log10kT, double log2T3,
                                                  const double* __restrict__ MUAX, int nmu, int mu_rule, int row_stride,
                                                  double inv_h, double x0_over_h, long long uef_first,
                                                  long long uef_last, long long s_top, double y_lo, double y_hi,
                                                  long long& pq, double& pb, double ww[4], int& info, int& flags)
{
    const double up = (log10(zp) - log10kT) * inv_h - x0_over_h;                 // (x - x0)/h less the energy part
    pq = __double2ll_rn(up * 4503599627370496.0);
    pb = log2(Fp) + log2T3;
    int mb;
    axis_w4(MUAX, nmu, mup, mu_rule, mb, ww);
#pragma unroll
    for (int q4 = 0; q4 < 4; ++q4) ww[q4] *= kLog2_10;
    const long long sa = pq + uef_first, sb2 = pq + uef_last;
    const long long sac = sa < 0 ? 0 : (sa > s_top ? s_top : sa);
    const long long sbc = sb2 < 0 ? 0 : (sb2 > s_top ? s_top : sb2);
    info = (mb * row_stride) | ((int)(sac >> 52) << 16) | ((int)(sbc >> 52) << 24);
    flags = (sa < 0 ? PAIR_CLAMP_LO : 0) | (sb2 > s_top ? PAIR_CLAMP_HI : 0) |
            ((!(pb + y_lo > -900.0) || !(pb + y_hi < 900.0)) ? PAIR_RANGE : 0);
}


// ------------------------------------------------------------------------------------------------
// K5: shift-and-add (Eq 45-47).  Block = (row chunk, group of `nw` consecutive output
// phases, vector x energy tile); warp w owns output phase k and the 32*EPL energies of the tile (lane
// owns energies e0+lane+32 i): the (k, e) accumulators live in registers for the whole chunk --
// output-stationary, no atomics.  Per row the ring template sits in shared memory.  Lanes first prepare
// 32 (cell, k) pairs in parallel (Eq 45-46), then the warp walks the pairs with F_p != 0.
// k_cells_bb: closed-form isotropic blackbody (Eq C.5).  k_cells_tab (below): table.
// ------------------------------------------------------------------------------------------------
template <int EPL>
__global__ void __launch_bounds__(512, 1) k_cells_bb(CellArgs A)
{
    extern __shared__ __align__(16) double sm[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int chunk = blockIdx.x, pg = blockIdx.y;
    const int b = blockIdx.z / A.n_etile, et = blockIdx.z % A.n_etile;
    const int k = pg * A.nw + w;
    const bool kvalid = k < A.n_phase;
    const int e0 = et * 32 * EPL;
    const int n1 = A.n_fp + 1;
    double* T = sm;                                  // F, z, phi_o, mu: [4][n1]

    double en[EPL], ok[EPL], acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) {
        const int e = e0 + lane + 32 * i;
        en[i] = (e < A.nE) ? A.en[e] : 1.0;
        ok[i] = (e < A.nE) ? 1.0 : 0.0;
        acc[i] = 0.0;
    }
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
        const double* ts = A.tmpl + (size_t)rid * 4 * n1;
        for (int i = threadIdx.x; i < 4 * n1; i += blockDim.x) T[i] = ts[i];
        __syncthreads();
        if (!kvalid) continue;
        const double* F = T;
        const double* Z = T + n1;
        const double* PO = T + 2 * n1;
        const double* MU = T + 3 * n1;
        const int* cl = A.cells + (size_t)rid * A.n_phi;
        const double po0 = PO[0];
        for (int base = 0; base < nact; base += 32) {
            const int idx = base + lane;
            double Fp = 0.0, pa = 0.0, pb = 0.0;      // pa = z_p / kT, pb = F_p z_p^3 2/(h^3 c^2)
            if (idx < nact) {
                const double phi_p = phase_of_cell(phi_out, cell_azimuth(A.mesh, row, sp, cl[idx]), phi_off, po0);   // Eq 45
                double zp, mup;
                template_interp(F, Z, PO, MU, A.n_fp, A.phase_order, phi_p, Fp, zp, mup);                            // Eq 46
                if (!(Fp > 0.0)) Fp = 0.0;
                if (Fp != 0.0) {
                    pa = zp / sp.kT;
                    pb = Fp * (2.0 / (kH_keV_s * kH_keV_s * kH_keV_s * kC_cm_s * kC_cm_s)) * zp * zp * zp;
                    if (A.beaming) pb *= (A.beaming == 1) ? mup * mup : 1.0 - mup * mup;      // cos(sigma') = mu_p (Eq 20)
                }
            }
            unsigned todo = __ballot_sync(0xffffffffu, Fp != 0.0);
            npairs += __popc(todo);
            while (todo) {
                const int j = __ffs(todo) - 1;
                todo &= todo - 1;
                const double qa = __shfl_sync(0xffffffffu, pa, j);
                const double qb = __shfl_sync(0xffffffffu, pb, j);
#pragma unroll
                for (int i = 0; i < EPL; ++i) {
                    const double E = en[i];
                    acc[i] += ok[i] * (qb * E * E / expm1(qa * E));             // F_p I(z_p E)/E, Eq 47 with Eq C.5
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

// ------------------------------------------------------------------------------------------------
// K5t: the table-emission cell kernel (the dominant kernel of the path).  Same block / warp / lane
// ownership as k_cells above (output-stationary accumulators, no atomics); what differs is how a
// (cell, phase) pair is turned into its energies' terms:
//  * logx coordinate in fixed point.  u = (log10(z_p E_e / kT) - x0)/h = u_pair + u_e is carried as a
//    64-bit integer in units of 2^-52 intervals: s = q_pair + uef[e] (two integer adds; on log-uniform energy
//    grids the lane steps s from one energy group to the next by one warp-uniform constant, EnergyCoord).  The
//    interval index is s >> 52 and the fraction, OR-ed under the exponent of 1.0, gives t = 1 + frac directly
//    as a double -- no floating-point round-and-subtract -- and the window below is found with the same integers.
//  * one fused pass per pair over the window of logx intervals its energies touch: lane l contracts
//    the mu stencil at NPL consecutive nodes (4 loads + 4 FMA each, slice rows in shared memory),
//    takes the three neighbouring node values from lanes l-1 / l+1 by shuffle, and writes the
//    monomial coefficients a0..a3 in t (forward differences, cubic_coeffs) of its NPL intervals -- cubic
//    Lagrange on the 4 surrounding nodes; linear (strategies c, d) or the inward-shifted stencil (strategies
//    a, b) in the first / last interval of the axis -- pre-scaled by log2(10), with log2(F_p T^3) in a0.  NPL is
//    odd so that the lanes' 8- and 16-byte accesses at stride NPL fall in distinct banks.
//  * per triple: 2 x LDS.128 (a0..a3), Horner in t (3 DFMA), exp2 (3 DADD + 8 DFMA), accumulate (1 DADD).
// The division by E_e of Eq 47 is the same for every term of a bin: applied once in the epilogue.
// ------------------------------------------------------------------------------------------------
constexpr double kTwo52 = 4503599627370496.0;

// (a & 0x000FFFFF) | 0x3FF00000 in one LOP3: the high word of 1 + frac
__device__ __forceinline__ int one_plus_frac_hi(int shi)
{
    int r;
    asm("lop3.b32 %0, %1, 0x000FFFFF, 0x3FF00000, 0xEA;" : "=r"(r) : "r"(shi));
    return r;
}

// node value of the pair at slice column `col` of the stencil's first mu row: log2(10) * sum_mu w_mu S[mu][col] + log2(F_p T^3)
// (the Lagrange weights of every x rule sum to 1, so adding the constant to the nodes adds it to k0 only)
__device__ __forceinline__ double node_value(const double* __restrict__ sp0, int nx, double v0, double v1, double v2,
                                             double v3, double qb)
{
    return fma(v3, sp0[3 * nx], fma(v2, sp0[2 * nx], fma(v1, sp0[nx], fma(v0, sp0[0], qb))));
}

// monomial coefficients, in t = 1 + (fraction of the interval) -- t runs over [1, 2) across the interval between the
// nodes c1 and c2; the four nodes sit at t = 0, 1, 2, 3 -- of the cubic through the node values c0..c3: Newton's forward
// differences (differences of neighbouring nodes first: no cancellation against the nodes' common magnitude) turned
// into monomials.  t is what the fixed-point coordinate yields directly (fraction bits under the exponent of 1.0), so a
// triple needs no subtraction to centre it.  Neighbouring intervals of a lane share their first and second differences.
__device__ __forceinline__ void cubic_coeffs(double c0, double c1, double c2, double c3, double& a0, double& a1,
                                             double& a2, double& a3)
{
    const double d1 = c1 - c0, d2 = c2 - c1, d3 = c3 - c2;
    const double e1 = d2 - d1, e2 = d3 - d2;
    const double t3 = e2 - e1;
    const double h2 = 0.5 * e1;
    a0 = c0;
    a1 = d1 - fma(t3, -1.0 / 3.0, h2);
    a2 = fma(t3, -0.5, h2);
    a3 = t3 * (1.0 / 6.0);
}

// debug build (-DPPM_BOUNDS): every shared-memory access of the table cell kernel is checked against the block's
// dynamic allocation and traps when it falls outside (compute-sanitizer is not available on the GPU pool)
#ifdef PPM_BOUNDS
__device__ __forceinline__ void smem_check(const void* p, size_t bytes, const void* base)
{
    unsigned dyn;
    asm volatile("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn));
    const char* c = static_cast<const char*>(p);
    const char* b = static_cast<const char*>(base);
    if (c < b || c + bytes > b + dyn) __trap();
}
#define PPM_SMEM_CHECK(p, bytes) smem_check((p), (bytes), sm)
#else
#define PPM_SMEM_CHECK(p, bytes) ((void)0)
#endif

// Node value of a pair at slice column n for the uniform-temperature kernels: the row's one (mu x logx) slice.
struct SliceNode {
    const double* srow;                  // slice row of the stencil's first mu node
    int nx;
    double v0, v1, v2, v3, qb;           // mu weights (pre-scaled by log2(10)) and log2(F_p T^3)
    __device__ __forceinline__ double operator()(int n) const { return node_value(srow + n, nx, v0, v1, v2, v3, qb); }
    __device__ __forceinline__ void check(int n0, int count, const double* sm) const
    {
        PPM_SMEM_CHECK(srow + n0, sizeof(double) * (3 * nx + count));
        (void)n0; (void)count; (void)sm;
    }
};

// ---- fused pass of a pair: node values -> interval coefficients.  Lane l holds nodes n0 .. n0+NPL-1, n0 = jlo-1 + NPL l;
// interval c (nodes c, c+1) has window offset c - (jlo-1).  Out-of-table nodes read neighbouring shared memory: they only
// feed window slots that no energy reads.  node(n) = the pair's value at slice column n (SliceNode; MapNode of
// ppm_cells_map.cuh blends two log T node slices).  Writes KA[0..KW) = (a0,a1), KA[KW..2KW) = (a2,a3); both
// __syncwarp's are inside (the previous pair's readers are done / the new coefficients are visible).
template <int NPL, class NodeFn>
__device__ __forceinline__ void fused_pass(const NodeFn& node, int nx, int jlo, int jhi, int lane, int x_linedge, double2* KA,
                                           const double* sm)
{
    constexpr int KW = 32 * NPL;
    const int n0 = jlo - 1 + NPL * lane;
    node.check(n0, NPL, sm);
    double f[NPL + 3];                    // f[1+j] = node n0+j; f[0] = node n0-1; f[NPL+1], f[NPL+2] = next lane's first two
#pragma unroll
    for (int jn = 0; jn < NPL; ++jn) f[1 + jn] = node(n0 + jn);
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
    for (int jn = 0; jn < NPL; ++jn) cubic_coeffs(f[jn], f[jn + 1], f[jn + 2], f[jn + 3], ka[jn].x, ka[jn].y, kb[jn].x, kb[jn].y);
    if (jlo == 0 || jhi == nx - 2) {      // the window holds the first / last interval of the axis (warp-uniform)
#pragma unroll
        for (int jn = 0; jn < NPL; ++jn) {
            const int c = n0 + jn;
            if (c != 0 && c != nx - 2) continue;
            if (x_linedge) {                                        // strategies c, d: linear
                const double d = f[jn + 2] - f[jn + 1];             // y = f1 + d (t - 1)
                ka[jn] = make_double2(f[jn + 1] - d, d);
                kb[jn] = make_double2(0.0, 0.0);
            } else {                                                // strategies a, b: stencil shifted inward
                const int s = (c == 0) ? 0 : nx - 4;
                double g[4];
#pragma unroll
                for (int m = 0; m < 4; ++m) g[m] = node(s + m);
                double k0, k1, k2, k3;
                cubic_coeffs(g[0], g[1], g[2], g[3], k0, k1, k2, k3);
                const double d = (double)(c - 1 - s);               // Taylor shift: this interval is [1, 2) of its own t
                ka[jn] = make_double2(fma(d, fma(d, fma(d, k3, k2), k1), k0), fma(d, fma(3.0 * d, k3, 2.0 * k2), k1));
                kb[jn] = make_double2(fma(3.0 * d, k3, k2), k3);
            }
        }
    }
    __syncwarp();                                                   // the previous pair's readers are done
#pragma unroll
    for (int jn = 0; jn < NPL; ++jn) {
        KA[NPL * lane + jn] = ka[jn];
        KA[NPL * lane + jn + KW] = kb[jn];
    }
    __syncwarp();
}

// one triple: logx coordinate s (fixed point) -> interval coefficients -> y -> 2^y (no range checks)
template <int KW>
__device__ __forceinline__ double triple_value(const double2* __restrict__ KAq, long long s)
{
    const int shi = (int)(s >> 32);
    const double2* kp = KAq + (shi >> 20);                                      // interval index = s >> 52
    const double t = __hiloint2double(one_plus_frac_hi(shi), (int)s);              // 1 + fraction of the interval
    const double2 c01 = kp[0], c23 = kp[KW];
    const double y = fma(fma(fma(c23.y, t, c23.x), t, c01.y), t, c01.x);
    const double r = y + kMagic;
    return exp2_frac_scaled(y - (r - kMagic), __double2loint(r));
}

// the same with the coordinate clamped to the table (reading R13b) and the exponent range checked on both sides:
// below 2^-1000 the term is 0, above 2^1000 it is +inf (the exponent add of exp2_frac_scaled would wrap)
template <int KW>
__device__ __forceinline__ double triple_value_checked(const double2* __restrict__ KAq, long long s, long long s_top)
{
    s = s < 0 ? 0 : (s > s_top ? s_top : s);
    const int shi = (int)(s >> 32);
    const double2* kp = KAq + (shi >> 20);
    const double t = __hiloint2double(one_plus_frac_hi(shi), (int)s);              // 1 + fraction of the interval
    const double2 c01 = kp[0], c23 = kp[KW];
    const double y = fma(fma(fma(c23.y, t, c23.x), t, c01.y), t, c01.x);
    const double r = y + kMagic;
    const int n = __double2loint(r);
    const double v = exp2_frac_scaled(y - (r - kMagic), n);
    return !(y > -1000.0) ? 0.0 : (y > 1000.0 ? INFINITY : v);
}

// How a triple gets its cubic.  CoefTriple: the interval's record (a0..a3) from the per-warp coefficient arrays -- 2 x
// LDS.128 per triple, the per-pair pass has built and stored every interval's record (fused_pass).  NodeTriple: the four
// NODE VALUES around the interval from a per-warp node array (4 x LDS.64 per triple; the per-pair pass stores 8 bytes per
// node instead of 32 per interval and skips the Lagrange -> monomial step), the triple forms its own cubic (9 FP64 more):
// cheaper when a lane owns few energies (EPL <= 4: the per-pair pass is amortised over few triples).  Used for the pairs
// whose window holds no end interval of the axis (those keep the records, which carry the end rules).
template <int KW>
struct CoefTriple {
    const double2* KAq;
    __device__ __forceinline__ double value(long long s) const { return triple_value<KW>(KAq, s); }
    __device__ __forceinline__ double checked(long long s, long long s_top) const { return triple_value_checked<KW>(KAq, s, s_top); }
};

struct NodeTriple {
    const double* NVq;                   // node value of table column n at NVq[n]
    __device__ __forceinline__ double y_of(long long s) const
    {
        const int shi = (int)(s >> 32);
        const double* p = NVq + (shi >> 20);
        double a0, a1, a2, a3;
        cubic_coeffs(p[-1], p[0], p[1], p[2], a0, a1, a2, a3);
        const double t = __hiloint2double(one_plus_frac_hi(shi), (int)s);
        return fma(fma(fma(a3, t, a2), t, a1), t, a0);
    }
    __device__ __forceinline__ double value(long long s) const
    {
        const double y = y_of(s);
        const double r = y + kMagic;
        return exp2_frac_scaled(y - (r - kMagic), __double2loint(r));
    }
    __device__ __forceinline__ double checked(long long s, long long s_top) const
    {
        s = s < 0 ? 0 : (s > s_top ? s_top : s);
        const double y = y_of(s);
        const double r = y + kMagic;
        const double v = exp2_frac_scaled(y - (r - kMagic), __double2loint(r));
        return !(y > -1000.0) ? 0.0 : (y > 1000.0 ? INFINITY : v);
    }
};

// The energy part of the logx coordinate for the EPL energies e0 + lane + 32 i a lane owns.
//  UNI = false: one 64-bit value per energy in registers (2 EPL registers).
//  UNI = true (log-uniform energy grid -- the paper's grids are, Eq 50): energy i sits at uef[e0 + lane] + i D with
//  ONE warp-uniform step D = 32 * (step of uef), so a lane carries its coordinate from group to group by one 64-bit add
//  and the 2 EPL registers become 2.  The host takes this path only when every energy's own uef differs from that
//  affine form by <= 256 units of 2^-52 intervals (5.7e-14 of a table interval: a relative change of the energy of 2.6e-15,
//  ~ 12 ulp of a double; worst-case effect on a term 2.6e-13, the seeded grids deviate by <= 105 units) and when only the
//  last group of a tile is ragged; a lane whose last energy does not exist evaluates the tile's last real one (the
//  result is never stored).
template <int EPL, bool UNI>
struct EnergyCoord {
    long long u[UNI ? 1 : EPL];
    long long D, Dlast;
    __device__ __forceinline__ void init(const long long* __restrict__ uef, long long step, int e0, int lane, int nE)
    {
        if constexpr (UNI) {
            u[0] = uef[imin_(e0 + lane, nE - 1)];
            D = step;
            // a lane without a last energy sits on the tile's last real energy (one address for all such lanes: a
            // broadcast, no bank conflict against the real lanes of its quarter-warp)
            const int e_last = imin_(e0 + 32 * EPL, nE) - 1;
            const long long last = uef[e0 + ((e_last - e0) & 31)] + (long long)((e_last - e0) >> 5) * step;
            Dlast = (e0 + lane + 32 * (EPL - 1) < nE) ? step : last - (u[0] + (long long)(EPL - 2) * step);
        } else {
#pragma unroll
            for (int i = 0; i < EPL; ++i) u[i] = uef[imin_(e0 + lane + 32 * i, nE - 1)];
            D = Dlast = 0;
        }
    }
    __device__ __forceinline__ long long first(long long q) const { return q + u[0]; }
    // coordinate of group i + 1 given s = that of group i
    __device__ __forceinline__ long long next(long long s, long long q, int i) const
    {
        if constexpr (UNI) return s + ((i == EPL - 2) ? Dlast : D);
        else return q + u[i + 1 < EPL ? i + 1 : EPL - 1];
    }
};

// Energies of a pair whose upper part lies beyond the top of the logx axis.  The lane's energies e0 + lane + 32 i rise
// with i and with the lane, so the groups i >= G (G warp-uniform: the groups whose FIRST energy is still inside the table)
// are clamped for every lane: their term is the pair's constant 2^y(s_top) and is not evaluated here (the caller defers it).
// Groups i < G - 1 are entirely inside the table; group G - 1 may straddle the end and clamps its coordinate.
// One fully unrolled instance per G keeps the G independent dependency chains interleaved.
template <int EPL, int G, bool UNI, class Tri>
__device__ __forceinline__ void energies_clamped_hi(double (&acc)[EPL], const EnergyCoord<EPL, UNI>& ec, const Tri& tri,
                                                    long long q, long long s_top)
{
    long long s = ec.first(q);
#pragma unroll
    for (int i = 0; i < G - 1; ++i) {
        acc[i] += tri.value(s);
        s = ec.next(s, q, i);
    }
    acc[G - 1] += tri.value(s > s_top ? s_top : s);
}

template <int EPL, int G, bool UNI, class Tri>
__device__ __forceinline__ void dispatch_clamped_hi(int g, double (&acc)[EPL], const EnergyCoord<EPL, UNI>& ec, const Tri& tri,
                                                    long long q, long long s_top)
{
    if (g == G) energies_clamped_hi<EPL, G, UNI>(acc, ec, tri, q, s_top);
    else if constexpr (G > 1) dispatch_clamped_hi<EPL, G - 1, UNI>(g, acc, ec, tri, q, s_top);
}

// Number of energy groups of a pair whose FIRST energy still lies inside the table (used when only PAIR_CLAMP_HI is set):
// UG[i] = coordinate part of group i's first energy (a group without any energy holds 2^62).
template <int NG>
__device__ __forceinline__ int clamped_groups(long long pq, const long long* __restrict__ UG, long long s_top)
{
    int g = 0;
#pragma unroll
    for (int i = 0; i < NG; ++i) g += (pq + UG[i] <= s_top) ? 1 : 0;
    return g;
}

// The energies of one pair (step B, part ii): tri = how a triple gets its cubic (above), q = the pair's coordinate,
// flg = its flags (bits 8.. = clamped_groups when only PAIR_CLAMP_HI is set), hdef = the lane's deferred sum.
template <int EPL, bool UNI, class Tri>
__device__ __forceinline__ void pair_energies_with(double (&acc)[EPL], double& hdef, const EnergyCoord<EPL, UNI>& ec, const Tri& tri,
                                                   long long q, int flg, long long s_top, int lane)
{
    if (flg == 0) {
        // every coordinate of the tile lies inside the table and every exponent is in range
        long long s = ec.first(q);
#pragma unroll
        for (int i = 0; i < EPL; ++i) {
            acc[i] += tri.value(s);
            s = ec.next(s, q, i);
        }
    } else if ((flg & 7) == PAIR_CLAMP_HI) {
        // the upper energies lie beyond the top of the logx axis: the clamped coordinate (reading R13b) makes their term
        // the pair's constant 2^y(s_top).  Groups g .. EPL-1 (g = flg >> 8) are clamped for every lane: the constant goes
        // to lane g's deferred sum and is spread over acc[g ..] once, in the epilogue (spread_deferred).
        const int g = flg >> 8;
        if (g < EPL) {                                                          // (g == EPL: only the last group straddles the end)
            const double vtop = tri.value(s_top);
            if (lane == g) hdef += vtop;
        }
        dispatch_clamped_hi<EPL, EPL, UNI>(g, acc, ec, tri, q, s_top);
    } else {
        // energies below the axis, or extreme table values (|exponent| may exceed the double range): clamped,
        // range-checked form
        long long s = ec.first(q);
#pragma unroll
        for (int i = 0; i < EPL; ++i) {
            acc[i] += tri.checked(s, s_top);
            s = ec.next(s, q, i);
        }
    }
}

// ... with the interval records of fused_pass (KAq = the pair's coefficient window indexed by interval)
template <int KW, int EPL, bool UNI>
__device__ __forceinline__ void pair_energies(double (&acc)[EPL], double& hdef, const EnergyCoord<EPL, UNI>& ec,
                                              const double2* __restrict__ KAq, long long q, int flg, long long s_top, int lane,
                                              const double* sm)
{
#ifdef PPM_BOUNDS
    {   // every record address of the plain loop (the other loops clamp into the same range)
        long long s = ec.first(q);
        for (int i = 0; i < EPL; ++i) {
            const long long sc = s < 0 ? 0 : (s > s_top ? s_top : s);
            PPM_SMEM_CHECK(KAq + (sc >> 52), sizeof(double2));
            PPM_SMEM_CHECK(KAq + (sc >> 52) + KW, sizeof(double2));
            s = ec.next(s, q, i);
        }
    }
#endif
    (void)sm;
    pair_energies_with<EPL, UNI>(acc, hdef, ec, CoefTriple<KW>{KAq}, q, flg, s_top, lane);
}

// deferred constants of the clamped groups: acc[i] += sum over g <= i of lane g's hdef (inclusive scan over lanes)
template <int EPL>
__device__ __forceinline__ void spread_deferred(double (&acc)[EPL], double hdef, int lane)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const double up = __shfl_up_sync(0xffffffffu, hdef, d);
        if (lane >= d) hdef += up;
    }
#pragma unroll
    for (int i = 0; i < EPL; ++i) acc[i] += __shfl_sync(0xffffffffu, hdef, i);
}

// NX = true ("node exchange", EPL <= 4): for the pairs whose window holds no end interval of the axis the per-pair pass
// stores node values and the triples form their own cubics (NodeTriple) instead of fetching interval records.
template <int EPL, int NPL, bool UNI, bool NX>
__global__ void __launch_bounds__(512, 1) k_cells_tab(CellArgs A)
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
    // shared layout (doubles): per warp { KA [KW] (k0,k1), KB [KW] (k2,k3), R0 [32] (q,qb), R1 [32] (v0,v1), R2 [32] (v2,v3)
    // as double2, RI [32] int2 (info, flags) } | S [nmu][nx] | T [4][n1] | MUAX [nmu].  Struct-of-arrays so that lanes
    // touch consecutive 16-byte words (no bank conflicts); KA / KB are indexed by node offset inside the pair's window.
    constexpr int KW = 32 * NPL;
    constexpr int WARP_DBL = 4 * KW + 3 * 64 + 32;
    double* wbase = sm + (size_t)w * WARP_DBL;
    double2* KA = reinterpret_cast<double2*>(wbase);
    double2* R0 = KA + 2 * KW;
    double2* R1 = R0 + 32;
    double2* R2 = R1 + 32;
    int2* RI = reinterpret_cast<int2*>(R2 + 32);
    double* S = sm + (size_t)A.nw * WARP_DBL;
    double* T = S + plane;
    double* MUAX = T + 4 * n1;
    long long* UG = reinterpret_cast<long long*>(MUAX + A.nmu);                 // [NG]: coordinate part of each group's first energy
    // energy group i = the 32 consecutive energies e0 + 32 i + lane: energies rise with the group index and with the lane
    constexpr int NG = EPL;

    EnergyCoord<EPL, UNI> ec;
    ec.init(A.uef, A.uef_step, e0, lane, A.nE);
    double acc[EPL];
#pragma unroll
    for (int i = 0; i < EPL; ++i) acc[i] = 0.0;
    double hdef = 0.0;                           // lane g: sum of the constants 2^y(s_top) of the pairs whose groups >= g are clamped
    // first / last coordinate of the tile's energies, in the same form the lanes use (EnergyCoord): the coordinates are
    // monotone in the energy index, so every index the energy loop forms lies inside the window found from these two
    const long long uef_first = A.uef[imin_(e0, A.nE - 1)];
    const int e_last = imin_(e0 + 32 * EPL, A.nE) - 1;
    const long long uef_last = UNI ? A.uef[e0 + ((e_last - e0) & 31)] + (long long)((e_last - e0) >> 5) * A.uef_step
                                   : A.uef[e_last];
    const long long s_top = ((long long)(nx - 1) << 52) - 1;                     // largest in-table coordinate
    for (int i = threadIdx.x; i < A.nmu; i += blockDim.x) MUAX[i] = A.axmu[i];
    if (threadIdx.x < NG) {                      // a group without any energy (ragged tail) counts as beyond the table
        const int ef = e0 + 32 * (int)threadIdx.x;
        UG[threadIdx.x] = (ef < A.nE) ? (UNI ? A.uef[e0] + (long long)threadIdx.x * A.uef_step : A.uef[ef]) : (1ll << 62);
    }

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
                const double qb = r0.y, v0 = r1.x, v1 = r1.y, v2 = r2.x, v3 = r2.y;
                const int jlo = (inf >> 16) & 255, jhi = (inf >> 24) & 255;
                const SliceNode node{S + (inf & 0xFFFF), nx, v0, v1, v2, v3, qb};
                if (NX && jlo != 0 && jhi != nx - 2) {
                    // node exchange (pairs whose window holds no end interval of the axis): lane l contracts the mu stencil
                    // at its NPL nodes and stores the VALUES; node n of the table sits at NV[n - (jlo - 1)]
                    const int n0 = jlo - 1 + NPL * lane;
                    double* NV = wbase;
                    double fv[NPL];
#pragma unroll
                    for (int jn = 0; jn < NPL; ++jn) fv[jn] = node(n0 + jn);
                    __syncwarp();                                               // the previous pair's readers are done
#pragma unroll
                    for (int jn = 0; jn < NPL; ++jn) NV[NPL * lane + jn] = fv[jn];
                    __syncwarp();
                    pair_energies_with<EPL, UNI>(acc, hdef, ec, NodeTriple{NV - (jlo - 1)}, q, flg, s_top, lane);
                } else {
                    fused_pass<NPL>(node, nx, jlo, jhi, lane, A.x_linedge, KA, sm);
                    const double2* KAq = KA + (1 - jlo);
                    pair_energies<KW, EPL, UNI>(acc, hdef, ec, KAq, q, flg, s_top, lane, sm);
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
