// ppm.cu -- C ABI (include/ppm.h) of the B200-native PPM hot path: context, table upload, launch
// sequencing.  All arithmetic of the path runs in the kernels of ppm_geodesic.cuh / ppm_cells.cuh /
// ppm_observe.cuh.  No CPU fallback.  Build: nvcc -gencode arch=compute_100a,code=sm_100a (see
// paper_2510_07764_b200/_build.py).
#include "ppm.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "ppm_common.cuh"
#include "ppm_geodesic.cuh"
#include "ppm_cells.cuh"
#include "ppm_rowops.cuh"
#include "ppm_launch.h"
#include "ppm_observe.cuh"
#include "ppm_chain.cuh"

using namespace ppm;

namespace {

thread_local char g_err[512] = "";

void set_err(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            set_err("%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);  \
            return PPM_ERR_CUDA;                                                                   \
        }                                                                                          \
    } while (0)

#define ARG(cond, msg)                     \
    do {                                   \
        if (!(cond)) {                     \
            set_err("invalid argument: %s", msg); \
            return PPM_ERR_ARG;            \
        }                                  \
    } while (0)

// n-point Gauss-Legendre rule on [-1, 1]: Newton on P_n from the Chebyshev-like guess (textbook).
void gauss_legendre(int n, double* x, double* w)
{
    for (int i = 0; i < n; ++i) {
        long double z = cosl(3.14159265358979323846264338327950288L * (i + 0.75L) / (n + 0.5L)), pp = 1.0L;
        for (int it = 0; it < 100; ++it) {
            long double p1 = 1.0L, p2 = 0.0L;
            for (int j = 1; j <= n; ++j) {
                const long double p3 = p2;
                p2 = p1;
                p1 = ((2.0L * j - 1.0L) * z * p2 - (j - 1.0L) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0L);
            const long double dz = p1 / pp;
            z -= dz;
            if (fabsl(dz) < 1e-19L) {
                p1 = 1.0L; p2 = 0.0L;
                for (int j = 1; j <= n; ++j) {
                    const long double p3 = p2;
                    p2 = p1;
                    p1 = ((2.0L * j - 1.0L) * z * p2 - (j - 1.0L) * p3) / j;
                }
                pp = n * (z * p1 - p2) / (z * z - 1.0L);
                break;
            }
        }
        x[i] = (double)z;
        w[i] = (double)(2.0L / ((1.0L - z * z) * pp * pp));
    }
}

template <typename T>
int dev_alloc(T** p, size_t n)
{
    *p = nullptr;
    if (n == 0) n = 1;
    cudaError_t e = cudaMalloc((void**)p, n * sizeof(T));
    if (e != cudaSuccess) {
        set_err("cudaMalloc of %zu bytes failed: %s", n * sizeof(T), cudaGetErrorString(e));
        return PPM_ERR_NOMEM;
    }
    return PPM_OK;
}

}  // namespace

struct ppm_ctx {
    ppm_config cfg;
    cudaStream_t stream = nullptr;
    int P = 0, RT = 0, n_fp = 0, SB = 1;          // params per vector, rows per vector, sub-batch size
    int nchunk = 1, rows_per_chunk = 1, nw = 1, npg = 1, epl = 1, n_etile = 1, wmax = 0;
    int64_t launches = 0;
    int last_nb = 0;
    // energy grid
    double* d_en = nullptr;
    long long* d_uef = nullptr;                   // log10(E)/h in fixed point (2^-52 intervals)
    int npl = 1;                                  // nodes per lane of the table cell kernel's fused pass
    bool uniform_e = false;                       // log-uniform energy grid: the cell kernels step the coordinate (EnergyCoord)
    int m4_epl = 0, m4_ntile = 0, m4_npl = 0, m4_nw = 0, m4_wst = 0;   // tiling of k_cells_map4 (0: does not fit)
    long long uef_step = 0;                       // 32 * the grid's step of uef
    std::vector<double> h_en;
    // atmosphere
    bool have_atm = false;
    int nT = 0, ng = 0, nmu = 0, nx = 0;
    double x0 = 0, hx = 1;
    double y_lo = 0, y_hi = 0;                    // bounds of log2(10) * (interpolated table value), see CellArgs
    double *d_axT = nullptr, *d_axg = nullptr, *d_axmu = nullptr, *d_values = nullptr;
    // response
    bool have_rsp = false;
    int n_channel = 0, band_w = 0;
    int *d_first = nullptr, *d_elo = nullptr, *d_ehi = nullptr;
    double *d_band = nullptr, *d_tau = nullptr;
    // scratch (sub-batch sized)
    StarD* d_stars = nullptr; SpotD* d_spots = nullptr; RowD* d_rows = nullptr; int* d_cells = nullptr;
    double *d_lookup = nullptr, *d_tmpl = nullptr, *d_slices = nullptr, *d_partial = nullptr;
    double* d_llpart = nullptr; int* d_llbad = nullptr; int llpart_cap = 0;   // ln L slice sums [cap][kLLSplit]
    // host-variant staging
    double *d_params_stage = nullptr, *d_flux_stage = nullptr, *d_ll_stage = nullptr, *d_counts_stage = nullptr;
    int* d_status_stage = nullptr;
    size_t cells_smem = 0;
    // profiling (ppm_profile_enable / ppm_profile_read): CUDA event pairs around every launch
    bool prof_on = false;
    std::vector<cudaEvent_t> prof_ev;             // pool, two per recorded launch
    std::vector<int> prof_kid;                    // kernel id of each recorded launch
    size_t prof_used = 0;
    unsigned long long* d_pairs = nullptr;        // [0] (cell, phase) pairs with F_p != 0 walked by k_cells; [1] temperature-map
                                                  // mode: rows left to the full-width launch
    // device-resident sampler loop (ppm_chain_*)
    ChainArgs chain{};
    double* d_chain_box = nullptr;                // lo | hi | sigma [3][P]
    double* d_chain_beta = nullptr;
    const double *chain_data = nullptr, *chain_bkg = nullptr;
    double chain_exposure = 0.0;
    cudaGraphExec_t chain_graph = nullptr;
    int64_t chain_launches_per_step = 0;
    cudaStream_t chain_stream = nullptr;          // own stream when the context runs on the legacy default stream (which
    cudaEvent_t chain_ev = nullptr;               // cannot be captured); ordered with it through chain_ev
};

// kernel ids of ppm_profile_read
enum { KID_STAR = 0, KID_ROWS, KID_LOOKUP, KID_TEMPLATE, KID_SLICE, KID_CELLS, KID_REDUCE, KID_FOLD, KID_LOGLIKE, KID_N };

static void prof_begin(ppm_ctx* c, int kid)
{
    if (!c->prof_on) return;
    if (c->prof_used + 2 > c->prof_ev.size()) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { c->prof_on = false; return; }
        c->prof_ev.push_back(a); c->prof_ev.push_back(b);
    }
    c->prof_kid.push_back(kid);
    cudaEventRecord(c->prof_ev[c->prof_used], c->stream);
}
static void prof_end(ppm_ctx* c)
{
    if (!c->prof_on) return;
    cudaEventRecord(c->prof_ev[c->prof_used + 1], c->stream);
    c->prof_used += 2;
}

extern "C" const char* ppm_last_error(void) { return g_err; }

static void chain_free(ppm_ctx* c)
{
    if (c->chain_graph) { cudaGraphExecDestroy(c->chain_graph); c->chain_graph = nullptr; }
    if (c->chain_stream) { cudaStreamSynchronize(c->chain_stream); cudaStreamDestroy(c->chain_stream); c->chain_stream = nullptr; }
    if (c->chain_ev) { cudaEventDestroy(c->chain_ev); c->chain_ev = nullptr; }
    void* ptrs[] = {c->chain.cur, c->chain.prop, c->chain.ll, c->chain.llp, c->chain.oob, c->chain.accepted, c->chain.swapped,
                    c->chain.t, c->d_chain_box, c->d_chain_beta};
    for (void* p : ptrs) if (p) cudaFree(p);
    c->chain = ChainArgs{};
    c->d_chain_box = nullptr; c->d_chain_beta = nullptr;
}

extern "C" int ppm_destroy(ppm_ctx* c)
{
    if (!c) return PPM_OK;
    cudaSetDevice(c->cfg.device);
    chain_free(c);
    void* ptrs[] = {c->d_en, c->d_uef, c->d_axT, c->d_axg, c->d_axmu, c->d_values, c->d_first, c->d_elo,
                    c->d_ehi, c->d_band, c->d_tau, c->d_stars, c->d_spots, c->d_rows, c->d_cells, c->d_lookup,
                    c->d_tmpl, c->d_slices, c->d_partial, c->d_params_stage, c->d_flux_stage,
                    c->d_ll_stage, c->d_counts_stage, c->d_status_stage};
    for (void* p : ptrs) if (p) cudaFree(p);
    if (c->d_pairs) cudaFree(c->d_pairs);
    if (c->d_llpart) cudaFree(c->d_llpart);
    if (c->d_llbad) cudaFree(c->d_llbad);
    for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
    delete c;
    return PPM_OK;
}

static void choose_map4_tiling(ppm_ctx* c, const std::vector<double>& ue);

// dynamic shared memory of the table cell kernels for `npl` nodes per lane (ppm_cells.cuh / ppm_cells32.cuh layouts)
static size_t cells_tab_smem(const ppm_ctx* c, int nmu, int nx, int npl)
{
    const size_t tmpl = 4 * (size_t)(c->n_fp + 1) + nmu + 16;            // + UG (first energy of each lane group)
    if (c->cfg.precision == 1)
        return sizeof(double) * (tmpl + (size_t)c->nw * (2 * 32 * npl + 64 + 64 + 16)) + sizeof(float) * ((size_t)nmu * nx + 32 * npl + 32);   // tail pad: out-of-window node reads stay inside
    return sizeof(double) * ((size_t)nmu * nx + tmpl + (size_t)c->nw * (4 * 32 * npl + 3 * 64 + 32));
}

// vectors per sub-batch: the per-launch scratch (row slices of `slice_doubles` doubles, templates, cell lists, lookup
// series, partial tiles) stays under the context's budget (ppm_config.scratch_mb)
static int compute_sb(const ppm_ctx* c, size_t slice_doubles)
{
    const ppm_config& g = c->cfg;
    const double budget = (g.scratch_mb > 0 ? (double)g.scratch_mb : 1536.0) * 1048576.0;
    const double per_row = (double)g.n_phase * g.n_energy * 8.0;
    const double per_vec = (double)c->nchunk * per_row +
                           (double)c->RT * ((double)slice_doubles * 8.0 + 4.0 * (c->n_fp + 1) * 8.0 + g.n_phi * 4.0 +
                                            2.0 * kNCheb * 8.0 + (double)sizeof(RowD));
    int sb = (int)std::max(1.0, std::min((double)g.max_batch, std::floor(budget / per_vec)));
    return std::min(sb, 65535 / std::max(1, (g.n_energy + 31) / 32));      // grid.z limit with the smallest energy tile
}

static void free_scratch(ppm_ctx* c)
{
    if (c->chain_graph) { cudaGraphExecDestroy(c->chain_graph); c->chain_graph = nullptr; }   // captured pointers go stale
    void** ptrs[] = {(void**)&c->d_stars, (void**)&c->d_spots, (void**)&c->d_rows, (void**)&c->d_cells, (void**)&c->d_lookup,
                     (void**)&c->d_tmpl, (void**)&c->d_partial, (void**)&c->d_pairs, (void**)&c->d_slices,
                     (void**)&c->d_flux_stage, (void**)&c->d_counts_stage};
    for (void** p : ptrs) { if (*p) cudaFree(*p); *p = nullptr; }
}

static int alloc_scratch(ppm_ctx* c)
{
    const ppm_config& g = c->cfg;
    const size_t rows = (size_t)c->SB * c->RT;
    int rc;
    if ((rc = dev_alloc(&c->d_stars, (size_t)c->SB))) return rc;
    if ((rc = dev_alloc(&c->d_spots, (size_t)c->SB * g.n_spots))) return rc;
    if ((rc = dev_alloc(&c->d_rows, rows))) return rc;
    if ((rc = dev_alloc(&c->d_cells, rows * g.n_phi))) return rc;
    if ((rc = dev_alloc(&c->d_lookup, rows * 2 * kNCheb))) return rc;
    if ((rc = dev_alloc(&c->d_tmpl, rows * 4 * (c->n_fp + 1)))) return rc;
    if ((rc = dev_alloc(&c->d_partial, (size_t)c->SB * c->nchunk * g.n_phase * g.n_energy))) return rc;
    if ((rc = dev_alloc(&c->d_pairs, (size_t)2))) return rc;
    if (cudaMemsetAsync(c->d_pairs, 0, 2 * sizeof(unsigned long long), c->stream) != cudaSuccess) return PPM_ERR_CUDA;
    return PPM_OK;
}

extern "C" int ppm_create(const ppm_config* cfg, const double* energies, void* stream, ppm_ctx** out)
{
    ARG(cfg && energies && out, "null pointer");
    ARG(cfg->n_spots >= 1 && cfg->n_spots <= PPM_MAX_SPOTS, "n_spots must be 1..4");
    ARG(cfg->n_theta >= 1 && cfg->n_phi >= 1 && cfg->n_phase >= 1 && cfg->n_energy >= 1, "grid sizes must be >= 1");
    ARG(cfg->n_fp >= 0, "n_fp must be >= 0");
    ARG(cfg->n_phi <= 12000, "n_phi must be <= 12000");
    ARG(cfg->emission >= 0 && cfg->emission <= 4, "emission must be 0 .. 4");
    ARG(cfg->precision == 0 || cfg->precision == 1, "precision must be 0 (fp64) or 1 (fp32 interpolation + exponential)");
    ARG(cfg->precision == 0 || cfg->emission != PPM_EMISSION_BLACKBODY, "precision = 1 applies to table emission only");
    ARG(cfg->max_batch >= 1, "max_batch must be >= 1");
    ARG(cfg->beaming >= 0 && cfg->beaming <= 2, "beaming must be 0, 1 or 2");
    ARG(cfg->beaming == 0 || cfg->emission == PPM_EMISSION_BLACKBODY, "beaming laws apply to blackbody emission only");
    ARG(cfg->mesh == 0 || cfg->mesh == 1, "mesh must be 0 (theta x phi box per spot) or 1 (HEALPix rings)");
    ARG(cfg->mesh == 0 || (cfg->n_phi % 4 == 0 && cfg->n_theta == cfg->n_phi - 1),
        "HEALPix mesh: n_phi = 4 N_side and n_theta = 4 N_side - 1");
    ARG(cfg->scratch_mb >= 0, "scratch_mb must be >= 0");
    ARG(cfg->phase_interp == 0 || cfg->phase_interp == 1 || cfg->phase_interp == 3, "phase_interp must be 0 / 1 (linear) or 3");
    ARG(cfg->interp_domain == 0 || cfg->interp_domain == 1, "interp_domain must be 0 (log10 I/T^3) or 1 (I/T^3)");
    ARG(cfg->interp_domain == 0 || (cfg->emission != PPM_EMISSION_BLACKBODY && cfg->precision == 0),
        "interp_domain = 1 applies to table emission with precision = 0");
    for (int e = 0; e < cfg->n_energy; ++e) {
        ARG(std::isfinite(energies[e]) && energies[e] > 0.0, "energies must be finite and > 0");
        if (e) ARG(energies[e] > energies[e - 1], "energies must be strictly increasing");
    }
    int ndev = 0;
    CK(cudaGetDeviceCount(&ndev));
    if (cfg->device < 0 || cfg->device >= ndev) { set_err("no CUDA device %d (found %d)", cfg->device, ndev); return PPM_ERR_CUDA; }
    CK(cudaSetDevice(cfg->device));
    ppm_ctx* c = new (std::nothrow) ppm_ctx;
    if (!c) { set_err("out of host memory"); return PPM_ERR_NOMEM; }
    c->cfg = *cfg;
    // strategy b = strategy a + clipping of negative intensities; I = T^3 10^v > 0 when the logarithm is interpolated
    if (cfg->emission == PPM_EMISSION_TABLE_CUBIC_CLIP && cfg->interp_domain == 0) c->cfg.emission = PPM_EMISSION_TABLE_CUBIC;
    c->stream = (cudaStream_t)stream;
    c->P = 8 + 8 * cfg->n_spots;
    c->RT = cfg->n_spots * cfg->n_theta;
    c->n_fp = cfg->n_fp > 0 ? cfg->n_fp : std::max(192, 2 * cfg->n_phase);           // reading R2
    c->h_en.assign(energies, energies + cfg->n_energy);
    // launch geometry of the cell kernel
    // 16 warps x 128 registers fill the register file; 32 warps x 64 registers measured slower (profiles/r1d_k_cells_tab_T_full.md)
    c->nw = std::min(16, cfg->n_phase);
    c->npg = (cfg->n_phase + c->nw - 1) / c->nw;
    const int need = (cfg->n_energy + 31) / 32;
    const int epls[] = {1, 2, 4, 5, 8, 10};
    c->epl = 10;
    for (int v : epls) if (v >= need) { c->epl = v; break; }
    c->n_etile = (cfg->n_energy + 32 * c->epl - 1) / (32 * c->epl);
    const double per_row = (double)cfg->n_phase * cfg->n_energy * 8.0;
    c->rows_per_chunk = 1;
    while ((double)((c->RT + c->rows_per_chunk - 1) / c->rows_per_chunk) * per_row > 96.0e6 && c->rows_per_chunk < c->RT)
        c->rows_per_chunk *= 2;
    c->nchunk = (c->RT + c->rows_per_chunk - 1) / c->rows_per_chunk;
    // sub-batch: keep the per-launch scratch inside the budget; table emission re-sizes it in ppm_load_atmosphere
    // once the slice size is known (blackbody emission has no slices)
    c->SB = compute_sb(c, 0);
    int rc = alloc_scratch(c);
    if (rc) { ppm_destroy(c); return rc; }
    // energy-derived constants: filled here for blackbody; refreshed by ppm_load_atmosphere (needs h)
    if ((rc = dev_alloc(&c->d_en, (size_t)cfg->n_energy)) || (rc = dev_alloc(&c->d_uef, (size_t)cfg->n_energy))) {
        ppm_destroy(c);
        return rc;
    }
    double glx[kNGL], glw[kNGL];
    gauss_legendre(kNGL, glx, glw);
    cudaError_t e = cudaMemcpyAsync(c->d_en, energies, sizeof(double) * cfg->n_energy, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyToSymbolAsync(c_glx, glx, sizeof(glx), 0, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyToSymbolAsync(c_glw, glw, sizeof(glw), 0, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) {
        set_err("ppm_create: %s", cudaGetErrorString(e));
        ppm_destroy(c);
        return PPM_ERR_CUDA;
    }
    *out = c;
    return PPM_OK;
}

extern "C" int ppm_n_fp(const ppm_ctx* c) { return c ? c->n_fp : 0; }
extern "C" int ppm_sub_batch(const ppm_ctx* c) { return c ? c->SB : 0; }
extern "C" int ppm_uniform_energy(const ppm_ctx* c) { return (c && c->uniform_e) ? 1 : 0; }
extern "C" int64_t ppm_launch_count(const ppm_ctx* c) { return c ? c->launches : 0; }

extern "C" int ppm_load_atmosphere(ppm_ctx* c, const double* logT, int nT, const double* logg, int ng,
                                   const double* mu, int nmu, const double* logx, int nx, const double* values,
                                   int values_on_device)
{
    ARG(c && logT && logg && mu && logx && values, "null pointer");
    ARG(nT >= 4 && ng >= 4 && nmu >= 4 && nx >= 4, "every table axis needs >= 4 nodes");
    ARG(nx <= 256 && (size_t)nmu * nx <= 32767, "the cell kernel packs stencil indices: nx <= 256 and nmu * nx <= 32767");
    const double* axs[4] = {logT, logg, mu, logx};
    const int ns[4] = {nT, ng, nmu, nx};
    for (int a = 0; a < 4; ++a)
        for (int i = 1; i < ns[a]; ++i) ARG(axs[a][i] > axs[a][i - 1], "table axes must be strictly increasing");
    const double h = (logx[nx - 1] - logx[0]) / (nx - 1);
    for (int i = 0; i < nx; ++i)
        ARG(std::fabs(logx[i] - (logx[0] + h * i)) <= 1e-10 * std::fabs(h), "logx axis must be uniformly spaced");
    CK(cudaSetDevice(c->cfg.device));
    for (double** p : {&c->d_axT, &c->d_axg, &c->d_axmu, &c->d_values, &c->d_slices}) { if (*p) cudaFree(*p); *p = nullptr; }
    c->have_atm = false;
    int rc;
    {   // the sub-batch follows the actual slice size (nmu x nx doubles per row)
        const int sb = compute_sb(c, (size_t)nmu * nx);
        if (sb != c->SB) {
            CK(cudaStreamSynchronize(c->stream));
            free_scratch(c);
            c->SB = sb;
            if ((rc = alloc_scratch(c))) return rc;
        }
    }
    const size_t nval = (size_t)nT * ng * nmu * nx;
    if ((rc = dev_alloc(&c->d_axT, (size_t)nT)) || (rc = dev_alloc(&c->d_axg, (size_t)ng)) ||
        (rc = dev_alloc(&c->d_axmu, (size_t)nmu)) || (rc = dev_alloc(&c->d_values, nval)) ||
        (rc = dev_alloc(&c->d_slices, (size_t)c->SB * c->RT * nmu * nx))) return rc;
    CK(cudaMemcpyAsync(c->d_axT, logT, sizeof(double) * nT, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_axg, logg, sizeof(double) * ng, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_axmu, mu, sizeof(double) * nmu, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_values, values, sizeof(double) * nval,
                       values_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    c->nT = nT; c->ng = ng; c->nmu = nmu; c->nx = nx; c->x0 = logx[0]; c->hx = h;
    {   // range of the table -> bound of every interpolated value.  Lagrange weights can leave [0, 1]: the sum of their
        // magnitudes is <= 1.25 per uniform cubic axis and stays below 2 on the non-uniform mu axis, so an interpolated value
        // lies within (1.25^3 * 2 - 1) / 2 < 1.5 table ranges of [vmin, vmax]; 2 ranges are taken.
        std::vector<double> hv;
        const double* v = values;
        if (values_on_device) {
            hv.resize(nval);
            CK(cudaMemcpy(hv.data(), values, sizeof(double) * nval, cudaMemcpyDeviceToHost));
            v = hv.data();
        }
        double vmin = v[0], vmax = v[0];
        for (size_t i = 0; i < nval; ++i) {
            ARG(std::isfinite(v[i]), "table values must be finite");
            vmin = std::min(vmin, v[i]); vmax = std::max(vmax, v[i]);
        }
        const double range = vmax - vmin;
        c->y_lo = kLog2_10 * (vmin - 2.0 * range);
        c->y_hi = kLog2_10 * (vmax + 2.0 * range);
    }
    std::vector<double> ue(c->cfg.n_energy);
    for (int e = 0; e < c->cfg.n_energy; ++e) ue[e] = std::log10(c->h_en[e]) / h;
    std::vector<long long> uef(c->cfg.n_energy);
    for (int e = 0; e < c->cfg.n_energy; ++e) {
        ARG(std::fabs(ue[e]) < 1000.0, "energies are too far outside the table's log10(E/kT) range");
        uef[e] = llrintl((long double)ue[e] * 4503599627370496.0L);
    }
    CK(cudaMemcpyAsync(c->d_uef, uef.data(), sizeof(long long) * uef.size(), cudaMemcpyHostToDevice, c->stream));
    // Energy tiling of the table cell kernel: the most energies per lane (fewest per-pair passes) whose per-warp window
    // of logx intervals still fits the 227 KB of shared memory beside the row slice and the template.
    {
        const int need = (c->cfg.n_energy + 31) / 32;
        const int epls[] = {10, 8, 5, 4, 2, 1};                     // descending
        int vbest = 10;                                             // smallest option that covers all energies in one tile
        for (int v : epls) if (v >= need) vbest = v;
        bool found = false;
        for (int v : epls) {
            if (v > vbest) continue;
            const int ntile = (c->cfg.n_energy + 32 * v - 1) / (32 * v);
            int wmax = 1;
            for (int t = 0; t < ntile; ++t) {
                const int ea = t * 32 * v, eb = std::min(c->cfg.n_energy, ea + 32 * v) - 1;
                wmax = std::max(wmax, std::min(nx - 1, (int)std::floor(ue[eb] - ue[ea]) + 3));
            }
            int npl = 1;
            while (32 * npl - 3 < wmax) npl += 2;                   // odd: conflict-free strided shared-memory accesses
            const size_t smem = cells_tab_smem(c, nmu, nx, npl);
            if (smem <= 227 * 1024 && npl <= 9) {
                c->epl = v; c->n_etile = ntile; c->wmax = wmax; c->npl = npl;
                found = true;
                break;
            }
        }
        if (!found) {
            set_err("table (%d x %d) + template (n_fp = %d) do not fit the cell kernel's shared memory", nmu, nx, c->n_fp);
            return PPM_ERR_ARG;
        }
        // Log-uniform energy grid?  Then energy e0 + lane + 32 i of a tile is evaluated at uef[e0 + lane] + i * step32 (see
        // EnergyCoord in ppm_cells.cuh).  Taken only if that affine form is within 256 units of 2^-52 table intervals of
        // every energy's own coordinate and only the last group of every tile is ragged.
        c->uniform_e = false; c->uef_step = 0;
        const int nE = c->cfg.n_energy;
        if (nE > 32 && c->epl >= 2) {
            const long long step32 = llrintl(32.0L * (long double)(uef[nE - 1] - uef[0]) / (long double)(nE - 1));
            bool ok = step32 > 0;
            for (int t = 0; t < c->n_etile && ok; ++t) {
                const int ea = t * 32 * c->epl, nt = std::min(nE, ea + 32 * c->epl) - ea;
                if (nt <= 32 * (c->epl - 1)) ok = false;            // more than the last group would be ragged
                for (int k = 0; k < nt && ok; ++k) {
                    const long long dev = uef[ea + k] - (uef[ea + (k & 31)] + (long long)(k >> 5) * step32);
                    if (dev > 256 || dev < -256) ok = false;
                }
            }
            if (ok) { c->uniform_e = true; c->uef_step = step32; }
        }
        choose_map4_tiling(c, ue);
    }
    CK(cudaStreamSynchronize(c->stream));
    c->have_atm = true;
    return PPM_OK;
}

extern "C" int ppm_set_response(ppm_ctx* c, int n_channel, int band_w, const int32_t* first_chan,
                                const double* rsp_band, int on_device, const double* tau_ref)
{
    ARG(c && first_chan && rsp_band && tau_ref, "null pointer");
    ARG(n_channel >= 1 && band_w >= 1, "n_channel and band_w must be >= 1");
    const int nE = c->cfg.n_energy;
    CK(cudaSetDevice(c->cfg.device));
    for (void** p : {(void**)&c->d_first, (void**)&c->d_elo, (void**)&c->d_ehi, (void**)&c->d_band, (void**)&c->d_tau,
                     (void**)&c->d_counts_stage}) { if (*p) cudaFree(*p); *p = nullptr; }
    c->have_rsp = false;
    // per channel: smallest range [e_lo, e_hi) containing every energy whose band covers it
    std::vector<int> elo(n_channel, nE), ehi(n_channel, 0);
    for (int e = 0; e < nE; ++e)
        for (int w = 0; w < band_w; ++w) {
            const long ch = (long)first_chan[e] + w;
            if (ch < 0 || ch >= n_channel) continue;
            elo[ch] = std::min(elo[ch], e);
            ehi[ch] = std::max(ehi[ch], e + 1);
        }
    for (int ch = 0; ch < n_channel; ++ch) if (elo[ch] > ehi[ch]) elo[ch] = ehi[ch] = 0;
    int rc;
    if ((rc = dev_alloc(&c->d_first, (size_t)nE)) || (rc = dev_alloc(&c->d_elo, (size_t)n_channel)) ||
        (rc = dev_alloc(&c->d_ehi, (size_t)n_channel)) || (rc = dev_alloc(&c->d_band, (size_t)nE * band_w)) ||
        (rc = dev_alloc(&c->d_tau, (size_t)nE))) return rc;
    CK(cudaMemcpyAsync(c->d_first, first_chan, sizeof(int) * nE, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_elo, elo.data(), sizeof(int) * n_channel, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_ehi, ehi.data(), sizeof(int) * n_channel, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_band, rsp_band, sizeof(double) * nE * band_w,
                       on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_tau, tau_ref, sizeof(double) * nE, cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    c->n_channel = n_channel; c->band_w = band_w;
    c->have_rsp = true;
    return PPM_OK;
}

// ------------------------------------------------------------------------------------------------
// evaluation
// ------------------------------------------------------------------------------------------------
static LaunchShape shape_of(const ppm_ctx* c, dim3 grid, int threads, size_t smem, int epl, int npl)
{
    LaunchShape L;
    L.stream = c->stream; L.grid = grid; L.threads = threads; L.smem = smem; L.epl = epl; L.npl = npl;
    return L;
}

// the uniform-temperature cell kernel of the context's mode (launch_*.cu)
static int dispatch_cells(ppm_ctx* c, bool table, const CellArgs& a, dim3 grid, int threads, size_t smem)
{
    const LaunchShape L = shape_of(c, grid, threads, smem, c->epl, c->npl);
    if (!table) CK(launch_cells_bb(L, a));
    else if (c->cfg.interp_domain == 1) CK(launch_cells_lin(L, a));
    else if (c->cfg.precision == 1) CK(launch_cells_tab32(L, a));
    else CK(launch_cells_tab(L, a));
    return PPM_OK;
}

// shared memory of k_cells_map with `nw` warps (ppm_cells_map.cuh layout)
static size_t cells_map_smem(const ppm_ctx* c, int nw, int wst)
{
    return sizeof(double) * ((size_t)nw * (4 * 32 * c->npl + 5 * 64 + 32) + 2 * (size_t)c->nmu * wst +
                             4 * (size_t)(c->n_fp + 1) + c->nmu + c->nT + 16);
}

// shared memory of k_cells_map4 with `nw` warps, `npl` nodes per lane and slices of `wst` columns (ppm_cells_map4.cuh layout)
static size_t cells_map4_smem(const ppm_ctx* c, int nw, int npl, int wst)
{
    return sizeof(double) * ((size_t)nw * (4 * 32 * npl + 5 * 64 + 32) + 4 * (size_t)c->nmu * wst +
                             4 * (size_t)(c->n_fp + 1) + c->nmu + c->nT + 16);
}

// Tiling of k_cells_map4 (temperature maps under the cubic-in-log-T strategies): the most energies per lane, then the
// most warps, for which four slices wide enough for a tile's window (+ 20 columns for the row's z range, the log T
// interval and the stencil's reach) fit the 227 KB beside the warps' coefficient arrays.
static void choose_map4_tiling(ppm_ctx* c, const std::vector<double>& ue)
{
    c->m4_epl = c->m4_ntile = c->m4_npl = c->m4_nw = c->m4_wst = 0;
    const int nE = c->cfg.n_energy, need = (nE + 31) / 32;
    const int epls[] = {10, 8, 5, 4, 2, 1};
    int vbest = 10;
    for (int v : epls) if (v >= need) vbest = v;
    for (int v : epls) {
        if (v > vbest) continue;
        const int ntile = (nE + 32 * v - 1) / (32 * v);
        int wmax = 1;
        for (int t = 0; t < ntile; ++t) {
            const int ea = t * 32 * v, eb = std::min(nE, ea + 32 * v) - 1;
            wmax = std::max(wmax, std::min(c->nx - 1, (int)std::floor(ue[eb] - ue[ea]) + 3));
        }
        int npl = 1;
        while (32 * npl - 3 < wmax) npl += 2;
        if (npl > 3) continue;
        for (int nw : {16, 8, 4}) {
            if (nw > std::max(4, c->cfg.n_phase)) continue;
            const long budget = 227 * 1024 / 8 - (long)(cells_map4_smem(c, nw, npl, 0) / 8);
            const int wst = (int)std::min<long>(c->nx, budget > 0 ? budget / (4 * c->nmu) : 0);
            if (wst >= std::min(c->nx, wmax + 20)) {
                c->m4_epl = v; c->m4_ntile = ntile; c->m4_npl = npl; c->m4_nw = nw; c->m4_wst = wst;
                return;
            }
        }
    }
}

// shared memory of k_cells_map32 (ppm_cells_map32.cuh layout; the tail pad keeps out-of-window node reads inside)
static size_t cells_map32_smem(const ppm_ctx* c, int nw)
{
    return sizeof(double) * ((size_t)nw * (2 * 32 * c->npl + 3 * 64 + 16) + 4 * (size_t)(c->n_fp + 1) + c->nmu + c->nT + 1) +
           sizeof(float) * (2 * (size_t)c->nmu * c->nx + 32 * c->npl + 32);
}


static int evaluate_sub(ppm_ctx* c, const double* params_dev, int nb, double* flux_dev, int32_t* status_dev,
                        const double* tmap_dev = nullptr)
{
    const ppm_config& g = c->cfg;
    const bool table = g.emission != PPM_EMISSION_BLACKBODY;
    GeoArgs G;
    G.params = params_dev; G.nb = nb; G.P = c->P; G.n_spots = g.n_spots; G.n_theta = g.n_theta; G.n_phi = g.n_phi;
    G.n_phase = g.n_phase; G.n_fp = c->n_fp; G.oblate = g.oblate; G.emission = g.emission; G.mesh = g.mesh;
    G.stars = c->d_stars; G.spots = c->d_spots; G.rows = c->d_rows; G.cells = c->d_cells;
    G.lookup = c->d_lookup; G.tmpl = c->d_tmpl;
    G.axT = c->d_axT; G.nT = c->nT; G.axg = c->d_axg; G.ng = c->ng;
    G.tmap = tmap_dev;
    const int rows = nb * c->RT;
    prof_begin(c, KID_STAR);
    k_star<<<(nb + 63) / 64, 64, 0, c->stream>>>(G);
    prof_end(c);
    prof_begin(c, KID_ROWS);
    k_rows<<<rows, 128, tmap_dev ? sizeof(int) * (size_t)g.n_phi : 0, c->stream>>>(G);
    prof_end(c);
    prof_begin(c, KID_LOOKUP);
    k_lookup<<<rows, kNCheb * kNGL, 0, c->stream>>>(G);
    prof_end(c);
    const size_t tsm = sizeof(double) * (2 * kNCheb + 4 * (size_t)(c->n_fp + 1));
    if (tsm > 48 * 1024) CK(cudaFuncSetAttribute(k_template, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tsm));
    prof_begin(c, KID_TEMPLATE);
    k_template<<<rows, 128, tsm, c->stream>>>(G);
    prof_end(c);
    c->launches += 4;
    if (table && !tmap_dev) {
        SliceArgs S;
        S.spots = c->d_spots; S.rows = c->d_rows; S.values = c->d_values; S.slices = c->d_slices;
        S.n_theta = g.n_theta; S.nT = c->nT; S.ng = c->ng; S.nmu = c->nmu; S.nx = c->nx; S.domain = g.interp_domain;
        dim3 sg((c->nmu * c->nx + 255) / 256, rows);
        prof_begin(c, KID_SLICE);
        k_slice<<<sg, 256, 0, c->stream>>>(S);
        prof_end(c);
        c->launches += 1;
    }
    CellArgs A{};
    A.stars = c->d_stars; A.spots = c->d_spots; A.rows = c->d_rows; A.cells = c->d_cells; A.tmpl = c->d_tmpl;
    A.slices = c->d_slices; A.axmu = c->d_axmu; A.uef = c->d_uef; A.en = c->d_en;
    A.uniform_e = (table && c->uniform_e) ? 1 : 0; A.uef_step = c->uef_step;
    A.partial = c->d_partial; A.pairs = c->d_pairs;
    A.x0_over_h = table ? c->x0 / c->hx : 0.0; A.inv_h = table ? 1.0 / c->hx : 0.0;
    A.nb = nb; A.RT = c->RT; A.n_spots = g.n_spots; A.n_theta = g.n_theta; A.n_phi = g.n_phi; A.n_phase = g.n_phase;
    A.n_fp = c->n_fp; A.nE = g.n_energy;
    A.nmu = table ? c->nmu : 0; A.nx = table ? c->nx : 0;
    const bool cubic_all = g.emission == PPM_EMISSION_TABLE_CUBIC || g.emission == PPM_EMISSION_TABLE_CUBIC_CLIP;   // a, b
    A.mu_rule = cubic_all ? AX_CUBIC_SHIFT : AX_MU_PROTECTED;
    A.x_linedge = cubic_all ? 0 : 1;
    A.t_rule = tg_rule(g.emission);
    A.clip = (g.interp_domain == 1 && g.emission == PPM_EMISSION_TABLE_CUBIC_CLIP) ? 1 : 0;
    A.nchunk = c->nchunk; A.rows_per_chunk = c->rows_per_chunk; A.nw = c->nw; A.n_etile = c->n_etile; A.mesh = g.mesh; A.beaming = g.beaming;
    A.phase_order = g.phase_interp == 3 ? 3 : 1; A.y_lo = c->y_lo; A.y_hi = c->y_hi;
    const size_t smem = table ? cells_tab_smem(c, c->nmu, c->nx, c->npl) : sizeof(double) * 4 * (size_t)(c->n_fp + 1);
    if (smem > 227 * 1024) { set_err("cell kernel needs %zu bytes of shared memory (> 227 KB)", smem); return PPM_ERR_ARG; }
    int rc;
    if (tmap_dev && g.emission != PPM_EMISSION_TABLE_MIXED) {
        // temperature-map mode under the strategies that are cubic in log T: four windowed node slices, own energy tiling
        A.tmap = tmap_dev; A.values = c->d_values; A.axT = c->d_axT; A.nT = c->nT; A.ng = c->ng;
        A.nw = c->m4_nw; A.n_etile = c->m4_ntile; A.wst = c->m4_wst; A.map_split = 0; A.uniform_e = 0;
        dim3 grid(c->nchunk, (g.n_phase + c->m4_nw - 1) / c->m4_nw, nb * c->m4_ntile);
        const size_t sm4 = cells_map4_smem(c, c->m4_nw, c->m4_npl, c->m4_wst);
        prof_begin(c, KID_CELLS);
        { const cudaError_t le = launch_cells_map4(shape_of(c, grid, c->m4_nw * 32, sm4, c->m4_epl, c->m4_npl), A, c->d_stars); CK(le); rc = PPM_OK; }
        c->launches += 1;
    } else if (tmap_dev && g.precision == 1) {
        // temperature-map mode with FP32 interpolation: two full-width FP32 node slices, 16 warps, one launch
        A.tmap = tmap_dev; A.values = c->d_values; A.axT = c->d_axT; A.nT = c->nT; A.ng = c->ng;
        A.map_split = 0; A.uniform_e = 0;
        const size_t sm32 = cells_map32_smem(c, c->nw);
        if (sm32 > 227 * 1024) { set_err("temperature-map mode (precision = 1): table and template do not fit in shared memory"); return PPM_ERR_ARG; }
        dim3 grid(c->nchunk, c->npg, nb * c->n_etile);
        prof_begin(c, KID_CELLS);
        { const cudaError_t le = launch_cells_map32(shape_of(c, grid, c->nw * 32, sm32, c->epl, c->npl), A, c->d_stars); CK(le); rc = PPM_OK; }
        c->launches += 1;
    } else if (tmap_dev) {
        // temperature-map mode: two FP64 log T node slices in shared memory.  Full-width slices leave room for 8 warps;
        // slices cut to the logx columns a row's interval can reach (wst columns) leave room for 16.  Both kernels are
        // launched, each row is taken by the windowed one if all its intervals fit wst columns, else by the full-width one.
        A.tmap = tmap_dev; A.values = c->d_values; A.axT = c->d_axT; A.nT = c->nT; A.ng = c->ng;
        int nwm = 0;
        for (int v : {8, 6, 4, 2, 1}) if (cells_map_smem(c, v, c->nx) <= 227 * 1024) { nwm = v; break; }
        if (!nwm) { set_err("temperature-map mode: table and template do not fit in shared memory"); return PPM_ERR_ARG; }
        nwm = std::min(nwm, g.n_phase);
        int wst = 0;
        if (g.n_phase >= 16) {
            const long budget = 227 * 1024 / 8 - (long)cells_map_smem(c, 16, 0) / 8;
            wst = (int)std::min<long>(c->nx, budget > 0 ? budget / (2 * c->nmu) : 0);
            if (wst < c->wmax + 12 || wst >= c->nx) wst = 0;                       // too narrow to be useful / nothing to gain
        }
        A.wst = wst; A.map_split = wst ? 1 : 0;
        prof_begin(c, KID_CELLS);
        rc = PPM_OK;
        if (wst) {
            CK(cudaMemsetAsync(c->d_pairs + 1, 0, sizeof(unsigned long long), c->stream));
            CellArgs W = A;
            W.nw = 16;
            dim3 gridw(c->nchunk, (g.n_phase + 15) / 16, nb * c->n_etile);
            const size_t smw = cells_map_smem(c, 16, wst);
            { const cudaError_t le = launch_cells_map(shape_of(c, gridw, 512, smw, c->epl, c->npl), W, true); CK(le); rc = PPM_OK; }
            c->launches += 1;
        }
        if (!rc) {
            A.nw = nwm;
            dim3 grid(c->nchunk, (g.n_phase + nwm - 1) / nwm, nb * c->n_etile);
            const size_t smem_map = cells_map_smem(c, nwm, c->nx);
            { const cudaError_t le = launch_cells_map(shape_of(c, grid, nwm * 32, smem_map, c->epl, c->npl), A, false); CK(le); rc = PPM_OK; }
        }
    } else {
        dim3 grid(c->nchunk, c->npg, nb * c->n_etile);
        prof_begin(c, KID_CELLS);
        rc = dispatch_cells(c, table, A, grid, c->nw * 32, smem);
    }
    prof_end(c);
    if (rc) return rc;
    const int n_out = g.n_phase * g.n_energy;
    dim3 rg((n_out + 255) / 256, nb);
    prof_begin(c, KID_REDUCE);
    k_reduce<<<rg, 256, 0, c->stream>>>(c->d_partial, c->d_stars, c->nchunk, n_out, flux_dev, status_dev);
    prof_end(c);
    c->launches += 2;
    CK(cudaGetLastError());
    c->last_nb = nb;
    return PPM_OK;
}

extern "C" int ppm_evaluate(ppm_ctx* c, const double* params_dev, int B, double* flux_dev, int32_t* status_dev)
{
    ARG(c, "null context");
    ARG(B >= 0, "B must be >= 0");
    if (B == 0) return PPM_OK;                                   // empty batch: nothing to do, pointers may be NULL
    ARG(params_dev && flux_dev, "null pointer");
    if (B > c->cfg.max_batch) { set_err("B = %d exceeds max_batch = %d", B, c->cfg.max_batch); return PPM_ERR_BATCH; }
    if (c->cfg.emission != PPM_EMISSION_BLACKBODY && !c->have_atm) {
        set_err("table emission requested but no atmosphere loaded"); return PPM_ERR_STATE;
    }
    CK(cudaSetDevice(c->cfg.device));
    const size_t fstride = (size_t)c->cfg.n_phase * c->cfg.n_energy;
    for (int b0 = 0; b0 < B; b0 += c->SB) {
        const int nb = std::min(c->SB, B - b0);
        int rc = evaluate_sub(c, params_dev + (size_t)b0 * c->P, nb, flux_dev + (size_t)b0 * fstride,
                              status_dev ? status_dev + b0 : nullptr);
        if (rc) return rc;
    }
    return PPM_OK;
}

extern "C" int ppm_evaluate_map(ppm_ctx* c, const double* params_dev, const double* logT_map_dev, int B, double* flux_dev,
                                int32_t* status_dev)
{
    ARG(c, "null context");
    ARG(B >= 0, "B must be >= 0");
    if (B == 0) return PPM_OK;
    ARG(params_dev && logT_map_dev && flux_dev, "null pointer");
    if (B > c->cfg.max_batch) { set_err("B = %d exceeds max_batch = %d", B, c->cfg.max_batch); return PPM_ERR_BATCH; }
    if (c->cfg.emission == PPM_EMISSION_BLACKBODY || c->cfg.interp_domain != 0 ||
        (c->cfg.precision != 0 && c->cfg.emission != PPM_EMISSION_TABLE_MIXED)) {
        set_err("temperature maps need table emission (1-4) and interp_domain = 0; precision = 1 only with emission = 2");
        return PPM_ERR_STATE;
    }
    if (!c->have_atm) { set_err("table emission requested but no atmosphere loaded"); return PPM_ERR_STATE; }
    if (c->nT > 64) { set_err("temperature maps support at most 64 log T nodes"); return PPM_ERR_STATE; }
    if (c->cfg.emission != PPM_EMISSION_TABLE_MIXED && !c->m4_epl) {
        set_err("temperature maps under strategies a-c: four log T node slices do not fit shared memory for this table / energy grid");
        return PPM_ERR_STATE;
    }
    CK(cudaSetDevice(c->cfg.device));
    const size_t fstride = (size_t)c->cfg.n_phase * c->cfg.n_energy;
    const size_t mstride = (size_t)c->RT * c->cfg.n_phi;
    for (int b0 = 0; b0 < B; b0 += c->SB) {
        const int nb = std::min(c->SB, B - b0);
        int rc = evaluate_sub(c, params_dev + (size_t)b0 * c->P, nb, flux_dev + (size_t)b0 * fstride,
                              status_dev ? status_dev + b0 : nullptr, logT_map_dev + (size_t)b0 * mstride);
        if (rc) return rc;
    }
    return PPM_OK;
}

extern "C" int ppm_fold_response(ppm_ctx* c, const double* flux_dev, const double* params_dev, int B, double* counts_dev)
{
    ARG(c, "null context");
    ARG(B >= 0, "B must be >= 0");
    if (B == 0) return PPM_OK;
    ARG(flux_dev && params_dev && counts_dev, "null pointer");
    if (B > c->cfg.max_batch) { set_err("B = %d exceeds max_batch = %d", B, c->cfg.max_batch); return PPM_ERR_BATCH; }
    if (!c->have_rsp) { set_err("no response set"); return PPM_ERR_STATE; }
    if (B == 0) return PPM_OK;
    CK(cudaSetDevice(c->cfg.device));
    FoldArgs F;
    F.flux = flux_dev; F.params = params_dev; F.band = c->d_band; F.tau = c->d_tau; F.first = c->d_first;
    F.e_lo = c->d_elo; F.e_hi = c->d_ehi; F.counts = counts_dev;
    F.P = c->P; F.n_phase = c->cfg.n_phase; F.nE = c->cfg.n_energy; F.n_channel = c->n_channel; F.band_w = c->band_w;
    const size_t smem = sizeof(double) * c->cfg.n_energy;
    if (smem > 48 * 1024) CK(cudaFuncSetAttribute(k_fold, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    for (int b0 = 0; b0 < B; b0 += 65535) {
        const int nb = std::min(65535, B - b0);
        FoldArgs Fs = F;
        Fs.flux = flux_dev + (size_t)b0 * F.n_phase * F.nE;
        Fs.params = params_dev + (size_t)b0 * F.P;
        Fs.counts = counts_dev + (size_t)b0 * F.n_phase * F.n_channel;
        dim3 grid((c->n_channel + 127) / 128, c->cfg.n_phase, nb);
        prof_begin(c, KID_FOLD);
        k_fold<<<grid, 128, smem, c->stream>>>(Fs);
        prof_end(c);
        c->launches += 1;
    }
    CK(cudaGetLastError());
    return PPM_OK;
}

extern "C" int ppm_loglike(ppm_ctx* c, const double* counts_dev, int B, const double* data_dev, const double* bkg_dev,
                           double exposure_s, double* loglike_dev)
{
    ARG(c, "null context");
    ARG(B >= 0, "B must be >= 0");
    if (B == 0) return PPM_OK;
    ARG(counts_dev && data_dev && loglike_dev, "null pointer");
    if (B > c->cfg.max_batch) { set_err("B = %d exceeds max_batch = %d", B, c->cfg.max_batch); return PPM_ERR_BATCH; }
    if (!c->have_rsp) { set_err("no response set"); return PPM_ERR_STATE; }
    if (B == 0) return PPM_OK;
    CK(cudaSetDevice(c->cfg.device));
    prof_begin(c, KID_LOGLIKE);
    for (int b0 = 0; b0 < B; b0 += 32768) {
        const int nb = std::min(32768, B - b0);
        if (!c->d_llpart || c->llpart_cap < nb + 1) {
            if (c->d_llpart) cudaFree(c->d_llpart);
            if (c->d_llbad) cudaFree(c->d_llbad);
            c->d_llpart = nullptr; c->d_llbad = nullptr;
            int rc;
            if ((rc = dev_alloc(&c->d_llpart, (size_t)(nb + 1) * kLLSplit)) || (rc = dev_alloc(&c->d_llbad, (size_t)(nb + 1) * kLLSplit)))
                return rc;
            c->llpart_cap = nb + 1;
        }
        dim3 grid(kLLSplit, nb + 1);
        k_loglike_part<<<grid, 256, 0, c->stream>>>(counts_dev + (size_t)b0 * c->cfg.n_phase * c->n_channel, data_dev, bkg_dev,
                                                    c->cfg.n_phase, c->n_channel, exposure_s, nb, c->d_llpart, c->d_llbad);
        k_loglike_final<<<(nb + 127) / 128, 128, 0, c->stream>>>(c->d_llpart, c->d_llbad, nb, loglike_dev + b0);
    }
    prof_end(c);
    c->launches += 2;
    CK(cudaGetLastError());
    return PPM_OK;
}

// ------------------------------------------------------------------------------------------------
// host-buffer variants (copies inside the call)
// ------------------------------------------------------------------------------------------------
static int ensure_stage(ppm_ctx* c)
{
    int rc;
    const size_t mb = (size_t)c->cfg.max_batch;
    if (!c->d_params_stage && (rc = dev_alloc(&c->d_params_stage, mb * c->P))) return rc;
    if (!c->d_status_stage && (rc = dev_alloc(&c->d_status_stage, mb))) return rc;
    if (!c->d_ll_stage && (rc = dev_alloc(&c->d_ll_stage, mb))) return rc;
    return PPM_OK;
}

extern "C" int ppm_evaluate_host(ppm_ctx* c, const double* params_host, int B, double* flux_host, int32_t* status_host)
{
    ARG(c, "null context");
    ARG(B >= 0, "B must be >= 0");
    if (B == 0) return PPM_OK;
    ARG(params_host && flux_host, "null pointer");
    if (B > c->cfg.max_batch) { set_err("B = %d exceeds max_batch = %d", B, c->cfg.max_batch); return PPM_ERR_BATCH; }
    CK(cudaSetDevice(c->cfg.device));
    int rc = ensure_stage(c);
    if (rc) return rc;
    const size_t fstride = (size_t)c->cfg.n_phase * c->cfg.n_energy;
    if (!c->d_flux_stage && (rc = dev_alloc(&c->d_flux_stage, (size_t)c->SB * fstride))) return rc;
    CK(cudaMemcpyAsync(c->d_params_stage, params_host, sizeof(double) * B * c->P, cudaMemcpyHostToDevice, c->stream));
    if (c->cfg.emission != PPM_EMISSION_BLACKBODY && !c->have_atm) {
        set_err("table emission requested but no atmosphere loaded"); return PPM_ERR_STATE;
    }
    for (int b0 = 0; b0 < B; b0 += c->SB) {
        const int nb = std::min(c->SB, B - b0);
        rc = evaluate_sub(c, c->d_params_stage + (size_t)b0 * c->P, nb, c->d_flux_stage, c->d_status_stage + b0);
        if (rc) return rc;
        CK(cudaMemcpyAsync(flux_host + (size_t)b0 * fstride, c->d_flux_stage, sizeof(double) * nb * fstride,
                           cudaMemcpyDeviceToHost, c->stream));
    }
    if (status_host)
        CK(cudaMemcpyAsync(status_host, c->d_status_stage, sizeof(int32_t) * B, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return PPM_OK;
}

extern "C" int ppm_loglike_host(ppm_ctx* c, const double* params_host, int B, const double* data_dev,
                                const double* bkg_dev, double exposure_s, double* loglike_host, int32_t* status_host)
{
    ARG(c, "null context");
    ARG(B >= 0, "B must be >= 0");
    if (B == 0) return PPM_OK;
    ARG(params_host && data_dev && loglike_host, "null pointer");
    if (B > c->cfg.max_batch) { set_err("B = %d exceeds max_batch = %d", B, c->cfg.max_batch); return PPM_ERR_BATCH; }
    if (!c->have_rsp) { set_err("no response set"); return PPM_ERR_STATE; }
    if (c->cfg.emission != PPM_EMISSION_BLACKBODY && !c->have_atm) {
        set_err("table emission requested but no atmosphere loaded"); return PPM_ERR_STATE;
    }
    CK(cudaSetDevice(c->cfg.device));
    int rc = ensure_stage(c);
    if (rc) return rc;
    const size_t fstride = (size_t)c->cfg.n_phase * c->cfg.n_energy;
    const size_t cstride = (size_t)c->cfg.n_phase * c->n_channel;
    if (!c->d_flux_stage && (rc = dev_alloc(&c->d_flux_stage, (size_t)c->SB * fstride))) return rc;
    if (!c->d_counts_stage && (rc = dev_alloc(&c->d_counts_stage, (size_t)c->SB * cstride))) return rc;
    CK(cudaMemcpyAsync(c->d_params_stage, params_host, sizeof(double) * B * c->P, cudaMemcpyHostToDevice, c->stream));
    for (int b0 = 0; b0 < B; b0 += c->SB) {
        const int nb = std::min(c->SB, B - b0);
        const double* pd = c->d_params_stage + (size_t)b0 * c->P;
        if ((rc = evaluate_sub(c, pd, nb, c->d_flux_stage, c->d_status_stage + b0))) return rc;
        if ((rc = ppm_fold_response(c, c->d_flux_stage, pd, nb, c->d_counts_stage))) return rc;
        if ((rc = ppm_loglike(c, c->d_counts_stage, nb, data_dev, bkg_dev, exposure_s, c->d_ll_stage + b0))) return rc;
    }
    CK(cudaMemcpyAsync(loglike_host, c->d_ll_stage, sizeof(double) * B, cudaMemcpyDeviceToHost, c->stream));
    if (status_host)
        CK(cudaMemcpyAsync(status_host, c->d_status_stage, sizeof(int32_t) * B, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return PPM_OK;
}

// ------------------------------------------------------------------------------------------------
// device-resident sampler loop (ppm_chain.cuh)
// ------------------------------------------------------------------------------------------------
// ln L of `n` parameter vectors that sit in device memory, into ll_dev: S0..S7 in sub-batches, nothing leaves the device
static int loglike_resident(ppm_ctx* c, const double* params_dev, int n, double* ll_dev)
{
    for (int b0 = 0; b0 < n; b0 += c->SB) {
        const int nb = std::min(c->SB, n - b0);
        const double* pd = params_dev + (size_t)b0 * c->P;
        int rc;
        if ((rc = evaluate_sub(c, pd, nb, c->d_flux_stage, c->d_status_stage + b0))) return rc;
        if ((rc = ppm_fold_response(c, c->d_flux_stage, pd, nb, c->d_counts_stage))) return rc;
        if ((rc = ppm_loglike(c, c->d_counts_stage, nb, c->chain_data, c->chain_bkg, c->chain_exposure, ll_dev + b0))) return rc;
    }
    return PPM_OK;
}

extern "C" int ppm_chain_create(ppm_ctx* c, int W, const double* params0, const double* lo, const double* hi,
                                const double* sigma, const double* beta, uint64_t seed, const double* data_dev,
                                const double* bkg_dev, double exposure_s)
{
    ARG(c, "null context");
    ARG(params0 && lo && hi && sigma && data_dev, "null pointer");
    ARG(W >= 1 && W <= c->cfg.max_batch, "n_walkers must be in 1 .. max_batch");
    if (!c->have_rsp) { set_err("no response set"); return PPM_ERR_STATE; }
    if (c->cfg.emission != PPM_EMISSION_BLACKBODY && !c->have_atm) {
        set_err("table emission requested but no atmosphere loaded"); return PPM_ERR_STATE;
    }
    const int P = c->P;
    for (int k = 0; k < P; ++k) ARG(sigma[k] >= 0.0 && (sigma[k] == 0.0 || lo[k] <= hi[k]), "sigma must be >= 0 and lo <= hi");
    CK(cudaSetDevice(c->cfg.device));
    CK(cudaStreamSynchronize(c->stream));
    chain_free(c);
    int rc = ensure_stage(c);
    if (rc) return rc;
    const size_t fstride = (size_t)c->cfg.n_phase * c->cfg.n_energy, cstride = (size_t)c->cfg.n_phase * c->n_channel;
    if (!c->d_flux_stage && (rc = dev_alloc(&c->d_flux_stage, (size_t)c->SB * fstride))) return rc;
    if (!c->d_counts_stage && (rc = dev_alloc(&c->d_counts_stage, (size_t)c->SB * cstride))) return rc;
    ChainArgs& A = c->chain;
    if ((rc = dev_alloc(&A.cur, (size_t)W * P)) || (rc = dev_alloc(&A.prop, (size_t)W * P)) || (rc = dev_alloc(&A.ll, (size_t)W)) ||
        (rc = dev_alloc(&A.llp, (size_t)W)) || (rc = dev_alloc(&A.oob, (size_t)W)) || (rc = dev_alloc(&A.accepted, (size_t)W)) ||
        (rc = dev_alloc(&A.swapped, (size_t)W)) || (rc = dev_alloc(&A.t, (size_t)1)) ||
        (rc = dev_alloc(&c->d_chain_box, (size_t)3 * P)) || (rc = dev_alloc(&c->d_chain_beta, (size_t)W))) {
        chain_free(c);
        return rc;
    }
    std::vector<double> bt(W, 1.0);
    if (beta) bt.assign(beta, beta + W);
    cudaError_t e = cudaMemcpyAsync(A.cur, params0, sizeof(double) * W * P, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_chain_box, lo, sizeof(double) * P, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_chain_box + P, hi, sizeof(double) * P, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_chain_box + 2 * P, sigma, sizeof(double) * P, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_chain_beta, bt.data(), sizeof(double) * W, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A.accepted, 0, sizeof(long long) * W, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A.swapped, 0, sizeof(long long) * W, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A.t, 0, sizeof(unsigned long long), c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(A.oob, 0, sizeof(int) * W, c->stream);
    if (e != cudaSuccess) { set_err("ppm_chain_create: %s", cudaGetErrorString(e)); chain_free(c); return PPM_ERR_CUDA; }
    A.lo = c->d_chain_box; A.hi = c->d_chain_box + P; A.sigma = c->d_chain_box + 2 * P; A.beta = c->d_chain_beta;
    A.seed = seed; A.W = W; A.P = P;
    c->chain_data = data_dev; c->chain_bkg = bkg_dev; c->chain_exposure = exposure_s;
    if ((rc = loglike_resident(c, A.cur, W, A.ll))) { chain_free(c); return rc; }     // ln L of the starting states (also warms
    CK(cudaStreamSynchronize(c->stream));                                               // every lazy allocation before a capture)
    return PPM_OK;
}

static int chain_enqueue_step(ppm_ctx* c)
{
    const ChainArgs& A = c->chain;
    const int blocks = (A.W + 127) / 128;
    k_chain_propose<<<blocks, 128, 0, c->stream>>>(A);
    int rc = loglike_resident(c, A.prop, A.W, A.llp);
    if (rc) return rc;
    k_chain_accept<<<blocks, 128, 0, c->stream>>>(A);
    k_chain_swap<<<1, 256, 0, c->stream>>>(A);
    c->launches += 3;
    return PPM_OK;
}

extern "C" int ppm_chain_run(ppm_ctx* c, int n_steps)
{
    ARG(c, "null context");
    ARG(n_steps >= 0, "n_steps must be >= 0");
    if (!c->chain.cur) { set_err("no chain: call ppm_chain_create first"); return PPM_ERR_STATE; }
    CK(cudaSetDevice(c->cfg.device));
    if (n_steps == 0) return PPM_OK;
    if (!c->stream && !c->chain_stream) {                            // the legacy default stream cannot be captured
        CK(cudaStreamCreateWithFlags(&c->chain_stream, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&c->chain_ev, cudaEventDisableTiming));
    }
    cudaStream_t user = c->stream, run = c->stream ? c->stream : c->chain_stream;
    if (!c->chain_graph) {
        const bool prof = c->prof_on;
        c->prof_on = false;                                          // no event records inside the captured step
        const int64_t l0 = c->launches;
        cudaGraph_t graph = nullptr;
        CK(cudaStreamBeginCapture(run, cudaStreamCaptureModeThreadLocal));
        c->stream = run;
        const int rc = chain_enqueue_step(c);
        c->stream = user;
        cudaError_t e = cudaStreamEndCapture(run, &graph);
        c->prof_on = prof;
        c->chain_launches_per_step = c->launches - l0;
        c->launches = l0;
        if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
        if (e != cudaSuccess) { set_err("capture of the sampler step failed: %s", cudaGetErrorString(e)); return PPM_ERR_CUDA; }
        e = cudaGraphInstantiate(&c->chain_graph, graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) { c->chain_graph = nullptr; set_err("cudaGraphInstantiate: %s", cudaGetErrorString(e)); return PPM_ERR_CUDA; }
    }
    if (run != user) {                                               // after whatever the context's stream holds ...
        CK(cudaEventRecord(c->chain_ev, user));
        CK(cudaStreamWaitEvent(run, c->chain_ev, 0));
    }
    for (int i = 0; i < n_steps; ++i) CK(cudaGraphLaunch(c->chain_graph, run));
    if (run != user) {                                               // ... and before whatever it receives next
        CK(cudaEventRecord(c->chain_ev, run));
        CK(cudaStreamWaitEvent(user, c->chain_ev, 0));
    }
    c->launches += (int64_t)n_steps * c->chain_launches_per_step;
    return PPM_OK;
}

extern "C" int ppm_chain_read(ppm_ctx* c, double* params, double* loglike, int64_t* accepted, int64_t* swapped, int64_t* steps)
{
    ARG(c, "null context");
    if (!c->chain.cur) { set_err("no chain: call ppm_chain_create first"); return PPM_ERR_STATE; }
    CK(cudaSetDevice(c->cfg.device));
    if (c->chain_stream) CK(cudaStreamSynchronize(c->chain_stream));
    CK(cudaStreamSynchronize(c->stream));
    const ChainArgs& A = c->chain;
    if (params) CK(cudaMemcpy(params, A.cur, sizeof(double) * A.W * A.P, cudaMemcpyDeviceToHost));
    if (loglike) CK(cudaMemcpy(loglike, A.ll, sizeof(double) * A.W, cudaMemcpyDeviceToHost));
    if (accepted) CK(cudaMemcpy(accepted, A.accepted, sizeof(long long) * A.W, cudaMemcpyDeviceToHost));
    if (swapped) CK(cudaMemcpy(swapped, A.swapped, sizeof(long long) * A.W, cudaMemcpyDeviceToHost));
    if (steps) { unsigned long long t = 0; CK(cudaMemcpy(&t, A.t, sizeof(t), cudaMemcpyDeviceToHost)); *steps = (int64_t)t; }
    return PPM_OK;
}

// ------------------------------------------------------------------------------------------------
// introspection (tests) and the FP64 peak probe
// ------------------------------------------------------------------------------------------------
static int debug_check(ppm_ctx* c, int b)
{
    ARG(c, "null context");
    if (b < 0 || b >= c->last_nb) {
        set_err("vector %d is not in the last evaluated sub-batch (size %d)", b, c->last_nb);
        return PPM_ERR_ARG;
    }
    CK(cudaSetDevice(c->cfg.device));
    CK(cudaStreamSynchronize(c->stream));
    return PPM_OK;
}

extern "C" int ppm_debug_rows(ppm_ctx* c, int b, double* out)
{
    int rc = debug_check(c, b);
    if (rc) return rc;
    ARG(out, "null pointer");
    std::vector<RowD> h(c->RT);
    CK(cudaMemcpy(h.data(), c->d_rows + (size_t)b * c->RT, sizeof(RowD) * c->RT, cudaMemcpyDeviceToHost));
    for (int r = 0; r < c->RT; ++r) {
        const RowD& q = h[r];
        const double v[16] = {q.theta, q.dcos, q.R, q.u, q.f, q.coseta, q.sineta, q.beta, q.gamma, q.log10g, q.c_dt,
                              q.dOmega, q.alpha_max, q.psi_max, (double)q.n_active, (double)q.visible};
        std::memcpy(out + (size_t)r * 16, v, sizeof(v));
    }
    return PPM_OK;
}

extern "C" int ppm_debug_mask(ppm_ctx* c, int b, uint8_t* out)
{
    int rc = debug_check(c, b);
    if (rc) return rc;
    ARG(out, "null pointer");
    const int nphi = c->cfg.n_phi;
    std::vector<RowD> h(c->RT);
    std::vector<int> cl((size_t)c->RT * nphi);
    CK(cudaMemcpy(h.data(), c->d_rows + (size_t)b * c->RT, sizeof(RowD) * c->RT, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(cl.data(), c->d_cells + (size_t)b * c->RT * nphi, sizeof(int) * cl.size(), cudaMemcpyDeviceToHost));
    std::memset(out, 0, (size_t)c->RT * nphi);
    for (int r = 0; r < c->RT; ++r)
        for (int i = 0; i < h[r].n_active; ++i) out[(size_t)r * nphi + (cl[(size_t)r * nphi + i] & 0xFFFF)] = 1;
    return PPM_OK;
}

extern "C" int ppm_debug_template(ppm_ctx* c, int b, double* out)
{
    int rc = debug_check(c, b);
    if (rc) return rc;
    ARG(out, "null pointer");
    const size_t n1 = (size_t)c->n_fp + 1, per = 4 * n1;
    std::vector<RowD> h(c->RT);
    CK(cudaMemcpy(h.data(), c->d_rows + (size_t)b * c->RT, sizeof(RowD) * c->RT, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(out, c->d_tmpl + (size_t)b * c->RT * per, sizeof(double) * c->RT * per, cudaMemcpyDeviceToHost));
    for (int r = 0; r < c->RT; ++r)                      // rows that were skipped hold stale scratch: report zeros
        if (h[r].n_active == 0) std::memset(out + (size_t)r * per, 0, sizeof(double) * per);
    return PPM_OK;
}

extern "C" int ppm_debug_lookup(ppm_ctx* c, int b, int row, const double* alpha, int n, double* psi, double* dpsi,
                                double* lag)
{
    int rc = debug_check(c, b);
    if (rc) return rc;
    ARG(alpha && psi && dpsi && lag && n >= 1, "null pointer or n < 1");
    ARG(row >= 0 && row < c->RT, "row out of range");
    RowD h;
    CK(cudaMemcpy(&h, c->d_rows + (size_t)b * c->RT + row, sizeof(RowD), cudaMemcpyDeviceToHost));
    if (h.n_active == 0) { set_err("row %d has no active cell: no lookup was built", row); return PPM_ERR_STATE; }
    double* d = nullptr;
    if ((rc = dev_alloc(&d, (size_t)4 * n))) return rc;
    cudaError_t e = cudaMemcpy(d, alpha, sizeof(double) * n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_lookup_eval<<<(n + 127) / 128, 128, 0, c->stream>>>(c->d_lookup + ((size_t)b * c->RT + row) * 2 * kNCheb,
                                                              h.alpha_max, d, n, d + n, d + 2 * n, d + 3 * n);
        c->launches += 1;
        e = cudaStreamSynchronize(c->stream);
    }
    if (e == cudaSuccess) e = cudaMemcpy(psi, d + n, sizeof(double) * n, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(dpsi, d + 2 * n, sizeof(double) * n, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(lag, d + 3 * n, sizeof(double) * n, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) { set_err("ppm_debug_lookup: %s", cudaGetErrorString(e)); return PPM_ERR_CUDA; }
    return PPM_OK;
}

extern "C" int ppm_profile_enable(ppm_ctx* c, int on)
{
    ARG(c, "null context");
    CK(cudaSetDevice(c->cfg.device));
    CK(cudaStreamSynchronize(c->stream));
    c->prof_on = on != 0;
    c->prof_used = 0;
    c->prof_kid.clear();
    CK(cudaMemsetAsync(c->d_pairs, 0, sizeof(unsigned long long), c->stream));
    return PPM_OK;
}

extern "C" int ppm_profile_read(ppm_ctx* c, double* ms, int64_t* launches, double* triples)
{
    ARG(c && ms && launches && triples, "null pointer");
    CK(cudaSetDevice(c->cfg.device));
    CK(cudaStreamSynchronize(c->stream));
    for (int i = 0; i < KID_N; ++i) { ms[i] = 0.0; launches[i] = 0; }
    for (size_t i = 0; i < c->prof_kid.size() && 2 * i + 1 < c->prof_used; ++i) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
        ms[c->prof_kid[i]] += (double)t;
        launches[c->prof_kid[i]] += (c->prof_kid[i] == KID_LOGLIKE) ? 2 : 1;
    }
    unsigned long long pairs = 0;
    CK(cudaMemcpy(&pairs, c->d_pairs, sizeof(pairs), cudaMemcpyDeviceToHost));
    *triples = (double)pairs * (double)c->cfg.n_energy;
    return PPM_OK;
}

extern "C" int ppm_measure_fp64_peak(int device, double* flops_per_s)
{
    ARG(flops_per_s, "null pointer");
    CK(cudaSetDevice(device));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, device));
    double* d = nullptr;
    int rc = dev_alloc(&d, (size_t)1);
    if (rc) return rc;
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 4096;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        CK(cudaEventRecord(e0, 0));
        k_dfma_peak<<<blocks, threads>>>(d, iters, 1.0 + rep);
        CK(cudaEventRecord(e1, 0));
        CK(cudaEventSynchronize(e1));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        const double fl = (double)blocks * threads * 8.0 * 8.0 * iters * 2.0 / (ms * 1.0e-3);
        if (rep > 0 && fl > best) best = fl;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    *flops_per_s = best;
    return PPM_OK;
}
