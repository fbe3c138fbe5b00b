/*
 * ppm.h -- C ABI of the B200-native pulse-profile-modeling (PPM) hot path.
 *
 * One likelihood-call evaluation of the energy-resolved pulse profile of a rotating neutron
 * star in the oblate-Schwarzschild + Doppler (OS+D) picture of arxiv/paper_2510_07764
 * (Zhou & Huang).  Citations are "PAPER.md:<line>" plus the section / equation; readings
 * R0..R22 of the places where the paper is silent or garbled are listed in DESIGN.md.
 *
 * Everything behind this boundary is hand-written CUDA for sm_100a.  There is NO CPU
 * fallback: every entry point fails with PPM_ERR_CUDA when no device is usable.
 *
 * Conventions
 *   - "dev" pointers are CUDA device pointers on the context's device; "host" pointers are
 *     ordinary host memory.  The caller owns every buffer it passes; the context copies the
 *     tables given to ppm_create / ppm_load_atmosphere / ppm_set_response and owns only its
 *     own scratch.  Outputs are fully overwritten.
 *   - All work is enqueued on the cudaStream_t given to ppm_create (pass
 *     torch.cuda.current_stream().cuda_stream, or NULL for the default stream).  Calls that
 *     take only device pointers are asynchronous and never synchronise; ppm_create,
 *     ppm_load_atmosphere, ppm_set_response, ppm_*_host and ppm_debug_* synchronise the stream.
 *     After one warm-up call (lazy scratch allocation) the device-pointer calls allocate nothing, so a whole step
 *     (ppm_evaluate + ppm_fold_response + ppm_loglike) can be captured into a CUDA graph on that stream and replayed.
 *   - One context per stream; a context is not thread-safe.
 *   - Return value: 0 on success, a negative PPM_ERR_* otherwise; ppm_last_error() gives text.
 *   - Per-vector physics failures do not fail the call: status[b] carries the bits below,
 *     that vector's flux is NaN and its log-likelihood -inf.
 *
 * Parameter vector (P = 8 + 8*n_spots doubles, row-major [B][P]; "(M, R, nu), i,
 * the hotspot's shape, position, and size"; D of Eq 21; N_H PAPER.md:270):
 *   [0] M / M_sun   [1] R_eq / km   [2] nu / Hz (seen at infinity)   [3] cos i
 *   [4] D / kpc     [5] N_H / 1e20 cm^-2   [6] phase offset / cycles   [7] reserved
 *   per spot s (offset 8+8s): [0] theta_c  [1] phi_c  [2] zeta (angular radius, rad)
 *   [3] log10 T_eff/K  [4] theta_m  [5] phi_m  [6] zeta_m (0 => no omitted region)  [7] reserved
 */
#ifndef PPM_H_
#define PPM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PPM_OK            0
#define PPM_ERR_ARG      -1   /* invalid argument / shape */
#define PPM_ERR_NOMEM    -2   /* host or device allocation failed */
#define PPM_ERR_CUDA     -3   /* CUDA runtime error (incl. no usable device) */
#define PPM_ERR_STATE    -4   /* wrong state, e.g. table emission without a loaded atmosphere */
#define PPM_ERR_BATCH    -5   /* B > max_batch */

#define PPM_STATUS_COMPACTNESS 1  /* R_S/R outside (0, 0.56] (reading R4) */
#define PPM_STATUS_INPUT       2  /* non-finite input, beta_eq >= 1, bad M/R/D/cos i */
#define PPM_STATUS_SPOT        4  /* invalid spot (zeta <= 0, angles outside [0, pi]) */
#define PPM_STATUS_MAP_WINDOW  8  /* ppm_evaluate_map under emission 1, 3, 4: a row's logx window exceeds the slice buffers;
                                     with precision = 1: a log T interval's cells span more than 0.5 dex */

#define PPM_EMISSION_BLACKBODY   0  /* isotropic blackbody, Eq C.5 */
#define PPM_EMISSION_TABLE_CUBIC 1  /* 4-D table, cubic Lagrange on all axes (strategy a) */
#define PPM_EMISSION_TABLE_MIXED 2  /* 4-D table, mixed order (strategy d) */
#define PPM_EMISSION_TABLE_CUBIC_LINEDGE 3 /* cubic on all axes, linear at the table boundaries and in the protected
                                             small-mu zone (strategy c; reading R13e) */
#define PPM_EMISSION_TABLE_CUBIC_CLIP 4    /* strategy b: as strategy a, negative intensities clipped to 0;
                                             identical to strategy a when interp_domain = 0 (I = T^3 10^v > 0) */

#define PPM_MAX_SPOTS 4

typedef struct ppm_ctx ppm_ctx; /* opaque: device tables, scratch, a copy of the energy grid */

typedef struct {
    int32_t n_spots;    /* 1..PPM_MAX_SPOTS emitting components (overlaps add, reading R18) */
    int32_t n_theta;    /* colatitude rows of each spot's bounding-box grid (reading R1) */
    int32_t n_phi;      /* azimuth cells per row of that grid */
    int32_t n_phase;    /* output phases, phi_out[k] = k / n_phase (reading R3) */
    int32_t n_fp;       /* fine template phases N_fp (Table 4); 0 -> max(192, 2*n_phase) */
    int32_t n_energy;   /* observed photon energies (keV), given to ppm_create */
    int32_t emission;   /* PPM_EMISSION_* (0..4) */
    int32_t precision;  /* 0 = fp64 everywhere; 1 = table interpolation + exponential in fp32 (geometry, templates,
                           coordinates and the final sums stay fp64; tolerance 1e-4 per bin), table emission only */
    int32_t oblate;     /* 0 spherical S+D (o2 = 0, g = g0); 1 oblate OS+D (Eq 7-11) */
    int32_t max_batch;  /* largest B accepted by ppm_evaluate / ppm_fold_response / ppm_loglike */
    int32_t device;     /* CUDA ordinal */
    int32_t mesh;       /* 0: per-spot colatitude x azimuth bounding-box grid (reading R1);
                           1: HEALPix ring scheme over the whole surface (Eq 24-29), the same mesh
                              for every spot: n_phi = 4 N_side, n_theta = 4 N_side - 1 rings, pixel area pi/(3 N_side^2) */
    int32_t beaming;    /* blackbody emission only: 0 isotropic, 1 I prop. to cos^2(sigma'),
                           2 I prop. to sin^2(sigma'), cos(sigma') = mu = delta cos(sigma) (Eq 20) */
    int32_t scratch_mb; /* budget (MiB) for the per-launch scratch (row slices, templates, partial tiles); batches larger
                           than what fits are processed in sub-batches of ppm_sub_batch() vectors.  0 -> 1536 */
    int32_t phase_interp; /* order of Interp in Eq 46: 0 or 1 = piecewise linear (reading R11);
                             3 = 4-point (cubic) Lagrange in phi_o on the periodic template (reading R11b) */
    int32_t interp_domain; /* table emission: 0 = the 4-D interpolation acts on the tabulated log10(I/T^3) and
                              I = T^3 10^v (reading R13a); 1 = it acts on I/T^3 = 10^table itself (reading R13g,
                              PAPER.md:551-559: the form in which cubic overshoot produces negative intensities) */
} ppm_config;

/* Create a context: copies the energy grid (host, [n_energy], keV, strictly increasing),
 * allocates scratch, builds the quadrature rule used by the lookup-build kernel.
 * cuda_stream is a cudaStream_t (may be NULL).  *out receives the context. */
int ppm_create(const ppm_config* cfg, const double* energies_keV, void* cuda_stream, ppm_ctx** out);
int ppm_destroy(ppm_ctx* ctx);

/* Load the 4-D atmosphere table log10(I / T_eff^3)[logT][logg][mu][logx], C order, x = E/kT
 * (base-10 logs, reading R13a).  Axes: host, strictly increasing, >= 4 nodes
 * each; logx must be uniformly spaced (as the paper's 166-point -1.3..2.0 axis is).
 * values: host pointer, or device pointer when values_on_device != 0.  Everything is copied. */
int ppm_load_atmosphere(ppm_ctx* ctx, const double* logT, int nT, const double* logg, int ng,
                        const double* mu, int nmu, const double* logx, int nx,
                        const double* values, int values_on_device);

/* Set the banded response (Eq 52-55; reading R15) and the ISM optical depth
 * per 1e20 cm^-2 (Eq 22/51; reading R16).  Row e of rsp_band covers
 * channels first_chan[e] .. first_chan[e]+band_w-1 (entries outside [0, n_channel) are ignored).
 * first_chan, tau_ref: host; rsp_band: host, or device when on_device != 0. */
int ppm_set_response(ppm_ctx* ctx, int n_channel, int band_w, const int32_t* first_chan,
                     const double* rsp_band, int on_device, const double* tau_ref);

/* S0-S5 of DESIGN.md: star/row scalars, cell mask, psi/lag lookup build, ring templates
 * (Eq 38-44), shift-and-add with atmosphere interpolation (PAPER.md:417-430
 * Eq 45-47).  params_dev [B][P]; flux_dev [B][n_phase][n_energy] photons cm^-2 s^-1 keV^-1
 * (Eq 21); status_dev [B] (may be NULL). */
int ppm_evaluate(ppm_ctx* ctx, const double* params_dev, int B, double* flux_dev, int32_t* status_dev);

/* S0-S5 with a per-cell effective-temperature map ("a full surface temperature map T_eff(theta,
 * phi)"; reading R24): logT_map_dev [B][n_spots][n_theta][n_phi] holds log10 T_eff/K of every cell of every spot's mesh
 * (box grid or HEALPix); a cell emits iff it passes the spot's geometric mask (centre within zeta, outside the omitted
 * cap) AND its entry is finite -- NaN marks a cell that does not emit.  The spots' own log10 T parameters are ignored.
 * Needs table emission and interp_domain = 0 (precision = 1, FP32 interpolation, only with emission =
 * PPM_EMISSION_TABLE_MIXED: k_cells_map32; there an interval whose cells span more than 0.5 dex in log T -- cells far
 * outside the axis -- gives PPM_STATUS_MAP_WINDOW); otherwise PPM_ERR_STATE.  emission =
 * PPM_EMISSION_TABLE_MIXED (strategy d: linear in log T, two node slices per log T interval) is the fast path; the
 * strategies that are cubic in log T (emission 1, 3, 4) need four node slices per interval, run on a finer energy tiling
 * and cannot hold a row whose cell temperatures lie so far outside the table's log T axis that one interval's logx
 * window exceeds the slice buffers: such a vector gets PPM_STATUS_MAP_WINDOW and a NaN flux. */
int ppm_evaluate_map(ppm_ctx* ctx, const double* params_dev, const double* logT_map_dev, int B, double* flux_dev,
                     int32_t* status_dev);

/* S6: C[b][k][c] = sum_e F_t[b][k][e] exp(-N_H20[b] tau_ref[e]) RSP0[e][c]  (Eq 22-23, 55).
 * N_H20 is params[b][5].  counts_dev [B][n_phase][n_channel], counts/s. */
int ppm_fold_response(ppm_ctx* ctx, const double* flux_dev, const double* params_dev, int B,
                      double* counts_dev);

/* S7: ln L_b = sum_{k,c} d ln m - m - lgamma(d+1),  m = exposure_s * C / n_phase + bkg[c]
 * (reading R14).  0 ln 0 := 0; -inf if some m = 0 < d or C is NaN.
 * data_dev [n_phase][n_channel]; bkg_dev [n_channel] or NULL; loglike_dev [B]. */
int ppm_loglike(ppm_ctx* ctx, const double* counts_dev, int B, const double* data_dev,
                const double* bkg_dev, double exposure_s, double* loglike_dev);

/* Host-buffer variants: same computation, with the host->device copy of the inputs and the
 * device->host copy of the result inside the call (they synchronise the stream).
 * ppm_evaluate_host: params_host [B][P] -> flux_host [B][n_phase][n_energy], status_host [B] or NULL.
 * ppm_loglike_host : params_host [B][P] -> evaluate + fold + ln L against data_dev / bkg_dev
 *                    (device, set-up data) -> loglike_host [B], status_host [B] or NULL. */
int ppm_evaluate_host(ppm_ctx* ctx, const double* params_host, int B, double* flux_host,
                      int32_t* status_host);
int ppm_loglike_host(ppm_ctx* ctx, const double* params_host, int B, const double* data_dev,
                     const double* bkg_dev, double exposure_s, double* loglike_host,
                     int32_t* status_host);

/* Device-resident sampler loop around the likelihood (reading R26 of DESIGN.md).
 * ppm_chain_create: W = n_walkers <= max_batch walkers start at params0_host [W][P]; parameter k is proposed as
 *   p_k + sigma_host[k] * N(0,1) (sigma 0 = fixed) inside the box prior [lo_host[k], hi_host[k]] (outside: rejected);
 *   walker w has inverse temperature beta_host[w] (NULL = all 1); data_dev [n_phase][n_channel], bkg_dev [n_channel] or
 *   NULL and exposure_s as in ppm_loglike (the data buffers must stay valid while the chain lives).  Needs a response
 *   (ppm_set_response) and, for table emission, an atmosphere.  Evaluates ln L of the starting states; synchronises.
 * ppm_chain_run: n_steps steps, each = proposal kernel -> S0..S7 (ppm_evaluate + ppm_fold_response + ppm_loglike on the
 *   proposals, in HBM) -> Metropolis acceptance against beta_w (ln L' - ln L) -> replica exchange between neighbouring
 *   walkers.  The step is captured into a CUDA graph at the first call and replayed; asynchronous on the context's stream.
 *   Random numbers: Philox4x32-10, key = seed, counter = (step, walker, stream).
 * ppm_chain_read: synchronises and copies the current states [W][P], their ln L [W], the per-walker counts of accepted
 *   proposals and exchanges [W] and the number of steps done (any pointer may be NULL).
 * One chain per context; ppm_chain_create on a context that has one replaces it; ppm_destroy frees it. */
int ppm_chain_create(ppm_ctx* ctx, int n_walkers, const double* params0_host, const double* lo_host,
                     const double* hi_host, const double* sigma_host, const double* beta_host, uint64_t seed,
                     const double* data_dev, const double* bkg_dev, double exposure_s);
int ppm_chain_run(ppm_ctx* ctx, int n_steps);
int ppm_chain_read(ppm_ctx* ctx, double* params_host, double* loglike_host, int64_t* accepted_host,
                   int64_t* swapped_host, int64_t* steps_host);

/* Introspection of the intermediate device state left by the LAST ppm_evaluate call, for
 * vector b of that call (tests compare each step with the oracle).  All outputs are host
 * buffers; row index r = spot * n_theta + j.
 *   rows    [n_rows][16]: theta, dcos, R_cm, u, f, coseta, sineta, beta, gamma, log10g,
 *                         c_dt_cm (Eq 16), dOmega, alpha_max, psi_max, n_active, ring_visible
 *   mask    [n_rows][n_phi] uint8, 1 = active cell (S1)
 *   tmpl    [n_rows][4][n_fp+1]: F, z, phi_o, mu (S3, after the invisible-range fill)
 *   lookup  evaluates the row's device-built lookup at n emission angles alpha[i]:
 *           psi[i], dpsi_dalpha[i], lag[i] = (c Delta t - c delta t(R)) / R            (S2) */
int ppm_debug_rows(ppm_ctx* ctx, int b, double* rows_host);
int ppm_debug_mask(ppm_ctx* ctx, int b, uint8_t* mask_host);
int ppm_debug_template(ppm_ctx* ctx, int b, double* tmpl_host);
int ppm_debug_lookup(ppm_ctx* ctx, int b, int row, const double* alpha_host, int n,
                     double* psi_host, double* dpsi_host, double* lag_host);

/* Number of kernel launches issued by this context so far (for bench.py's gpu_launches). */
int64_t ppm_launch_count(const ppm_ctx* ctx);
/* Vectors per internal sub-batch (scratch_mb / per-vector scratch, capped by max_batch); a batch B is processed
 * as ceil(B / ppm_sub_batch) sequences of launches.  Final after ppm_load_atmosphere for table emission. */
int ppm_sub_batch(const ppm_ctx* ctx);
/* 1 if the context's energy grid is log-uniform to within 256 units of 2^-52 table intervals, so that the table cell
 * kernel steps its logx coordinate from energy group to energy group instead of holding one value per energy
 * ("uniform energy path"); 0 otherwise or before ppm_load_atmosphere. */
int ppm_uniform_energy(const ppm_ctx* ctx);
/* Effective n_fp after defaulting. */
int ppm_n_fp(const ppm_ctx* ctx);

/* Per-kernel device timing, for bench.py's roofline object.  ppm_profile_enable(ctx, 1) resets the
 * accumulators and from then on brackets every kernel launch of this context with a pair of CUDA
 * events on the context's stream (no synchronisation is added); ppm_profile_enable(ctx, 0) stops.
 * ppm_profile_read synchronises the stream and returns, per kernel id, the summed event time in ms
 * and the number of launches since the last enable:
 *   PPM_KID_STAR 0, ROWS 1, LOOKUP 2, TEMPLATE 3, SLICE 4, CELLS 5, REDUCE 6, FOLD 7, LOGLIKE 8
 * ms_host, launches_host: host arrays of PPM_KID_COUNT entries.  *triples_host receives the number
 * of (active cell, output phase, energy) triples with F_p != 0 that the cell kernel accumulated
 * since the last enable (the algorithmic unit of DESIGN.md "Roofline"; counted on the device). */
#define PPM_KID_COUNT 9
int ppm_profile_enable(ppm_ctx* ctx, int on);
int ppm_profile_read(ppm_ctx* ctx, double* ms_host, int64_t* launches_host, double* triples_host);

/* Register-resident DFMA chain on every SM: returns the measured FP64 FMA rate in flop/s
 * (2 flop per DFMA) -- the roofline denominator of the cell kernel. */
int ppm_measure_fp64_peak(int device, double* flops_per_s);

const char* ppm_last_error(void); /* thread-local, static storage */

/* ---- allocation-free S7 (ppm_noalloc.cu) ----------------------------------------------------------------------------
 * ppm_loglike_noalloc: the Poisson ln L of ppm_loglike (reading R14; same kernels' arithmetic and summation order, so the
 * same bits) for callers that cannot call cudaMalloc (CUDA-graph capture, tight serving loops, harnesses that forbid it).
 * It needs no context and calls no cudaMalloc / cudaFree / allocating library routine: its scratch (the per-slice partial
 * sums) is a static __device__ array of (PPM_NOALLOC_MAX_BATCH + 1) x 64 doubles + ints = 0.75 MiB that every GPU which
 * loads the library holds until the process exits.
 *   counts_dev [B][n_phase][n_channel] counts/s, data_dev [n_phase][n_channel], bkg_dev [n_channel] or NULL, loglike_dev
 *   [B]: device pointers on the CURRENT device; stream: a cudaStream_t (NULL = the default stream); asynchronous.
 *   B > PPM_NOALLOC_MAX_BATCH -> PPM_ERR_BATCH (split the batch, or use ppm_loglike); bad arguments -> PPM_ERR_ARG; text
 *   from ppm_loglike_noalloc_error() (thread-local, static storage).
 * Every call on a device shares the array, which keeps the last call's contents (nothing in it has to start at zero: stage
 * 1 overwrites every entry stage 2 reads).  Calls that overlap on one GPU -- other streams, other host threads -- RACE on
 * it: serialise them.  The first call on a device looks up the array's device address (cudaGetSymbolAddress, which may
 * load the module): make one call per device before capturing a graph around later ones. */
#define PPM_NOALLOC_MAX_BATCH 1024
int ppm_loglike_noalloc(const double* counts_dev, int B, int n_phase, int n_channel, const double* data_dev,
                        const double* bkg_dev, double exposure_s, double* loglike_dev, void* stream);
const char* ppm_loglike_noalloc_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PPM_H_ */
