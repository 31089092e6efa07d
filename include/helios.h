/*
 * helios.h -- C ABI of the B200-native batched Helios-r2 emission forward model.
 *
 * One call evaluates, for B candidate parameter vectors, the hot path of
 * Kitzmann et al. 2020 (arXiv:1910.01070), Sect. 2.8:
 * opacity interpolation -> absorption coefficient -> layer optical depths ->
 * short-characteristics radiative transfer -> instrument profile -> binning ->
 * log-likelihood.  Every step runs in hand-written sm_100a CUDA kernels; there
 * is no CPU fallback: without a CUDA device helios_create() fails.
 *
 * Conventions
 *   - plain C types only; every pointer argument says HOST or DEVICE.
 *   - return value: 0 (HELIOS_OK) or a negative HELIOS_E* code; the message is
 *     available from helios_last_error().  No C++ exception crosses the ABI.
 *   - DEVICE-pointer entry points only ENQUEUE work on the context's CUDA stream
 *     and return; they never synchronise the host.  The caller owns params and
 *     output buffers and must keep them alive until the stream has passed the
 *     enqueued work.  The *_host entry points copy, run and synchronise.
 *   - the context owns its device copies of tables, observation and workspace;
 *     host tables may be freed as soon as helios_load_opacity() returns.
 *   - level index 0 = bottom of the atmosphere (highest pressure).
 *   - units: cgs; wavenumbers in cm^-1; pressures in bar at the interface.
 *   - not thread-safe per context; use one context per host thread / stream.
 */
#ifndef HELIOS_B200_H
#define HELIOS_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct helios_ctx helios_ctx;   /* opaque */

enum {
    HELIOS_OK      =  0,
    HELIOS_EINVAL  = -1,   /* bad argument (sizes, non-monotonic grids, bins outside the grid ...) */
    HELIOS_ENOMEM  = -2,   /* device or host allocation failed                                     */
    HELIOS_ECUDA   = -3,   /* a CUDA runtime call or kernel launch failed                          */
    HELIOS_ESTATE  = -4    /* called before the tables / atmosphere / observation were set        */
};

#define HELIOS_PTRS_ON_DEVICE 1u   /* helios_load_opacity: sigma[s] / cia[c] are DEVICE pointers */

/* helios_set_option keys */
#define HELIOS_OPT_KERNEL      1   /* 0 = auto (level-parallel for a handful of models, else staged whenever the table planes fit
                                      shared memory, else direct), 1 = direct (4 taps from global memory; fallback),
                                      2 = staged TMA kernel, 3 = level-parallel kernel (2, 3: error if unavailable).
                                      Reproducibility: each kernel gives a model the same bits whatever batch it is submitted in, but
                                      the level-parallel kernel composes the layer updates in another floating-point order than the
                                      staged one (difference <= 5e-6 relative on the flux), and "auto" picks by batch size (B <= 8).
                                      A sampler that re-evaluates a point in a batch of another size and needs a bitwise-equal logL
                                      must pin the kernel with 2 or 3. */
#define HELIOS_OPT_MODELS_PER_CTA 2/* staged kernel: models (= compute warps) per CTA: 8, 16, 20, 24, 27 or 0 = auto */
#define HELIOS_OPT_NU_ORDER    4   /* column order of the resident tables, read by the NEXT helios_load_opacity: 1 (default) =
                                      sorted by a reference opacity, so that the 64 columns a warp owns are optically alike and
                                      take the kernels' warp-uniform thin / thick shortcuts; 0 = wavenumber order.  Results are
                                      always returned in wavenumber order. */
#define HELIOS_OPT_FUSED_OBS   5   /* 1 = helios_forward_batch / helios_loglike_batch apply the instrument profile and the binning in
                                      the epilogue of the RT kernel (bitwise-reproducible 64-bit integer atomics into M[b][j]) and never
                                      write a high-resolution flux: no B x nNu buffer traffic, but the atomics cost more time than the
                                      second kernel they replace (configs[3]: +2.1 ms of 44.5).  0 (default) = the
                                      RT kernel writes the flux, k_obs_apply applies the operator. */
#define HELIOS_OPT_GRAPHS      6   /* 1 (default) = a helios_forward_batch / helios_loglike_batch call that repeats with the same batch
                                      size and the same buffers is captured once into a CUDA graph (prep -> RT -> observation) and
                                      replayed with a single launch from then on (up to 32 distinct calls are kept); 0 = plain launches.
                                      Only the device-pointer entry points; never under HELIOS_OPT_TIMING.  Every call that changes
                                      the context (load_opacity, set_atmosphere, set_tp_elements, set_extras, set_observation,
                                      set_option, set_stream, a workspace that grows) drops all captured calls. */
#define HELIOS_OPT_TIMING      3   /* 1 = bracket every stage of the next calls with CUDA events on the context's stream */

typedef struct helios_stats {
    unsigned long long n_clamped;      /* (model, level) pairs whose (T, p) fell outside the table and were clamped */
    unsigned long long n_nonfinite;    /* models rejected: a parameter was NaN/Inf, or the model is unphysical
                                          (see helios_forward_batch)                                               */
    unsigned long long n_models;       /* models evaluated since the last reset                                    */
    unsigned long long n_launches;     /* kernels launched by this context since the last reset                    */
    unsigned long long n_graph_launches; /* calls since the last reset that went out as ONE CUDA-graph launch
                                          (HELIOS_OPT_GRAPHS) instead of separate kernel launches; their kernels are
                                          counted in n_launches all the same                                        */
} helios_stats;

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t
 * (may be NULL = the legacy default stream); all work is enqueued on it.
 * Fails with HELIOS_ECUDA if no CUDA device / sm_100 kernel image is usable. */
int  helios_create (helios_ctx** out, int device, void* cuda_stream);
void helios_destroy(helios_ctx* ctx);
int  helios_set_stream(helios_ctx* ctx, void* cuda_stream);
/* Message of the last failing call on this context (static storage inside ctx;
 * ctx == NULL returns the message of the last failing helios_create). */
const char* helios_last_error(const helios_ctx* ctx);
int  helios_set_option(helios_ctx* ctx, int key, int value);

/* Opacity tables.  Copies everything to HBM as fp32, one wavenumber per column,
 * rows padded to 256 B (64 floats, the kernels' tile).  The columns are kept in the order HELIOS_OPT_NU_ORDER
 * selects (default: sorted by a reference opacity; the library maps column <-> wavenumber itself, every result
 * is in wavenumber order).  Host tables are staged through one device buffer of nT*nP*nNu floats.
 *   T_grid_K        HOST [nT]  strictly increasing, arbitrary spacing (nT >= 2)
 *   log10p_grid_bar HOST [nP]  strictly increasing, arbitrary spacing (nP >= 2)
 *   wavenumber grid nu_i = nu0_cm1 + i*dnu_cm1, i < nNu (uniform, dnu > 0)
 *   sigma           HOST array of n_species pointers, each -> [nT][nP][nNu] fp32 cm^2
 *                   (HOST data, or DEVICE data with HELIOS_PTRS_ON_DEVICE)
 *   cia             HOST array of n_cia (0..2) pointers, each -> [nT][nNu] fp32,
 *                   cm^-1 amagat^-2; pair 0 = H2-H2, pair 1 = H2-He (R4)
 * Interpolation is bilinear in (T, log10 p) on sigma itself, linear in T for CIA;
 * (T, p) outside the table is clamped to the edge and counted in helios_stats. */
int helios_load_opacity(helios_ctx* ctx, int n_species,
                        int nT, const double* T_grid_K,
                        int nP, const double* log10p_grid_bar,
                        int nNu, double nu0_cm1, double dnu_cm1,
                        const float* const* sigma,
                        int n_cia, const float* const* cia,
                        unsigned flags);

/* Atmosphere discretisation.
 *   n_levels levels equidistant in log p from p_bottom_bar (level 0) to p_top_bar;
 *   n_knots temperature nodes equidistant in log p (first-order elements);
 *   n_angles Gauss-Legendre angles in mu in (0,1), 1..8;
 *   mean_mol_weight in atomic mass units; he_to_h2 = He/H2 number ratio of the
 *   background gas; flux_const = (R_star/d)^2 of Eq. 9, > 0 (HELIOS_EINVAL otherwise).
 * Requires helios_load_opacity() first (the pressure cells are resolved here). */
int helios_set_atmosphere(helios_ctx* ctx, int n_levels, double p_bottom_bar, double p_top_bar,
                          int n_knots, int n_angles, double mean_mol_weight, double he_to_h2,
                          double flux_const);

/* Temperature parametrisation by finite elements (Sect. 2.5.1, Eq. 12-16):
 * n_elements elements equidistant in log p between p_bottom and p_top, polynomial order 1..4,
 * Gauss-Lobatto points on the reference element, continuous across elements, so the profile has
 * N_T = n_elements * order + 1 temperature parameters (bottom -> top) which replace the n_knots
 * values of helios_set_atmosphere in the parameter vector.
 *   ratio_form = 0: the N_T nodal temperatures [K];
 *   ratio_form = 1: T_1 and the ratios b_2 .. b_N with T_i = b_i T_{i-1} (R28).
 * Call after helios_set_atmosphere (which selects n_knots nodes / first order again). */
int helios_set_tp_elements(helios_ctx* ctx, int n_elements, int order, int ratio_form);

/* Extra parameters appended to every parameter vector, in this order:
 *   HELIOS_EXTRA_DISTANCE         d        Eq. 9 with flux_const = R_*^2: F = F+ f flux_const / d^2
 *   HELIOS_EXTRA_ERROR_INFLATION  epsilon  Eq. 22-23: s_j^2 = sigma_j^2 + 10^epsilon in ln L
 *   HELIOS_EXTRA_GREY_CLOUD       log10 tau_c, log10 p_top [bar], log10 phi   (App. B, R29: grey cloud
 *                                 of vertical optical depth tau_c between p_top and p_top (1 + phi)) */
#define HELIOS_EXTRA_DISTANCE        1u
#define HELIOS_EXTRA_ERROR_INFLATION 2u
#define HELIOS_EXTRA_GREY_CLOUD      4u
int helios_set_extras(helios_ctx* ctx, unsigned flags);
/* HOST out: P = 2 + N_T + n_species + number of extras, the row length of `params`. */
int helios_get_n_params(const helios_ctx* ctx, int* n_params_out);

/* Observation (Eq. 17, 255, 267-270 Eq. 19).
 *   bin_edges_cm1 HOST [n_bins+1] ascending, inside [nu_0, nu_{nNu-1}]
 *   obs, obs_err  HOST [n_bins] (may both be NULL: spectra only, logL unavailable)
 *   inst_sigma_cm1 HOST [nNu] Gaussian standard deviation at each grid point,
 *                 or NULL = no instrument profile
 * Builds, on the device, the banded operator that applies "convolve (cut at
 * 5 sigma, renormalised) then bin-average" (R15, R17, R18). */
int helios_set_observation(helios_ctx* ctx, int n_bins, const double* bin_edges_cm1,
                           const double* obs, const double* obs_err,
                           const double* inst_sigma_cm1);

/* Pre-allocate workspace for batches up to max_batch.  Otherwise every entry point below that
 * takes a batch (forward_batch, loglike_batch, forward_highres, teff_batch, forward_batch_host)
 * grows it on first use of a larger B, which synchronises the stream ONCE; after that they only
 * enqueue. */
int helios_reserve(helios_ctx* ctx, int max_batch);

/* The hot path.  params: DEVICE, row-major [B][n_params] fp64 with
 *   n_params = P = 2 + N_T + n_species + n_extras  (= helios_get_n_params(); N_T = n_knots unless
 *   helios_set_tp_elements changed it; n_extras from helios_set_extras):
 *   log10 g (cgs), f (Eq. 9), the N_T temperature parameters (bottom -> top), log10 VMR[0..S-1],
 *   then the extras that are switched on.
 * n_params is the row length the CALLER built params with; a value different from
 * helios_get_n_params() returns HELIOS_EINVAL (a buffer laid out for another parametrisation would
 * otherwise be read with the wrong stride).
 * spectra_out: DEVICE [B][n_bins] fp32 or NULL; logl_out: DEVICE [B] fp64 or NULL.
 * Rejected models get NaN spectra and logL = -inf (never NaN), the other models of the batch are
 * unaffected, and helios_stats.n_nonfinite counts them.  A model is rejected when a parameter is
 * NaN/Inf or when it is unphysical [paper silent; R31]: a level temperature <= 0 (possible
 * with elements of order >= 2 or ratio parameters), sum of the VMRs > 1 (negative H2/He fill), f < 0,
 * d <= 0, or g, 10^epsilon or a cloud parameter that overflows.  Enqueues only. */
int helios_forward_batch(helios_ctx* ctx, int B, int n_params, const double* params,
                         float* spectra_out, double* logl_out);
/* == helios_forward_batch(ctx, B, n_params, params, NULL, logl_out): spectra never written. */
int helios_loglike_batch(helios_ctx* ctx, int B, int n_params, const double* params, double* logl_out);
/* Test hook: the flux of Eq. 9 on the native grid, before the instrument
 * profile.  flux_out: DEVICE [B][nNu] fp32.  Needs no observation. */
int helios_forward_highres(helios_ctx* ctx, int B, int n_params, const double* params, float* flux_out);

/* Effective temperature (Sect. 2.6): the outgoing flux F+ of Eq. 8 (without the
 * f (R/d)^2 of Eq. 9) integrated over [nu_a, nu_b] on the native grid (trapezoid, interpolated end
 * points) and converted with the Stefan-Boltzmann law.  teff_out: DEVICE [B] fp64, Kelvin.
 * Runs steps 0-4 of the hot path and one reduction kernel; needs no observation.  Enqueues only. */
int helios_teff_batch(helios_ctx* ctx, int B, int n_params, const double* params, double nu_a_cm1,
                      double nu_b_cm1, double* teff_out);

/* End-to-end variant: params, spectra_out (or NULL), logl_out (or NULL) are HOST
 * buffers (pinned for full speed).  Copies params to the device, runs the hot
 * path, copies the results back and synchronises the stream before returning. */
int helios_forward_batch_host(helios_ctx* ctx, int B, int n_params, const double* params_host,
                              float* spectra_out_host, double* logl_out_host);

/* The same for helios_teff_batch: HOST params [B][n_params] in, HOST teff_out [B] out. */
int helios_teff_batch_host(helios_ctx* ctx, int B, int n_params, const double* params_host, double nu_a_cm1,
                           double nu_b_cm1, double* teff_out_host);

/* Step 5 alone (instrument profile, binning, chi-square; Eq. 17, 239, 267-270 Eq. 19), for
 * callers that must not allocate device memory while they run: a likelihood callback invoked inside a region some
 * other library is capturing into a CUDA graph, a process whose GPU memory was all handed to a pool at start-up, a
 * loop that cannot afford the device-wide synchronisation of a cudaFree.  All the other batch entry points size
 * their workspace with cudaMalloc (helios_reserve); this one calls no cudaMalloc, no cudaFree and no library routine
 * that allocates.  Its workspace -- the per-model chi-square partial sums and arrival counters of the reduction -- is
 * a fixed array inside the library image, about 0.5 MB, which every GPU that loads the library holds until the
 * process ends.
 *   flux        DEVICE [B][nNu] fp32, rows contiguous: the flux of Eq. 9 on the native grid in wavenumber order, e.g.
 *               what helios_forward_highres wrote earlier into a buffer the caller owns.
 *   spectra_out DEVICE [B][n_bins] fp32 or NULL;  logl_out DEVICE [B] fp64 or NULL (needs obs / obs_err).
 * On the same flux the results are bitwise those of helios_forward_batch.  There are no model flags here: a row of
 * `flux` that holds NaN/Inf (helios_forward_highres writes NaN for a rejected model) gives NaN bins and logL = -inf.
 * Limits, fixed by the size of the array: B <= 4096 and B * ceil(n_bins / 8) <= 65536; anything larger returns
 * HELIOS_EINVAL and enqueues nothing (split the batch).  HELIOS_ESTATE without helios_set_observation, or when
 * HELIOS_EXTRA_ERROR_INFLATION is on (its variance term comes from the parameter vector, which is not passed here).
 * The FIRST call on each GPU looks up the array's device address (cudaGetSymbolAddress, which may load the library's
 * kernels onto that GPU): make that call once during set-up, before any stream capture begins.  Every call, from
 * every context on that GPU, uses the same array: the counters are cleared on the context's stream at the start of
 * each call, and two calls that can overlap on the GPU (different streams, different contexts or host threads) race
 * on it -- keep them on one stream or order them with events.  Enqueues only. */
int helios_observe_noalloc(helios_ctx* ctx, int B, const float* flux, float* spectra_out, double* logl_out);

/* Copies the counters (synchronises the stream); reset != 0 clears them. */
int helios_get_stats(helios_ctx* ctx, helios_stats* out, int reset);
/* Average device time per call of each stage (prep, fused interpolate+RT kernel, fused
 * convolve/bin/chi-square kernel) over the calls made since HELIOS_OPT_TIMING was set to 1
 * (at most the last 64), from CUDA events recorded on the context's stream.
 * HOST out: stage_ms[3], n_calls.  Synchronises the stream. */
int helios_get_stage_ms(helios_ctx* ctx, double* stage_ms, int* n_calls);
/* Measured arithmetic peaks of the device this context lives on (micro-benchmarks of a few hundred
 * microseconds each: dependency-free FFMA / FFMA2 / MUFU.EX2 loops on every SM, 16 warps per scheduler).
 * These are the denominators of the "alu" roofline bench.py reports ("the build must
 * microbenchmark them") and the evidence for the dispatch-cost argument of DESIGN.md section 6.
 * Runs on the context's stream and synchronises it. */
typedef struct helios_peaks {
    double sm_clock_mhz;        /* SM clock while the loops ran (clock64 against %globaltimer)                     */
    double ffma_per_clk_sm;     /* FP32 FMAs per clock per SM through scalar FFMA                                   */
    double ffma2_per_clk_sm;    /* FP32 FMAs per clock per SM through packed FFMA2 (fma.rn.f32x2)                   */
    double mufu_per_clk_sm;     /* MUFU.EX2 results per clock per SM                                                */
    double ffma2_cycles[3];     /* scheduler cycles one FFMA2 warp instruction occupies when its source operands
                                   are 1 register pair + 2 scalars / 2 pairs + 1 scalar / 3 distinct pairs          */
    double alu_extra_cycles;    /* extra scheduler cycles per LOP3 issued among FFMA2 (1.0 = no co-issue)           */
    double fsel_extra_cycles;   /* extra scheduler cycles per FSETP + FSEL pair issued among FFMA2                  */
    double ffma_3reg_cycles;    /* scheduler cycles of a scalar FFMA with three distinct register operands          */
    double mufu_extra_cycles;   /* extra scheduler cycles per MUFU.EX2 issued among FFMA2 (8 FFMA2 : 8 MUFU)        */
    int    n_sms;
} helios_peaks;
int helios_measure_peaks(helios_ctx* ctx, helios_peaks* out);
/* HOST out: the angle set in use, mu[n_angles], w[n_angles]. */
int helios_get_angles(const helios_ctx* ctx, double* mu_out, double* w_out);

#ifdef __cplusplus
}
#endif
#endif /* HELIOS_B200_H */
