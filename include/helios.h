/*
 * helios.h -- C-ABI of the B200-native (sm_100a) two-stream radiative-transfer hot path of
 * HELIOS (Malik et al., arXiv:1606.05474).  Citations "PAPER.md:<line>" refer to the paper text
 * the build was written from; "DESIGN.md Gx/Sx" are the readings taken where the paper is
 * garbled or silent.
 *
 * What the library computes, for nc independent columns (PAPER.md:121-191, 216-259, 261-324,
 * 336-358, 376):
 *   a0  level temperatures: interfaces from layer centres, linear in log P
 *   a1  kappa(level, bin, g): bilinear in (log10 P, T) on the k-table, clamped
 *   a2  bin-mean Planck function at every level + pi*B(T_intern)
 *   a3  sublayer optical depth (eq. 19), transmission (eq. 8), coupling
 *       coefficients (eq. 12-13) and linear-in-tau source terms (eq. 15; eq. 11
 *       below dtau_iso; eq. 14 when 1-w0 < one_minus_w0_min)
 *   a4-a7  (1 + n_scat) x [down sweep, BOA condition eq. 22, up sweep]
 *          or, with n_scat = HELIOS_NSCAT_DIRECT, the solution of the coupled system these sweeps
 *          iterate on (their n_scat -> infinity limit), by an O(n) direct solve     (S12)
 *   a8  F(j) = sum_bins dnu sum_g w_g F(interface j; bin, g), up and down
 *   a9  radiative-equilibrium temperature step with per-layer adaptive
 *       pseudo-timestep, oscillation rule and convergence tests
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback: without a CUDA device
 * every call that needs one returns HELIOS_E_CUDA.
 *
 * Conventions.  cgs units (P in dyn cm^-2, wavenumber in cm^-1, flux in erg s^-1 cm^-2).
 * n layers, n+1 interfaces; index 0 = bottom of the atmosphere (BOA), n = top (TOA)
 * (PAPER.md:216, 236, 255).  All arrays are dense, row-major, fp64 unless stated.
 *
 * Precision.  params.precision = HELIOS_PREC_FP32 runs the per-ray arithmetic (a1, a3-a7) in fp32
 * with cancellation-free coefficient forms; inputs and outputs stay fp64, as do the Planck integrals,
 * the reductions and the RE step.  An fp32 copy of the k-table is kept in the workspace.  The fluxes then
 * carry ~1e-6 relative noise.  RE runs in fp32: individual layers wander by ~1 K in the transient (a layer whose dF
 * is fp32 noise is still moved), but the run converges to the fp64 answer -- measured with the default
 * flux_floor = 1e-7: 3.5e-3 K (config 0), 7.9e-3 K (config 1), median 1e-3 K (config 3 sample) from the fp64 oracle's
 * converged temperatures, in a similar number of iterations.  Do NOT raise flux_floor to silence the noise: a wider
 * dead zone stops layers early in either precision (config 1 at 1e-5: 26 K from the 1e-7 answer).
 *
 * Memory and ownership.  Pointers named d_* (and everything not marked "host") are DEVICE
 * pointers owned by the caller; the library never frees or reallocates them.  ktab is kept BY
 * REFERENCE (it must stay valid and unchanged until helios_destroy); all other setup/column
 * arrays are copied into the workspace during the call.  The library owns only the opaque
 * context; all device scratch lives in the caller-provided workspace of
 * helios_workspace_bytes(params) bytes (256-byte aligned).  The *_host entry points take HOST
 * pointers for the per-call inputs/outputs and do the host<->device copies themselves (inside
 * the call, on the context's stream, through the workspace).
 *
 * Streams.  All work is ordered on the cudaStream_t given to helios_setup.  helios_fluxes
 * does not synchronise.  helios_iterate_re synchronises when it polls the device's "columns still
 * running" counter (every poll_every iterations when a tolerance is set) and once before it
 * returns.  When max_iter >= poll_every and kernel timing is off, the iterations are replayed from a
 * CUDA graph of poll_every (ray kernel, RE step) pairs on a context-owned non-blocking stream that
 * waits on the caller's stream at entry and that the caller's stream waits on at exit, so the
 * ordering the caller sees is unchanged.  The *_host entry points synchronise before returning.
 *
 * Errors.  Every int-returning call returns HELIOS_OK (0) or a negative HELIOS_E_* code and
 * never throws; helios_last_error(ctx) returns a static or context-owned string describing
 * the last failure.  Passing ctx == NULL returns HELIOS_E_BADARG.
 */
#ifndef HELIOS_H_
#define HELIOS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HELIOS_OK            0
#define HELIOS_E_BADARG     (-1)  /* NULL pointer, non-positive size, unsupported option      */
#define HELIOS_E_NOTSETUP   (-2)  /* helios_set_columns not called before fluxes / iterate    */
#define HELIOS_E_CUDA       (-3)  /* CUDA runtime error or no device                          */
#define HELIOS_E_NONFINITE  (-4)  /* a NaN/Inf reached the bolometric fluxes or temperatures  */
#define HELIOS_E_WORKSPACE  (-5)  /* workspace NULL, misaligned or smaller than required      */

#define HELIOS_PREC_FP64 0
#define HELIOS_PREC_FP32 1

/* n_scat value that replaces the sweeps of PAPER.md:292 by the direct O(n) solve of the coupled
 * system they iterate on (all sublayer relations eq. 14/15 + the boundary conditions eq. 20, 22):
 * the n_scat -> infinity limit, by the adding method scanned over the layers (S12). */
#define HELIOS_NSCAT_DIRECT (-1)

/* Largest supported number of sublayers (2*n_layers, or n_layers with isothermal_layers=1):
 * the ray kernel holds a whole ray in the registers of one warp, at most 16 sublayers per lane. */
#define HELIOS_MAX_SUBLAYERS 512

typedef struct helios_ctx helios_ctx;

typedef struct {
    int32_t n_cols, n_layers, n_bins, n_g, ntab_p, ntab_t;
    int32_t precision;         /* HELIOS_PREC_FP64 / HELIOS_PREC_FP32 (per-ray arithmetic; inputs,
                                  Planck function, reductions and outputs stay fp64)                */
    int32_t n_scat;            /* extra sweeps after the first; paper: 4 per RE step, 80 one-shot
                                  (PAPER.md:292).  Ignored (0) when every w0 == 0.
                                  HELIOS_NSCAT_DIRECT (-1): direct solve of the coupled system
                                  (not with warm_start: HELIOS_E_BADARG)                           */
    int32_t warm_start;        /* 0 = upward fluxes start from zero in every evaluation (default,
                                  DESIGN.md S4); 1 = the RE steps of helios_iterate_re start from the
                                  previous step's upward fluxes, kept per ray in the
                                  workspace -- rejected (HELIOS_E_BADARG) above 16 GiB of state;
                                  helios_set_columns zeroes the state, helios_fluxes is always cold */
    int32_t isothermal_layers; /* 0 = non-isothermal layers, two sublayers per layer
                                  (PAPER.md:230, 274); 1 = eq. 11 on whole layers */
    double  D;                 /* diffusivity factor, 2                          */
    double  gravity;           /* cm s^-2, eq. 19                                    */
    double  dtau_iso;          /* sublayers thinner than this use the isothermal formula: 1e-4
                                                                                     */
    double  one_minus_w0_min;  /* bins with 1-w0 below this use eq. 14: 1e-6         */
    double  dT_frac_max;       /* RE limiter |dT_i| <= dT_frac_max*T_i (S7; not in paper)  */
    double  T_floor;           /* RE limiter T_i >= T_floor [K]          (S7)             */
    double  flux_floor;        /* RE dead zone (S11): a layer with |dF_i| < flux_floor *
                                  sigma_SB T_i^4 -- eq. 29's own per-layer test, 1e-7
                                  -- is not moved; 0 = the bare method                              */
    int32_t exact_absorption;  /* 1 = exact solution of the radiative transfer equation in the
                                  pure-absorption limit instead of the two-stream formulas: eq. 4
                                  (eq. 3 below dtau_iso) with the transmissivity of eq. 6,
                                  T = (1-dtau) e^-dtau + dtau^2 E_1(dtau)  (DESIGN.md
                                  S13).  w0, g0, D and n_scat are then not used.  0 = two-stream     */
    double  planck_table_dT;   /* > 0: the bin-mean Planck function of the levels is read from a table
                                  built at set-up on the grid T_k = k * planck_table_dT, k = 0 ...
                                  ("a grid in T (Delta T = 10 K)"), linear in T between the
                                  nodes (S15): an opt-in approximation, ~7e-5 relative on the
                                  fluxes at 10 K.  0 = exact series (default)                        */
    double  planck_table_Tmax; /* end of that table [K]; a column with a level at or above it falls back
                                  to the exact series.  The table takes n_bins * (Tmax/dT + 2) doubles
                                  of the workspace                                                   */
    double  trans_table_dlog10k; /* > 0: the transmission function of eq. 8 is taken from a table on the
                                  opacity grid kappa_k = 10^(k * trans_table_dlog10k) cm^2/g (PAPER.md:423:
                                  "opacity (Delta log10 kappa = 0.1)"), linear in log10 kappa between the
                                  nodes, at the sublayer's opacity (the kappa of eq. 19) (S16): an
                                  opt-in approximation (<= 2.1e-3 absolute on the transmission at 0.1) and
                                  NOT a speed-up on this hardware.  Not with exact_absorption or
                                  helios_set_scattering.  0 = exact (default)                        */
} helios_params;

/* Bytes of device workspace helios_setup needs for these parameters (0 if they are invalid). */
size_t helios_workspace_bytes(const helios_params* params);

/*
 * Creates a context: validates params, lays the workspace out, precomputes the per-level and
 * per-bin constants on the device (level pressures, table P-axis cell and weight, interface
 * interpolation weights, eq. 8/13 constants of each bin, bin widths) and stores ktab by
 * reference.  All arrays are device pointers.
 *   p_layer      [n]     layer-centre pressures, index 0 = BOA
 *   p_interface  [n+1]   interface pressures, index 0 = BOA, n = TOA
 *   bin_edges    [nb+1]  wavenumber bin edges, cm^-1, ascending
 *   g_pts,g_wts  [ng]    Gauss-Legendre nodes / weights on [0,1], weights sum to 1 (eq. 31-33)
 *   ktab         [ntab_p][ntab_t][nb][ng]  total extinction opacity, cm^2 g^-1
 *   tab_log10p   [ntab_p] uniform ascending log10(P / dyn cm^-2) axis
 *   tab_t        [ntab_t] uniform ascending temperature axis, K
 *   w0, g0       [nb]    single-scattering albedo and asymmetry per bin
 *   workspace    device memory, >= helios_workspace_bytes(params), 256-byte aligned
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream)
 * Returns HELIOS_OK and *out, or an error with *out = NULL.
 */
int helios_setup(helios_ctx** out, const helios_params* params,
                 const double* p_layer, const double* p_interface, const double* bin_edges,
                 const double* g_pts, const double* g_wts, const double* ktab,
                 const double* tab_log10p, const double* tab_t,
                 const double* w0, const double* g0,
                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Sets the per-column state (device pointers; copied) and resets the RE state (step factors to
 * 1, sign histories, iteration counters and convergence flags to 0).
 *   T             [nc][n]  layer-centre temperatures, K
 *   f_star        [nb]     TOA downward flux per unit wavenumber, eq. 20
 *   f_star_scale  [nc] or NULL (= 1): per-column factor on f_star
 *   t_intern      [nc]     internal temperature of eq. 21-22, K (0 = none)
 *   kscale        [nc] or NULL (= 1): per-column factor on every table value
 */
int helios_set_columns(helios_ctx* ctx, const double* T, const double* f_star,
                       const double* f_star_scale, const double* t_intern, const double* kscale);

/* Same with HOST pointers (pageable or pinned); synchronises the stream before returning. */
int helios_set_columns_host(helios_ctx* ctx, const double* T, const double* f_star,
                            const double* f_star_scale, const double* t_intern,
                            const double* kscale);

/*
 * Scattering opacity per bin, kappa_scat [nb] in cm^2/g (device pointer; copied), e.g. the Rayleigh
 * cross-section of eq. 16-17 over the mean molecular mass (S14).  From this call
 * on it is added to the table (absorption) opacity at every level, and the single-scattering albedo becomes a
 * quantity of the sublayer: w0 = kappa_scat / (mean total opacity of the sublayer), entering eq. 8, 12-13, 15
 * and the switch to eq. 14 (1 - w0 < one_minus_w0_min) sublayer by sublayer; the w0 array of helios_setup is no
 * longer used, g0 still is; kscale multiplies the table value only.  Works with the sweeps and with
 * HELIOS_NSCAT_DIRECT, in both precisions (these coefficients are always formed in fp64).  All zeros =
 * pure absorption.  HELIOS_E_BADARG with exact_absorption = 1.  Asynchronous on the context's stream.
 */
int helios_set_scattering(helios_ctx* ctx, const double* kappa_scat);

/* Replaces only the temperatures (device pointer [nc][n]); the RE state is left untouched. */
int helios_set_temperatures(helios_ctx* ctx, const double* T);

/*
 * One flux evaluation (steps a0-a8) at the current temperatures.  Outputs (device):
 *   F_up, F_dn    [nc][n+1]  bolometric interface fluxes (eq. 23's F-up, F-down)
 *   spec_up_toa   [nc][nb] or NULL: sum_g w_g F_up(TOA) per bin (emission spectrum)
 *   spec_dn_boa   [nc][nb] or NULL: sum_g w_g F_dn(BOA) per bin
 * Asynchronous on the context's stream.
 */
int helios_fluxes(helios_ctx* ctx, double* F_up, double* F_dn,
                  double* spec_up_toa, double* spec_dn_boa);

/*
 * The same evaluation for callers that must not allocate (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the per-block partial sums of step a8 -- the ray kernel's scratch, otherwise
 * a slice of the caller's workspace -- live in a file-scope `static __device__` array of
 * HELIOS_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads the library holds until the process
 * exits.  Its device address is looked up once per device at helios_setup (cudaGetSymbolAddress, with that device
 * current); this call itself launches kernels and two device-to-device copies and calls no cudaMalloc, cudaFree or
 * other allocating routine, does not synchronise, and records no timing events.
 *   F_up, F_dn  [nc][n+1] device outputs, as helios_fluxes (each may be NULL); no spectra.
 * Limit: n_chunks * nc * 4 * (n+1) * 8 bytes of partial sums (n_chunks = out[1] of helios_launch_shape) must fit
 * HELIOS_STATIC_SCRATCH_BYTES -- i.e. n_chunks * n_cols <= 1297 at 100 layers: single columns (148 chunks), small
 * batches, a few hundred columns of a batch plan; beyond it the call returns HELIOS_E_WORKSPACE with the two sizes in
 * helios_last_error.  HELIOS_E_BADARG if the context's device is not the current one.
 * Sharing: all contexts and all calls on a device use the one array, and it keeps the last call's contents.
 * Nothing in it has to start at zero (every word the reduction reads is written by the ray kernel of the same
 * call), but two calls that overlap on the GPU (different streams, or concurrent graph launches) race on it:
 * serialise them.  Results are bit-identical to helios_fluxes (same kernels, same summation order).
 */
#define HELIOS_STATIC_SCRATCH_BYTES (4u * 1024u * 1024u)
int helios_fluxes_static(helios_ctx* ctx, double* F_up, double* F_dn);

/* Host-buffer variant: copies T_host [nc][n] (or NULL = keep current) to the device, evaluates,
 * copies F_up / F_dn [nc][n+1] back to HOST memory and synchronises. */
int helios_fluxes_host(helios_ctx* ctx, const double* T_host, double* F_up_host, double* F_dn_host);

/*
 * Radiative-equilibrium iteration on the device (step a9 around a0-a8), at most max_iter flux
 * evaluations per column, chained with earlier calls (state kept in the context).  Per
 * iteration and column, in this order: fluxes(T) -> dT_i -> convergence test -> if not
 * converged: T_i <- max(T_i + dT_i, T_floor), push sgn(dT_i), step_factor_i *= rule(history).
 *   dT_i = -a_i * 1e5 * (P_i/dP_i) * sgn(dF_i)|dF_i|^0.1 / (sigma_SB T_i^3), clipped to
 *          +-dT_frac_max*T_i;  dF_i = Fnet(i+1) - Fnet(i)  (eq. 23-28; S6, G3)
 *   converged when max_i|dT_i| < tol_dT (if tol_dT > 0) or max_i|dF_i|/(sigma T_i^4) < tol_flux
 *          (eq. 29, if tol_flux > 0); a converged column is frozen.
 * Outputs (device, each may be NULL): T_out [nc][n]; iters [nc] flux evaluations done so far;
 * converged [nc] 0/1.  poll_every <= 0 selects the default (16).
 * Returns HELIOS_E_NONFINITE if a column produced a non-finite flux or temperature step (see
 * helios_get_re_metrics for which; the other columns' results are valid).
 */
int helios_iterate_re(helios_ctx* ctx, int32_t max_iter, double tol_dT, double tol_flux,
                      int32_t poll_every, double* T_out, int32_t* iters, int32_t* converged);

/* Host-buffer variant: T_host_inout [nc][n] is copied in (NULL = keep current state), the
 * iteration runs, and T / iters / converged are copied back to HOST memory. */
int helios_iterate_re_host(helios_ctx* ctx, int32_t max_iter, double tol_dT, double tol_flux,
                           int32_t poll_every, double* T_host_inout, int32_t* iters_host,
                           int32_t* converged_host);

/*
 * RE state of every layer (device outputs, each may be NULL):
 *   step_factor [nc][n]  a_i
 *   sign_hist   [nc][n]  packed history: bits 0..11 six 2-bit codes, newest in bits 0..1
 *                        (0 = zero step, 1 = dT > 0, 2 = dT < 0); bits 12..15 = entries pushed,
 *                        saturating at 6
 *   dT_last     [nc][n]  the last computed dT_i
 */
int helios_get_re_state(helios_ctx* ctx, double* step_factor, int32_t* sign_hist, double* dT_last);

/*
 * Per-column convergence metrics of the last RE iteration each column took part in (device outputs [nc], each may
 * be NULL):
 *   max_dT      max_i |dT_i| [K]                      (the quantity tol_dT tests)
 *   max_rel_dF  max_i |dF_i| / (sigma_SB T_i^4)       (eq. 29; the quantity tol_flux tests)
 *   nonfinite   1 if the column produced a non-finite flux or temperature step in the last helios_fluxes /
 *               helios_iterate_re call: such a column is left untouched from then on (its T is not updated) while
 *               the other columns carry on, and the call returns HELIOS_E_NONFINITE when it ends.  The flags are
 *               cleared at the start of every helios_fluxes* / helios_iterate_re* call.
 */
int helios_get_re_metrics(helios_ctx* ctx, double* max_dT, double* max_rel_dF, int32_t* nonfinite);

/*
 * Restores an RE state saved with helios_get_re_state / helios_iterate_re (checkpoint / resume;
 * device pointers, each may be NULL = keep): step_factor [nc][n], sign_hist [nc][n], iters [nc],
 * converged [nc].  The count of running columns is recomputed from `converged`.
 */
int helios_set_re_state(helios_ctx* ctx, const double* step_factor, const int32_t* sign_hist,
                        const int32_t* iters, const int32_t* converged);

/* Bolometric fluxes of the last evaluation (device outputs [nc][n+1], each may be NULL). */
int helios_get_fluxes(helios_ctx* ctx, double* F_up, double* F_dn);

/*
 * Device-side timing of the ray kernel (the dominant kernel).  After helios_enable_timing(ctx, 1)
 * every launch of the ray kernel is bracketed by a pair of CUDA events on the context's stream
 * (at most 4096 pairs are kept between reads).  helios_kernel_time_ms synchronises the stream,
 * returns the summed duration in milliseconds and the number of launches since the last read,
 * and clears the record.
 */
int helios_enable_timing(helios_ctx* ctx, int32_t on);
int helios_kernel_time_ms(helios_ctx* ctx, double* total_ms, int64_t* launches);

/* Number of kernels the library has launched on this context so far. */
int64_t helios_launch_count(const helios_ctx* ctx);

/* Launch shape of the ray kernel: out[0] = grid.x (columns), out[1] = grid.y (bin chunks),
 * out[2] = threads per block, out[3] = dynamic shared memory bytes, out[4] = sublayers per lane. */
int helios_launch_shape(const helios_ctx* ctx, int32_t out[5]);

/* Measures the device's sustained FP64 (precision 0) or FP32 (precision 1) FMA issue rate with a
 * register-resident dependent-chain kernel; returns FMA lane-instructions per second (x2 = flop/s),
 * or a negative HELIOS_E_* code.  Used by bench.py as the ALU roofline denominator. */
double helios_measure_fma_peak(int32_t precision, void* cuda_stream);

/* The same with three distinct register operands per FMA.  On B200 an FP64 FMA of this kind issues at
 * ~65 % of the rate above (it reads six 32-bit registers: the register file is the limit); most FMAs of
 * the sweeps are of this kind, so this is the practical ceiling bench.py reports next to the nominal one. */
double helios_measure_fma3_peak(int32_t precision, void* cuda_stream);

const char* helios_last_error(const helios_ctx* ctx);
void helios_destroy(helios_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* HELIOS_H_ */
