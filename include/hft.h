/*
 * hft.h -- C ABI of the B200-native HipFT time-stepping hot path (libhft.so).
 *
 * The library advances the surface radial field Br(theta, phi) of a batch of independent
 * realizations with the scheme of arxiv 2501.06377 (cited as PAPER.md:<line> of the extracted text):
 *   advection  -div_s(Br v)  by differential rotation and meridional flow (Eq. 2-4),
 *              WENO3-CS(h) / upwind fluxes (Sec. 3.6.1 :348-388, App. B :650-691), SSPRK (Eq. 25 :410-424)
 *   diffusion  div_s(nu grad_s Br) (Eq. 6 :109, Eq. 27-28 :436-460) by explicit super time stepping
 *              RKL2 / RKG2(3/2) (Sec. 3.7.2 :466-476)
 *   finite-volume polar caps (App. A :622-648), periodic phi, operator splitting A then D (Eq. 21 :308-313),
 *   data-assimilation blend (Eq. 8-11 :131-153) and flux diagnostics (:225-230).
 * Every step of that path runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   - Every function returns HFT_OK (0) or a negative hft_status; nothing throws across the ABI.
 *     hft_error_string() names a code.  A context is not thread-safe.  The only process-wide state is internal and
 *     guarded: per-device caches of kernel occupancy, and the owner of the constant-bank coefficient table of k_sts_upipe
 *     (contexts that alternate on one device re-upload it, waiting for the device first).
 *   - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.  All buffers are owned by the
 *     caller (e.g. allocated with PyTorch) and must stay valid until the stream work that uses them has
 *     completed; the context never frees them.  Calls enqueue work on the stream given to hft_create
 *     and return without synchronising unless stated otherwise.
 *   - User-facing maps are dense row-major [n_theta][n_phi] in the context's dtype: row i (0-based) is
 *     the cell centred at colatitude (i+1)*pi/(n_theta+1), column k at longitude 2*pi*k/n_phi.  The two
 *     polar caps and the padding of the internal layout [R][n_theta+2][pitch] are
 *     internal; see DESIGN.md "Data layout".
 *   - Units are the paper's input units: Gauss, hours, m/s, km^2/s.
 */
#ifndef HFT_H
#define HFT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hft_ctx hft_ctx; /* opaque */

typedef enum {
    HFT_OK = 0,
    HFT_ERR_ARG = -1,       /* null pointer, size or enum out of range */
    HFT_ERR_WORKSPACE = -2, /* workspace too small or not 256-byte aligned */
    HFT_ERR_CUDA = -3,      /* a CUDA runtime call failed; see hft_last_cuda_error */
    HFT_ERR_UNSTABLE = -4,  /* forced sts_stages too small for dt, or dt <= 0 */
    HFT_ERR_NOMEM = -5,     /* host or small device table allocation failed */
    HFT_ERR_DEVICE = -6     /* no sm_100 device / kernels not loadable on the current device */
} hft_status;

/* Grid: n_theta x n_phi regular cells; the two polar caps are added internally. */
typedef struct {
    int32_t n_theta;  /* >= 8 */
    int32_t n_phi;    /* >= 8 */
    int32_t dtype;    /* 0 = fp32, 1 = fp64: storage and arithmetic of the state */
    int32_t reserved; /* must be 0 */
    double radius_cm; /* scales hft_diagnostics to Mx: 6.96e10; 1.0 = unit sphere */
} hft_grid;

/* Per-realization model parameters. */
typedef struct {
    double eta_km2_s;  /* diffusivity nu of Eq. 6, km^2/s */
    double d0, d2, d4; /* differential rotation, Eq. 3 (:78): v_phi = [d0 + d2 cos^2 + d4 cos^4] sin(theta), m/s */
    double m1, m3, m5; /* meridional flow, Eq. 4 (:84): v_theta = -[m1 cos + m3 cos^3 + m5 cos^5] sin(theta), m/s */
} hft_params;

typedef struct {
    int32_t adv_flux;   /* 0 off, 1 upwind (:362), 2 WENO3-CS(h) (default, App. B) */
    int32_t adv_time;   /* 1 forward Euler (Eq. 23), 3 SSPRK(3,3), 4 SSPRK(4,3) (default, Eq. 25) */
    int32_t diff_time;  /* 0 off, 1 explicit Euler, 2 RKL2, 3 RKG2(3/2) (default, :476) */
    int32_t sts_stages; /* 0 = smallest stable count for dt (hft_sts_stage_count); else forced, >= 2 */
    int32_t sts_block;  /* STS stages fused per kernel launch (temporal blocking): 0 = library default,
                           1 = one launch per stage, k > 1 = k stages per launch (even, <= 8) */
    int32_t rfe;        /* 1 = reserve workspace for the two random-flux-emergence source maps (Sec. 2.4; 2 more field
                           arrays) and allow hft_set_rfe.  0 (default) = off */
    int32_t strang;     /* 0 = Eq. 21 (:308-313): A(dt) then D(dt) per step (default);
                           1 = Strang splitting, Eq. 22 (:317-326) with S omitted: A(dt/2), D(dt), A(dt/2) */
    int32_t flow_attenuation; /* 1 = reserve workspace for flow attenuation (Eq. 5, :100) and allow hft_set_attenuation;
                                 6 more field arrays.  0 (default) = off */
    int32_t diffusivity_map;  /* 1 = reserve workspace for a spatially varying diffusivity nu(theta, phi) (Eq. 27-28, :438-460;
                                 1 more field array) and allow hft_set_diffusivity_map.  0 (default) = off */
    int32_t f32_arith;        /* dtype fp32 only.  0 (default) = the temporally blocked STS kernel keeps the state in fp32 in memory but
                                 does the arithmetic of a block of 8 stages in fp64 registers, rounding to fp32 only at the two
                                 stores per block (the scheme integrated is Sec. 3.7.2 :470-476 unchanged): BASELINE config 3 at
                                 full length ends 2.0e-6 .. 2.7e-6 from the fp64 oracle (north_star: <= 1e-5), at the rate of the
                                 fp64 kernel and half its memory.  1 = fp32 arithmetic throughout: 2.1 x the rate, but every stage
                                 rounds to 24 bits and the same run ends 1.4e-5 .. 2.2e-5 from the fp64 oracle.  The fp64-register
                                 path needs k_sts_upipe (see sts_kernel); batches it cannot take run in fp32 arithmetic */
    int32_t sts_kernel;       /* which temporally blocked kernel: 0 (default) = the library's choice (k_sts_upipe, where the batch
                                 allows it, for fp64 states and for fp32 states with f32_arith = 0; k_sts_pipe for fp32
                                 arithmetic); 1 = k_sts_pipe (per-realization
                                 coefficient tables through shared memory; any batch); 2 = k_sts_upipe (one coefficient table
                                 through the uniform datapath) whenever the batch shares one table up to the factor nu_r and it
                                 fits the constant bank (n_theta <= 2048), else k_sts_pipe */
} hft_options;

/* Bytes of device workspace hft_create needs for this grid / batch (state + 5 stage arrays, + 6 with
 * opt->flow_attenuation, + 2 with opt->rfe, + 1 with opt->diffusivity_map).  opt may be NULL (defaults). */
int hft_workspace_bytes(const hft_grid* grid, int32_t n_real, const hft_options* opt, size_t* h_bytes);

/* Create a context.  d_workspace: caller-allocated device memory of at least hft_workspace_bytes,
 * 256-byte aligned, owned by the caller; it holds the state and must not be touched while the context
 * lives.  cuda_stream: a cudaStream_t (0 = legacy default stream) on which all work is enqueued.
 * The state starts as zero.  Builds the per-row metric / flow / diffusion tables. */
int hft_create(const hft_grid* grid, int32_t n_real, const hft_params* h_params /*[n_real]*/,
               const hft_options* opt, void* d_workspace, size_t workspace_bytes, void* cuda_stream,
               hft_ctx** out);

void hft_destroy(hft_ctx* ctx);

/* Non-uniform theta grid ("logically-rectangular non-uniform spherical surface grid"; Eq. 27-28 :438-460 with
 * Delta theta_{j+-1/2}, Delta theta_j; :354; App. A :624-648; App. B :662-680).  h_theta[n_theta+2]: HOST, the colatitudes of
 * the rows where B_r lives, strictly increasing, h_theta[0] = 0 and h_theta[n_theta+1] = pi (the two polar caps); user map row
 * i is the cell at h_theta[i+1].  The half grid (flow speeds, fluxes, nu) lies midway between the nodes; Delta theta_{j+1/2} =
 * theta_{j+1} - theta_j, Delta theta_j = theta_{j+1/2} - theta_{j-1/2}; each polar cap reaches to its first half-mesh point and
 * takes the prefactor of App. A with its own half width; the WENO3-CS(h) constants are the D-factors of App. B with Delta x =
 * the cell widths and eps_w = the local node spacing (readings U12, U33).  phi stays uniform.  Re-makes the
 * metric, diffusion and analytic flow tables (Eq. 3-4 evaluated at the new angles): call it BEFORE hft_set_flow_tables; not
 * allowed once a diffusivity map is set (HFT_ERR_ARG).  Every kernel, the temporally blocked ones included, runs unchanged:
 * all coefficients stay phi-independent.  Synchronises the stream. */
int hft_set_theta_nodes(hft_ctx* ctx, const double* h_theta);

/* Replace the analytic flow of realization r (-1: all) by per-row tables (PAPER.md:90 custom flows,
 * phi-independent subset; needed for the App. C test :703): h_vtheta[n_theta+1] = v_theta at the
 * theta-faces (j+1/2)*dtheta, j = 0..n_theta, in m/s; h_omega[n_theta+2] = v_phi/sin(theta) at the rows
 * j*dtheta, j = 0..n_theta+1, in m/s (i.e. the bracket of Eq. 3). */
int hft_set_flow_tables(hft_ctx* ctx, int32_t r, const double* h_vtheta, const double* h_omega);

/* Latitude-dependent diffusivity nu(theta) (Eq. 6 :109 with nu on the half grid of :288, phi-independent): h_nu_face
 * [n_theta+1] in km^2/s at the theta-faces (j+1/2)*dtheta, j = 0..n_theta, for realization r (-1: all).  The theta-fluxes
 * take nu at their face, the phi-term the mean of the row's two faces (Eq. 28 :450-458); hft_stable_dt and the STS stage
 * count follow.  hft_set_grid_diffusivity sets the grid-based diffusivity of the map smoother, Eq. 7 (:121):
 * nu_g = alpha_nu [dtheta^2 + (dphi sin(theta))^2], alpha_nu in km^2/s per rad^2.  Both synchronise the stream. */
int hft_set_diffusivity_profile(hft_ctx* ctx, int32_t r, const double* h_nu_face);
int hft_set_grid_diffusivity(hft_ctx* ctx, int32_t r, double alpha_nu);

/* Spatially varying diffusivity nu(theta, phi) (Eq. 6 :109; Eq. 27-28 :438-460: nu on the grid staggered in both directions).
 * h_nu_hh: HOST, [n_theta+1][n_phi] doubles in km^2/s; entry [f][k] is nu at colatitude (f+1/2)*dtheta and longitude
 * (k+1/2)*dphi (between columns k and k+1; column n_phi-1 wraps to column 0), every value >= 0, for realization r (-1: all).
 * Owned by the caller, consumed before the call returns (synchronises the stream).  Each theta-flux takes the mean of the two
 * nu values on its face, each phi-flux likewise, the polar-cap fluxes of App. A (:624-648) the face means of row f = 0 / n_theta:
 * exactly the coefficients a_{j+-1,k}, a_{j,k+-1} of Eq. 28, applied in difference form.  Once any realization has a map,
 * every realization is advanced through the nu(theta, phi) kernels (the others with their nu(theta) profile or scalar value):
 * k_sts_mpipe, 4 stages per launch, with the polar-cap values of a block from the polar-band kernel k_sts_mcapseq (n_phi a
 * multiple of 16 bytes / sizeof(value), more than 8 stages per step), else one launch per stage (k_sts_stage_mapv /
 * k_sts_stage_map; also with sts_block = 1).  The zonal-mean cap recurrence of k_sts_pipe does not apply: the coefficients
 * depend on phi.
 * hft_stable_dt and the STS stage count use the Gershgorin bound max |a_{j,k}| over every cell of the map.  A later
 * hft_set_diffusivity_profile / hft_set_grid_diffusivity for realization r replaces its map.  Needs
 * hft_options.diffusivity_map = 1 at hft_create, else HFT_ERR_ARG. */
int hft_set_diffusivity_map(hft_ctx* ctx, int32_t r, const double* h_nu_hh);

/* Flow attenuation (Sec. 2.1.3, Eq. 5 :100-103): v -> v [1 - tanh(|Br| / B0)] with the saturation field b0_gauss of
 * realization r (-1: all; the paper's default is 500 G); b0_gauss <= 0 switches it off for that realization.  Needs
 * hft_options.flow_attenuation = 1 at hft_create, else HFT_ERR_ARG.  |Br| at a face is the magnitude of the mean of the
 * two cells the face separates; the speeds are formed once per time step from the field at its start and held through
 * the SSPRK stages (readings U22, U23).  hft_stable_dt keeps returning the un-attenuated limit, which the
 * attenuated flow (|v| can only shrink) also satisfies.  Synchronises the stream. */
int hft_set_attenuation(hft_ctx* ctx, int32_t r, double b0_gauss);

/* Random flux emergence source term S (Sec. 2.4, :155-209).  model 0 = off, 1 = uniform unsigned flux per cell (Eq. 13),
 * 2 = uniform unsigned flux per unit area (Eq. 14, the paper's default).  flux_per_hr: total unsigned flux per hour in
 * G*radius_cm^2/hr (Mx/hr for radius_cm = 6.96e10); tau_hours: lifetime of the random flux elements = time between
 * source maps (INFINITY: the first map stays); seed: of the counter-based generator (Philox4x32-10, counter = (cell,
 * map index, realization, 0), Box-Muller in fp64: DESIGN.md reading U27).  Two source maps are kept, each balanced
 * like Eq. 11; every hft_step integrates S(t) = (1-alpha) S1 + alpha S2, alpha = (t - t1)/tau (Eq. 15), with forward
 * Euler after D (Eq. 21) or as two half advances around A D A (Eq. 22); when t reaches t1 + tau, map 2 becomes map 1 and a
 * new map is drawn.  The call resets the run clock to 0 and draws maps 0 and 1.  Needs hft_options.rfe = 1. */
int hft_set_rfe(hft_ctx* ctx, int32_t model, double flux_per_hr, double tau_hours, uint64_t seed);

/* Copy source map `which` (0 = S1, 1 = S2) of realization r to d_out [n_theta][n_phi] (G/hr; tests). */
int hft_get_rfe_map(hft_ctx* ctx, int32_t r, int32_t which, void* d_out);

/* Set the map of realization r (r = -1: broadcast the one map to all).  d_map: device, [n_theta][n_phi]
 * in the context dtype.  Each polar cap is set to the dphi-weighted mean of its adjacent row. */
int hft_set_map(hft_ctx* ctx, int32_t r, const void* d_map);

/* Copy the map of realization r to d_out [n_theta][n_phi] (r = -1: all, [n_real][n_theta][n_phi]). */
int hft_get_map(hft_ctx* ctx, int32_t r, void* d_out);

/* Full internal field of realization r incl. the two cap rows: [n_theta+2][n_phi] (tests, restart). */
int hft_get_full(hft_ctx* ctx, int32_t r, void* d_out);
int hft_set_full(hft_ctx* ctx, int32_t r, const void* d_in);

/* Advance all realizations by n_steps steps of dt_hours: B <- D(A(B)) per step (Eq. 21).  Asynchronous.
 * HFT_ERR_UNSTABLE if a forced stage count is below the stable one for dt, or dt <= 0. */
int hft_step(hft_ctx* ctx, int32_t n_steps, double dt_hours);

/* Data assimilation (Eq. 8): B <- w*obs + (1-w)*B.  d_obs, d_weights: device, [n_real or 1][n_theta][n_phi]
 * in the context dtype (shared != 0: one map for all realizations).  flags bit 0: flux-balanced form
 * (Eq. 10-11).  Caps are blended with the row means of obs and w (reading U18). */
int hft_assimilate(hft_ctx* ctx, const void* d_obs, const void* d_weights, int32_t shared, int32_t flags);

/* hft_assimilate followed by hft_diagnostics of the blended state, fused: the blend kernel accumulates Phi+ / Phi- of the values
 * it writes, so the state is read once instead of twice (north_star's "fused assimilation/diagnostics kernel"; SURVEY.md 8(a)
 * row A8).  h_out[n_real][4] as hft_diagnostics.  Synchronises the stream. */
int hft_assimilate_diagnostics(hft_ctx* ctx, const void* d_obs, const void* d_weights, int32_t shared, int32_t flags, double* h_out);

/* Flux diagnostics (:225-230): h_out[n_real][4] = {signed, unsigned, Phi+, Phi-} in G*radius_cm^2.
 * Synchronises the stream. */
int hft_diagnostics(hft_ctx* ctx, double* h_out);

/* hft_diagnostics for callers that may not allocate or synchronise (code under CUDA graph capture, tight serving loops):
 * the same flux integrals (:225-230) of a field the CALLER holds, written to device memory the caller holds.
 *   d_field  device, [n_real][n_theta+2][n_phi] dense in the context dtype, rows 0 and n_theta+1 the polar caps (the layout of
 *            hft_get_full, realizations back to back); read only.
 *   d_out    device, [n_real][4] doubles = {signed, unsigned, Phi+, Phi-} in G*radius_cm^2, as hft_diagnostics.
 * Enqueues two kernels on the context's stream and returns: no cudaMalloc / cudaFree, no copy to the host, no synchronisation.
 * The per-CTA partial sums live in ONE static device array of the library (HFT_NOALLOC_MAX_REAL x 64 x 2 doubles = 1 MiB,
 * held by every GPU that loads the library until the process exits); the first call on a device resolves its address
 * (cudaGetSymbolAddress, no allocation).  n_real > HFT_NOALLOC_MAX_REAL: HFT_ERR_ARG, text in hft_last_cuda_error.
 * Every call -- of every context on that device -- uses the same array: it keeps the previous call's contents (each call
 * overwrites all it reads, nothing needs clearing), and two calls that overlap on the GPU (different streams / contexts
 * without an ordering between them) RACE on it.  Results are bit-identical to hft_diagnostics of the same field. */
#define HFT_NOALLOC_MAX_REAL 1024
int hft_diagnostics_noalloc(hft_ctx* ctx, const void* d_field, double* d_out);

/* Remaining run-history diagnostics.  h_out[n_real][13]:
 *   0..3  Phi+ and Phi- over the north polar region, then over the south polar region: the cells whose centre has
 *         |latitude| >= polar_lat_deg (0..90), polar caps included, in G*radius_cm^2;
 *   4, 5  area of the two regions, radius_cm^2;
 *   6..8  min, max and min |Br| over the whole map (caps included);
 *   9     equatorial dipole strength H = sqrt(h1^2 + h2^2) (Eq. 16), 10 axial dipole D (Eq. 17), 11 h1, 12 h2 (Eq. 16a, b),
 *         with dOmega on the unit sphere and the quadrature weights of hft_diagnostics (reading U19).
 * Synchronises the stream. */
int hft_diagnostics_ext(hft_ctx* ctx, double polar_lat_deg, double* h_out);

/* Host helpers (not timed): Eq. 26 advective limit over all rows and realizations (no safety factor),
 * explicit-Euler diffusion limit 2/rho (Gershgorin), and the STS stage count for dt.
 * The advective limit is ALWAYS the Eq. 26 form (:430), the limit of SSPRK(4,3), whatever adv_time the context was created
 * with: forward Euler / upwind and SSPRK(3,3) are bound by Eq. 24 (:404), HALF of it -- a caller that selects adv_time 1 or 3
 * multiplies by 0.5 itself (the paper applies a further safety factor of ~0.9, :406).  hft_step does not check dt against
 * either: Eq. 24 is the paper's approximation for two-dimensional flow (a one-dimensional upwind step is stable, and exact,
 * at twice that).  The diffusive side IS checked: a forced sts_stages below the stable count returns HFT_ERR_UNSTABLE. */
int hft_stable_dt(hft_ctx* ctx, double* h_dt_adv_limit_hours, double* h_dt_diff_euler_hours);
int hft_sts_stage_count(hft_ctx* ctx, double dt_hours, int32_t* h_stages);

/* Wait for everything this context has enqueued and report it: hft_step and the other asynchronous calls return once their
 * kernels are QUEUED, so a fault inside a kernel surfaces at the next synchronising call; calling hft_synchronize after a
 * step attributes it to that step (HFT_ERR_CUDA, text in hft_last_cuda_error). */
int hft_synchronize(hft_ctx* ctx);

/* Number of kernel launches enqueued by this context so far. */
int hft_launch_count(hft_ctx* ctx, int64_t* h_count);

/* Enable per-kernel CUDA-event timing on the context's stream for the kernel class `which`
 * (0 = none, 1 = STS stage kernels, 2 = advection stage kernels); every 16th launch of the class
 * is bracketed by events.  hft_kernel_time returns the accumulated milliseconds of the sampled launches,
 * their number and the number of stages (STS stages / SSPRK stages) they covered since the last call,
 * and resets them (synchronises). */
int hft_profile_kernels(hft_ctx* ctx, int32_t which);
int hft_kernel_time(hft_ctx* ctx, double* h_ms, int64_t* h_launches, int64_t* h_stages);

/* Not part of the time-stepping path: the FMA issue rate of the current device, measured with a register-only loop (16
 * independent chains per thread, 4 CTAs of 128 threads per SM, ~1 ms) -- the denominator of bench.py's "alu" roofline
 * (DESIGN.md section 6), so that it can be re-measured on any box.  dtype 0 = fp32, 1 = fp64.  pattern 0: x = fma(x, a, b)
 * with a, b shared by all FMAs of a thread; 1: three distinct register operands per FMA; 2: one operand from the constant
 * bank.  *h_lane_fma_per_s = FMA lane-operations per second (x 2 = flop/s).  Allocates and frees two small device buffers,
 * runs on the default stream, synchronises. */
int hft_probe_fma_rate(int32_t dtype, int32_t pattern, double* h_lane_fma_per_s);

const char* hft_error_string(int code);
const char* hft_last_cuda_error(hft_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* HFT_H */
