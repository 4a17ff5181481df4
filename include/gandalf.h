/* gandalf.h -- C ABI of the B200-native GANDALF KRMHD hot path (arXiv 2511.21891).
 *
 * The library evaluates the pseudo-spectral right-hand side of the Kinetic Reduced MHD
 * equations and advances them with the integrating-factor RK2 step, entirely in hand-written
 * sm_100a CUDA kernels (no cuFFT, no CPU fallback).  Citations are PAPER.md line numbers with
 * the section / equation they fall in; readings of ambiguous passages are DESIGN.md Q1-Q24.
 *
 * Conventions
 *  - All functions return GANDALF_OK (0) or a negative error code; they never throw or abort.
 *    gandalf_last_error(ctx) returns a ctx-owned, NUL-terminated message for the last failure.
 *  - The handle owns every device buffer.  Caller arrays are only read / written during a call.
 *    `on_device` says whether caller array pointers are HOST (0) or DEVICE (1) pointers on the
 *    ctx's device.  Host-pointer calls synchronise the ctx's stream before returning; device-
 *    pointer calls are stream-ordered on the ctx's stream and do not synchronise.
 *  - No global state; contexts are independent; one context must not be used from two threads
 *    at once.
 *
 * Boundary array layout ("half-plane"): complex fp64, interleaved (re,im) doubles,
 *    a[field][kz][ky][kx],  kx = 0..nx/2 fastest (nx/2+1 entries), ky and kz in FFT order
 *    (0..N/2-1, -N/2..-1), physical normalisation  f(x) = sum_k fhat(k) exp(+i k.x),
 *    fhat(k) = (1/(nx ny nz)) sum_x f(x) exp(-i k.x)            [PAPER.md:125-130, Eq. 9]
 *    with k_j = 2 pi n_j / L_j                                   [PAPER.md:128].
 *    Bytes per field: 16 * (nx/2+1) * ny * nz.
 */
#ifndef GANDALF_H_
#define GANDALF_H_

#ifdef __cplusplus
extern "C" {
#endif

#define GANDALF_OK               0
#define GANDALF_ERR_INVALID     -1   /* NULL pointer, bad size or parameter                     */
#define GANDALF_ERR_CUDA        -2   /* a CUDA runtime call or kernel launch failed             */
#define GANDALF_ERR_NONFINITE   -3   /* NaN/Inf seen in the energy reduction of the last step   */
#define GANDALF_ERR_UNSUPPORTED -4   /* e.g. M > 0 with vA != 1 (Eq. 6 is written for v_A = 1)  */
#define GANDALF_ERR_CFL         -5   /* dt <= 0 asked for the CFL step of Eq. 16 but max|grad Phi| = 0 and no dt_max */

typedef struct gandalf_ctx gandalf_ctx;   /* opaque */

#define GANDALF_HERMITE_EXACT_MAX_M 256   /* largest M with hermite_exact = 1 (shared-memory rows of the propagator, host eigen-solve) */

typedef struct gandalf_params {
  int    nx, ny, nz;      /* grid; powers of two, 8 <= nx,ny <= 512, 2 <= nz <= 512               */
  int    M;               /* number of Hermite moments g_0..g_{M-1}; 0 = RMHD only (Q10)          */
  double Lx, Ly, Lz;      /* box lengths (> 0)                                                    */
  double vA;              /* Alfven speed in exp(+-i kz vA dt)  [Eq. 12-13, PAPER.md:154-158]     */
  double eta;             /* (hyper)resistivity coefficient on w+-  [Eq. 17-18, PAPER.md:230-236] */
  int    r;               /* hyper order r >= 1                                                   */
  int    eta_normalized;  /* 1: exp(-eta (kperp^2/kperp_max^2)^r dt) [Eq. 18]; 0: exp(-eta kperp^(2r) dt) */
  double eta_z;           /* k_z hyperdissipation exp(-eta_z (kz^2/kz_max^2)^r_z dt); 0 = off (Q9) */
  int    r_z;
  double eta_g;           /* same perpendicular (and k_z) factor applied to g_m; 0 = paper-literal */
  double nu_coll;         /* exp(-nu_coll (m/M)^(2p) dt) on g_m  [Eq. 19, PAPER.md:240]            */
  double p;               /* hyper-collision exponent p >= 1/2                                    */
  int    closure;         /* 0: g_M = 0 (absorbing); 1: g_M = g_{M-2} (reflecting) [PAPER.md:105]  */
  int    if_variant;      /* 0: paper-literal double phase [Eq. 15, Alg. 1]; 1: standard IF midpoint (Q6) */
  int    g_sign;          /* +1: upper signs of Eq. 6 (g^+), -1: lower signs (g^-)                */
  int    nonlinear;       /* 1: brackets on; 0: brackets replaced by zero (linear tests)          */
  int    hermite_coeff;   /* 0: sqrt(m/2), sqrt((m+1)/2) for every m [Eq. 6c]; 1: literal sqrt(2), sqrt(3/2) of Eq. 6a/6b (Q24) */
  double force_eps;       /* energy injection rate of the white-noise forcing; 0 = off [Eq. 25]; > 0 with an
                             empty forced shell is GANDALF_ERR_INVALID                              */
  int    force_nperp_min, force_nperp_max, force_nz_max;  /* forced shell in mode numbers          */
  unsigned long long seed;/* forcing RNG key (counter-based, Q17)                       */
  double cfl;             /* C of Eq. 16, used when gandalf_step gets dt <= 0      */
  double force_g_amp;     /* white-noise forcing of g_0 at k = (0,0,+-force_g_nz): amplitude a_g, mean injected
                             power a_g^2 into W_g; 0 = off  [velocity-space benchmark; Q26].  With
                             nspecies = 2 only g^+_0 (the first species) is forced                        */
  int    force_g_nz;      /* forced parallel mode number (>= 1, retained); paper: 1               */
  int    nspecies;        /* 1: one set g_0..g_{M-1} with sign g_sign.  2: both slow-mode species [Eq. 2-4, PAPER.md:57-66;
                             memory layout of PAPER.md:357]: g_hat holds 2M fields, g^+ (sign g_sign) then g^- (sign
                             -g_sign); they share Phi, Psi and do not couple in Eq. 6 as printed (Q11, Q27) */
  double dt_max;          /* > 0: upper bound of the CFL step of Eq. 16, and the step taken when max|grad Phi| = 0;
                             0 = no bound (paper-literal Eq. 16; a vanishing flow is then GANDALF_ERR_CFL)  (Q29) */
  int    hermite_exact;   /* 0: Hermite moments by plain RK2 [Alg. 1 l.4, l.9] (default).  1: the streaming / phase-mixing
                             operator s i kz (I - T) of Eq. 6 is integrated exactly (matrix exponential in m per kz,
                             integrating-factor midpoint for the brackets) [future work of PAPER.md:657, 829; lifts the
                             dt < dz/v_th constraint of PAPER.md:214; Q30].  Needs the absorbing
                             closure, hermite_coeff = 0 and M <= GANDALF_HERMITE_EXACT_MAX_M (else GANDALF_ERR_UNSUPPORTED) */
  int    m_offset;        /* Moment shard [SURVEY.md 8(e)(i); PAPER.md:832, 975 list multi-device runs as future work; Q31]: */
  int    M_global;        /* this context holds the moments m_offset .. m_offset+M-1 of a hierarchy of M_global moments (0 = not
                             sharded).  If m_offset > 0 its FIRST moment field is a halo copy of the lower neighbour's last owned
                             moment, if m_offset+M < M_global its LAST one a halo copy of the upper neighbour's first: halos are
                             inputs the caller refreshes after every stage (gandalf_step_stage, gandalf_field_ptr,
                             gandalf_halo_refresh); they are left out of W_g.  Coefficients sqrt(m/2), sqrt((m+1)/2), the
                             closure and (m/M)^(2p) use the global m and M_global; xi+- are replicated.  nspecies = 1,
                             hermite_exact = 0 only.                                                   */
  int    device;          /* CUDA device ordinal                                                  */
  void*  stream;          /* cudaStream_t to enqueue on; NULL = the legacy default stream         */
} gandalf_params;

/* Fill *p with defaults: M=0, L=2pi, vA=1, no dissipation, r=r_z=1, p=1, absorbing closure,
 * paper-literal IF, g_sign=+1, nonlinear=1, no forcing (shell 1..2, |nz|<=1), cfl=0.3, device 0. */
int gandalf_default_params(gandalf_params* p);

/* Allocate a context (all device buffers, FFT twiddle tables) for the given problem.
 * Errors: INVALID for NULL / non-power-of-two / out-of-range sizes, M < 0, L <= 0;
 * UNSUPPORTED for M > 0 with vA != 1 (Q12); CUDA if allocation fails (nothing is leaked). */
int gandalf_create(const gandalf_params* p, gandalf_ctx** out);
int gandalf_destroy(gandalf_ctx* ctx);

/* State exchange.  zeta_hat: the Elsasser POTENTIALS xi^+ then xi^- (2 fields, not the
 * vorticities; w = -kperp^2 xi is formed inside).  g_hat: M fields (may be NULL
 * when M = 0).  gandalf_set_state PROJECTS its input: it applies the Eq. 20 mask (a mode is
 * kept iff 3|n| <= N on every axis), zeroes kperp = 0 for zeta, and replaces
 * the kx = 0 plane by (a(0,ky,kz) + conj a(0,-ky,-kz))/2 so the real-space field is real.
 * It also resets time, step counter and energy history.  gandalf_get_state returns the current
 * (projected) state with zeros at removed modes.
 * With HOST pointers only the retained modes of large inputs cross PCIe (30 % of the array: four pitched sub-block copies per
 * field; the entries Eq. 20 removes are never read). */
int gandalf_set_state(gandalf_ctx* ctx, const double* zeta_hat, const double* g_hat, int on_device);
int gandalf_get_state(gandalf_ctx* ctx, double* zeta_hat, double* g_hat, int on_device);

/* Exact checkpoint / restart of the evolved variables (SURVEY.md section 5 "Checkpoint / resume"; PAPER.md:389-391
 * "bit-exact restarts").  The raw state is what the library time-steps: the vorticities w^+, w^- = -kperp^2 xi^+-
 * [PAPER.md:156] and g_m, complex fp64, RETAINED modes only, a[field][cz][cy][cx] with cx = 0..nx/3 (n_x = cx),
 * cy = 0..2(ny/3) (n_y = cy for cy <= ny/3, else cy - (2(ny/3)+1)), cz likewise: gandalf_state_raw_doubles() doubles.
 * (gandalf_get_state / gandalf_set_state convert to potentials and back, which is not bit exact.)
 * gandalf_set_state_raw copies the array in without projection and keeps time, step counter and history;
 * gandalf_set_time sets the simulation time and the step counter -- the forcing RNG counters derive from the step
 * number (Q17, Q26), so a run resumed with {get_state_raw, get_time} -> new context -> {set_state_raw,
 * set_time} continues bit for bit.  The energy history restarts at the resumed step. */
int gandalf_state_raw_doubles(const gandalf_ctx* ctx, long long* n);
int gandalf_get_state_raw(gandalf_ctx* ctx, double* out, int on_device);
int gandalf_set_state_raw(gandalf_ctx* ctx, const double* in, int on_device);
int gandalf_set_time(gandalf_ctx* ctx, double t, long long step);

/* Right-hand side at the current state, boundary layout, without advancing it:
 *   dw_hat[2] = N^+, N^-  : -1/2 [ {xi+,w-} + {xi-,w+} -+ lap_perp {xi+,xi-} ]  (Eq. 1 / Eq. 12 RHS,
 *               vorticity units, the linear -+ i kz vA w term is NOT included -- the integrating
 *               factor carries it), each bracket evaluated pseudo-spectrally and dealiased
 *               [PAPER.md:49, 140-142, 154, 251-257];
 *   dg_hat[M] = H_m = -{Phi,g_m} + sqrt(m/2){Psi,g_{m-1}} + sqrt((m+1)/2){Psi,g_{m+1}}
 *               + s i kz [ g_m - sqrt(m/2) g_{m-1} - sqrt((m+1)/2) g_{m+1} ]   (Eq. 6, no collisions)
 *               [PAPER.md:89-93]. */
int gandalf_rhs(gandalf_ctx* ctx, double* dw_hat, double* dg_hat, int on_device);

/* Advance nsteps complete steps of Algorithm 2 [PAPER.md:297-315]: (CFL dt) -> RHS -> half-step
 * predictor with integrating factors (Eq. 15) and plain RK2 for g_m -> midpoint RHS -> full-step
 * corrector (Alg. 1 l.8-9) -> exponential dissipation (Eq. 17-19) -> forcing increment (Eq. 25).
 * dt > 0: fixed step.  dt <= 0: dt = min(dt_max, cfl * min(Lx/nx, Ly/ny) / max|grad_perp Phi|) recomputed every
 * step ON THE DEVICE from the state at t_n (Eq. 16), no host synchronisation.  If the flow vanishes (max = 0) and
 * dt_max = 0 the step and all later ones are no-ops on the state (dt = 0: it survives unchanged, as in the oracle, which
 * refuses such a step) and every synchronising call returns GANDALF_ERR_CFL until a new state is loaded: gandalf_set_state,
 * gandalf_set_state_raw and gandalf_set_time clear the flag.  Unlike the oracle, the no-op steps are still COUNTED: the step
 * number (and with it the forcing counters) moves on and each appends a history record of the unchanged state at the
 * unchanged time -- the step is enqueued without a host round trip, so the host cannot take it back.
 * One energy record is appended per step to the device-resident history.  The call is
 * asynchronous on the ctx's stream; errors detected on the device (non-finite energy) are
 * reported by gandalf_energy_history / gandalf_energy / gandalf_get_time, which synchronise. */
int gandalf_step(gandalf_ctx* ctx, double dt, int nsteps);

/* Moment-sharded stepping (Q31).  gandalf_step(dt, 1) == gandalf_step_stage(dt, 0) followed by
 * gandalf_step_stage(dt, 1): stage 0 is the RHS at t_n, the dt of this step and the half-step predictor (Alg. 1 l.2-4), stage 1
 * the midpoint RHS, corrector, dissipation, forcing and the energy record (Alg. 1 l.6-9, Alg. 2 l.12-14).  Between the stages
 * (and after stage 1) a sharded run overwrites its halo moments with the neighbours' values:
 *   gandalf_field_ptr(ctx, state, field, &p, &n)  device address and length (complex entries) of one field of the raw retained-
 *       mode array (layout of gandalf_get_state_raw); state 0 = the state at t_n / t_{n+1}, 1 = the half-step (stage) state;
 *       field 0, 1 = w+-, 2+j = local moment j.  The caller copies / sends / receives in place (stream-ordered on ctx's stream
 *       or after synchronising it); the pointers stay valid for the life of the context.
 *   gandalf_halo_refresh(ctx, state)  re-derives what the library keeps besides the raw array for the halo fields (their
 *       z-real hybrid copy, the input of the next RHS evaluation) from the given state.  Call it after the halos were written. */
int gandalf_step_stage(gandalf_ctx* ctx, double dt, int stage);
int gandalf_field_ptr(gandalf_ctx* ctx, int state, int field, void** device_ptr, long long* ncomplex);
int gandalf_halo_refresh(gandalf_ctx* ctx, int state);

/* Energies of the current state (host output, synchronises):
 * out = { E_A, E_plus, E_minus, E_kin, E_mag, W_g } with E_+- = 1/4 sum_k kperp^2 |xi+-|^2,
 * E_A = E_plus + E_minus, E_kin = 1/2 sum kperp^2 |Phi|^2, E_mag = 1/2 sum kperp^2 |Psi|^2,
 * W_g = 1/2 sum_m sum_k |g_m|^2, sums over the full spectrum [PAPER.md:115, 383, 442; Q14].
 * The other two diagnostics PAPER.md:383 names follow from these without another pass over the state: cross-helicity
 * H_c = E_plus - E_minus, residual energy E_r = E_kin - E_mag (the paper gives no formulas; these are the standard Elsasser
 * definitions, Schekochihin et al. 2009, which PAPER.md:115 refers to). */
int gandalf_energy(gandalf_ctx* ctx, double out[6]);

/* Perpendicular shell spectrum [Eq. 26; Q15]: bin j = floor(kperp/dk + 1/2),
 * dk = 2 pi / max(Lx, Ly), summed over kz.  literal_eq26 = 0: mode energy 1/4 kperp^2 (|xi+|^2 +
 * |xi-|^2) (bins sum to E_A); 1: |xi+|^2 + |xi-|^2 as printed.  out: nbins doubles on the HOST. */
int gandalf_kperp_spectrum(gandalf_ctx* ctx, int nbins, int literal_eq26, double* out);

/* The same shell spectrum for callers that must not allocate device memory [Eq. 26; Q15].
 * Everything else in this header needs a gandalf_ctx, and a context (like gandalf_kperp_spectrum itself) gets its buffers from
 * cudaMalloc.  That rules the library out for two kinds of caller: an application that gave all of the GPU's memory to its own
 * pool when it started (a new cudaMalloc fails there, or makes the pool hand memory back), and a diagnostics hook that runs while
 * other streams are busy and must not trigger the device-wide synchronisation cudaMalloc / cudaFree imply.  This one entry point
 * takes no context, allocates nothing and frees nothing: the caller passes the state and the output as DEVICE pointers, and the
 * per-column partial sums go to a fixed array of GANDALF_NOALLOC_MAX_COLUMNS doubles (256 KB) that is part of the library image.
 *   device, stream   where to run; stream = NULL is the legacy default stream.  Two kernels are enqueued; the call does not
 *                    synchronise.  The caller's current device is restored before returning.
 *   nx, ny, nz       grid, as for gandalf_create (powers of two, 8 <= nx, ny <= 512, 2 <= nz <= 512), with
 *                    (nx/3 + 1) * (2 (ny/3) + 1) <= GANDALF_NOALLOC_MAX_COLUMNS: 256 x 256 and 512 x 256 fit, 512 x 512 does not
 *                    and is refused (GANDALF_ERR_INVALID, nothing launched) -- use gandalf_kperp_spectrum there.
 *   Lx, Ly           box lengths (> 0); dk = 2 pi / max(Lx, Ly)
 *   w_raw            device pointer, read only: the vorticities w^+ then w^- on the retained modes, i.e. the first two fields of
 *                    the gandalf_get_state_raw layout (2 * 2 * Kz * Ky * Kx doubles; gandalf_field_ptr(ctx, 0, 0, ..) of a
 *                    context the caller created earlier points at exactly this)
 *   nbins, literal_eq26   as for gandalf_kperp_spectrum (1 <= nbins <= 65535)
 *   out              device pointer, nbins doubles, overwritten; same values as gandalf_kperp_spectrum (same arithmetic and
 *                    summation order)
 *   err, errlen      optional caller buffer for a NUL-terminated message when the return value is not GANDALF_OK (may be NULL, 0)
 * The fixed array is shared: every GPU that loads this library holds its 256 KB until the process exits; all calls on a device
 * use it and it keeps the previous call's contents (harmless: each call writes every entry it later reads); calls that can
 * overlap on the GPU -- two streams with no ordering between them, two host threads -- corrupt each other's sums, so order them.
 * The FIRST call on a device also looks up the array's device address (cudaGetSymbolAddress; the driver may load the library's
 * code on that device then): make it once at start-up, before any stream capture begins.
 * Errors: INVALID (NULL array, bad grid / box / nbins / device, grid beyond the fixed array), CUDA (launch failed). */
#define GANDALF_NOALLOC_MAX_COLUMNS 32768
int gandalf_kperp_spectrum_noalloc(int device, void* stream, int nx, int ny, int nz, double Lx, double Ly,
                                   const double* w_raw, int nbins, int literal_eq26, double* out, char* err, int errlen);

/* Hermite spectrum [Eq. 27: C_m = <|g_m|^2>], instantaneous and volume averaged:
 * C_m = sum_k |g_m(k)|^2 over the full spectrum (so that sum_m C_m = 2 W_g).  out: M doubles on the HOST
 * (nothing is written when M = 0).  SURVEY.md 8(f) rank 1. */
int gandalf_hermite_spectrum(gandalf_ctx* ctx, double* out);

/* Truncation monitor of the Hermite expansion [PAPER.md:269, section 3.5: "GANDALF monitors convergence via the energy ratio
 * E_M/E_total (energy in the single highest retained moment m = M relative to total energy), typically requiring this to fall
 * below 1e-3"; Q32]: *out = E_M / (E_A + W_g) with E_M = 1/2 sum_k |g_{M-1}(k)|^2 (summed over the species).
 * Host output, synchronises.  INVALID when M = 0; UNSUPPORTED on a moment shard (the driver combines the shards' spectra). */
int gandalf_truncation_ratio(gandalf_ctx* ctx, double* out);

/* Parallel spectrum E(k_par) [PAPER.md:385; Q25]: bin j = |n_z|, j = 0..nbins-1, of the Alfvenic mode
 * energy 1/4 kperp^2 (|xi+|^2 + |xi-|^2) summed over (kx, ky) (bins sum to E_A; bins above nz/3 are zero).
 * out: nbins doubles on the HOST. */
int gandalf_kpar_spectrum(gandalf_ctx* ctx, int nbins, double* out);

/* Copy up to max_records of the per-step records {t, E_A, E_plus, E_minus, E_kin, E_mag, W_g}
 * (7 doubles each, oldest first, host output) and the count.  Returns GANDALF_ERR_NONFINITE
 * if any recorded energy is NaN/Inf (records are still copied). */
int gandalf_energy_history(gandalf_ctx* ctx, int max_records, double* t_and_E, int* n);

/* Simulation time, number of completed steps and the last dt used (host output, synchronises). */
int gandalf_get_time(gandalf_ctx* ctx, double* t, long long* step, double* last_dt);

/* Bytes the host-pointer entry points of this context have copied host -> device and device -> host so far (state, RHS, energy
 * and history transfers); bench.py's e2e.h2d_bytes_per_step / d2h_bytes_per_step are differences of these counters. */
int gandalf_transfer_bytes(const gandalf_ctx* ctx, long long* h2d, long long* d2h);

/* Number of kernels this context has launched so far (bench.py's gpu_launches); kernels of a replayed graph count as launched. */
long long gandalf_launch_count(const gandalf_ctx* ctx);

/* Launch path of gandalf_step [Algorithm 2, is the same kernel sequence every step].  enable = 1 (the default):
 * one step is captured into a CUDA graph the first time gandalf_step runs two or more steps (or is called a second time with the
 * same dt) and replayed afterwards -- the launch-bound small grids (BASELINE configs 0-2) step faster, the results are bit for bit
 * those of plain launches (same kernels, same arguments; dt, time and the step number live in device memory).  The graph is rebuilt
 * when dt or the history buffer changes.  Plain launches are used on the legacy default stream (stream = NULL: capture is not allowed
 * there), while per-kernel timing is on, and for gandalf_step_stage.  enable = 0: plain launches; enable = -1: query only.
 * *replays (may be NULL) receives the number of graph launches made so far.  Returns GANDALF_ERR_INVALID for another enable. */
int gandalf_graph_mode(gandalf_ctx* ctx, int enable, long long* replays);

/* Event-timed average duration (ms) of one named kernel class since the last reset; used by
 * bench.py for the roofline line.  which: 0 z-inverse (set_state / after forcing only), 1 y-inverse (P1),
 * 2 x-pass (P2), 3 y-forward (P3), 4 fused z-forward + stage update + z-inverse (P4).
 * Timing is off unless enabled (it inserts events). */
int gandalf_kernel_timing(gandalf_ctx* ctx, int enable);
int gandalf_kernel_time_ms(gandalf_ctx* ctx, int which, double* avg_ms, long long* launches);

/* Measured ceilings of the units the hot path leans on (instrumentation; needs no context; synchronises the device).
 * which = 0: fp64 FMA rate      out = { TFLOP/s, T fp64 instructions/s, ms of the best launch, SM count }
 *         1: lane-group FFT-256 out = { G transforms/s of the plan 16*16 on 16 lanes with 8 register twiddles, 8 warps per SM;
 *                                       the same with all twiddles from shared memory; G transforms/s of the plan 8*8*4 on
 *                                       32 lanes, 16 warps per SM (the x-pass's transform alone: csrc/fft.cuh); ms of the first }
 *         2: tensor-memory load out = { bytes per clock per SM, TB/s over the chip, ms, mean cycles per CTA }
 *         3: shared-memory load out = same four numbers for conflict-free 16-byte loads
 * nout >= 4.  Used by `bench.py --microbench` and for the fp64 ceiling in the bench line. */
int gandalf_microbench(int which, int device, double* out, int nout);

const char* gandalf_last_error(const gandalf_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif  /* GANDALF_H_ */
