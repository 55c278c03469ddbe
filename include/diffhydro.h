/* diffhydro.h -- C ABI of the B200-native diffHydro hot path.
 *
 * One coupled time step of the relaxing-TVD finite-volume Euler solver and the dark-matter particle-mesh gravity
 * solver of Horowitz & Lukic, arXiv 2502.02294 (section 2.2 Eq. 2-3, section 2.3 Eq. 4-20), and that
 * step's reverse-mode adjoint (section 2.3.5, :198-220), as hand-written CUDA kernels for sm_100a.
 * The Poisson solve runs on the library's own 1-D FFT passes with the Green multiply fused into the z pass (grids
 * whose side is a power of two); other sides fall back to cuFFT for the 3-D real transforms only.  There is no CPU
 * fallback: dh_init fails with DH_ERR_NO_DEVICE when no sm_100 device is present.
 *
 * Conventions
 *   - Every entry point returns int: DH_OK (0) or a negative DH_ERR_* code; dh_last_error() gives a thread-local
 *     message.  No exception crosses this boundary.
 *   - "device pointer" = CUDA global memory owned by the CALLER (e.g. a torch tensor); the library never frees
 *     it.  "host pointer" = ordinary host memory.  The context owns cuFFT plans, scratch meshes and snapshots.
 *   - Grids are N^3 fp32, C order [z][y][x], x fastest.  Gas state = 5 conserved fields in the paper's variables
 *     (PAPER.md:95-97): gas[0] = rho_b, gas[1..3] = a rho_b U_{x,y,z}, gas[4] = a^2 rho_b E.  Particles are
 *     structure-of-arrays: part[0..2] = comoving position in GRID UNITS [0, N), part[3..5] = w = a u = a^2 dx/dt in
 *     km/s (Eq. 2-3).  Density unit = mean comoving total matter density; length h^-1 Mpc; velocity
 *     km/s; time (h^-1 Mpc)/(km/s).
 *   - All work is issued on the one CUDA stream given at dh_init (NULL: the legacy default stream) and is asynchronous
 *     unless stated; calls that return host scalars synchronise that stream.
 *   - Readings of the paper where it is silent or garbled (R1..R27) are listed in DESIGN.md.
 */
#ifndef DIFFHYDRO_H
#define DIFFHYDRO_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DH_OK 0
#define DH_ERR_INVALID (-1)    /* bad argument / unsupported size */
#define DH_ERR_NO_DEVICE (-2)  /* no CUDA device of compute capability 10.x */
#define DH_ERR_CUDA (-3)
#define DH_ERR_CUFFT (-4)
#define DH_ERR_NONFINITE (-5)  /* the CFL reduction saw NaN/Inf */
#define DH_ERR_OOM (-6)
#define DH_ERR_STATE (-7)      /* call order (e.g. dh_run_vjp without a checkpointed dh_run) */

typedef struct dh_ctx dh_ctx;

/* Flat matter + Lambda background.  static_mode = 1: a == 1 for all time (non-cosmological runs, config 1). */
typedef struct {
    double H0;       /* km/s per h^-1 Mpc (100) */
    double Omega_m;  /* total matter */
    double Omega_b;  /* baryons; f_b = Omega_b / Omega_m sets the particle mass (1 - f_b) N^3 / N_p */
    double Omega_L;
    int32_t static_mode;
} dh_cosmology;

typedef struct {
    int32_t n_part_side;          /* particles per side, N_p = n_part_side^3; 0 = no particles */
    int32_t gravity_on;           /* 0: no Poisson solve, g' = 0 */
    int32_t hydro_on;             /* 0: particles only */
    int32_t gas_sources_gravity;  /* 1: delta_tot includes rho_gas (reading R12) */
    double e_floor;               /* floor of the DERIVED thermal energy e~ used in fluxes (reading R17), > 0 */
    double lim_eps;               /* epsilon of the altered Van Leer limiter, Eq. 18 (reading R8) */
    void* cuda_stream;            /* cudaStream_t to issue all work on; NULL = the legacy default stream */
    int32_t want_dA;              /* 1: dh_step_vjp also accumulates dparams.dA (one extra pass over g') */
    int32_t want_dsched;          /* 1: the sweep adjoints also accumulate the cotangents of Dtau and kappa (dparams.dDtau,
                                   * dparams.dkappa: needed for cosmological-parameter gradients); 0: they are skipped (about
                                   * 6 % of the adjoint sweeps' arithmetic) and both fields come back as NaN */
    int32_t dual_energy;          /* 1: dual-energy formalism (readings R33-R36 of DESIGN.md): a sixth mesh field
                                   * q = a^2 rho_b e (dh_state.eint) is advanced by the internal-energy equation whose source
                                   * S_e = -p div U the paper prints at :101, and replaces eps - |m|^2/(2 rho) in the pressure
                                   * and the freezing speed wherever the thermal energy is less than dual_eta of the total.
                                   * The five conserved fields keep their equations.  0: single energy (the paper's runs) */
    double dual_eta;              /* thermal fraction below which q is used (customary: 1e-3) */
} dh_options;

/* State of the simulation.  gas/part: caller-owned DEVICE pointers (N^3 and N_p floats each).
 * a, dt_prev, step: host scalars the library updates (S5 of the step: a <- a_next, dt_prev <- dt, step++). */
typedef struct {
    float* gas[5];
    float* part[6];
    double a;        /* scale factor of this state (1 in static mode) */
    double dt_prev;  /* cosmic-time length of the previous step; 0 before the first step (reading R15) */
    int64_t step;    /* step counter; step mod 6 selects the Strang order (reading R9) */
    float* eint;     /* dual_energy = 1 only: caller-owned DEVICE pointer, N^3 floats, q = a^2 rho_b e; else ignored (NULL) */
} dh_state;

/* Cotangent of a state: same 11 arrays, caller-owned DEVICE pointers. */
typedef struct {
    float* gas[5];
    float* part[6];
    float* eint;     /* dual_energy = 1 only: cotangent of dh_state.eint; else ignored (NULL) */
} dh_cot;

/* Gradients w.r.t. the scalars of the scheme, ACCUMULATED (+=) by the VJP calls (host struct, fp64).
 * dgamma: adiabatic index (through p~ and c~_s; reading R20).  dDtau, dkappa, dK: the per-step factors
 * Dtau = dt/a_h^2 (drift and hydro), kappa = dt/a_h (gas gravity), K = (dt_prev+dt)/(2 a_i) (particle kick), summed
 * over steps (reading R15).  dA: Poisson amplitude A = 1.5 Omega_m H0^2 (reading R12). */
typedef struct {
    double dgamma, dDtau, dkappa, dK, dA;
} dh_dparams;

/* ---- the four calls of the north star (+ dh_run_vjp, which consumes dh_run's checkpoints) ------------------- */

/* Create a context for an N^3 grid in a periodic box of side `box` (h^-1 Mpc) with adiabatic index gamma.
 * Allocates the scratch meshes (and, for a side that is not a power of two, the cuFFT R2C/C2R plans; a power-of-two
 * side makes them only when dh_tune("own_fft", 0) asks for the cuFFT route).  grid_n must be a multiple of 32,
 * 32 <= grid_n <= 1024 (a warp's 32 lanes are 32 consecutive x in every mesh kernel).
 * Errors: DH_ERR_INVALID, DH_ERR_NO_DEVICE, DH_ERR_CUFFT, DH_ERR_OOM. */
int dh_init(dh_ctx** out, int grid_n, double box, double gamma, const dh_cosmology* cosmo, const dh_options* opt);
int dh_free(dh_ctx* ctx);

/* One coupled step in place (Eq. 2-3, 8-18):
 *   S1 delta_tot = rho_gas - rho_bar + CIC deposit of the particles
 *   S2 g'_d = IFFT( i k_d A delta^ / k^2 )
 *   S3 w += K g'(x);  x += w Dtau/dx, wrapped                            (Eq. 2-3)
 *   S4 three 1-D relaxing-TVD sweeps in Strang order, each with its gravity source (Eq. 8-18)
 * dt = cosmic-time length of the step, a = scale factor at the END of the step.
 * cfl_cmax_out: DEVICE pointer to 3 floats (or NULL): max freezing speed |v~_d| + c~_s over the input of each of
 * the three sweeps, in sweep order (Eq. 19-20).  Asynchronous. */
int dh_step(dh_ctx* ctx, dh_state* state, double dt, double a, float* cfl_cmax_out);

/* Reverse-mode adjoint of dh_step.  state_checkpoint: the step's INPUT state (its a, dt_prev, step are used; its
 * arrays are read only); intermediates are recomputed.  cotangent_out: cotangent of the step's OUTPUT state (read
 * only).  cotangent_in: receives the cotangent of the INPUT state (overwritten; may alias cotangent_out).
 * dparams: accumulated.  Synchronises the stream (host scalars are returned). */
int dh_step_vjp(dh_ctx* ctx, const dh_state* state_checkpoint, double dt, double a, const dh_cot* cotangent_out,
                dh_cot* cotangent_in, dh_dparams* dparams);

/* n_steps forward steps; a_sched[k] = scale factor at the END of step k, dt_sched[k] = its cosmic-time length (host
 * arrays).  checkpoint_stride > 0: a snapshot of the state is stored in the context before steps 0, stride,
 * 2 stride, ... for dh_run_vjp; <= 0: none.  With a stride, and while the device has the room, every
 * step's g' and the particles entering it are kept too (dh_tune "gstore", "pstore": 12 + 24 bytes per cell and step),
 * which the reverse pass then does not recompute; the caller's particle arrays receive the final particles from the
 * last step (they are not updated step by step).  The per-sweep CFL maxima are kept in the context (dh_get_cmax).  Synchronises at the end and returns DH_ERR_NONFINITE if any maximum is NaN/Inf. */
int dh_run(dh_ctx* ctx, dh_state* state, const double* a_sched, const double* dt_sched, int n_steps,
           int checkpoint_stride);

/* Reverse sweep over the last checkpointed dh_run: for each segment (last first) re-run the forward from its
 * snapshot keeping every step's input, then apply the step VJP in reverse (recompute-from-checkpoint schedule).
 * cot_final: cotangent of the final state (read only); cot_initial: cotangent of the initial state (overwritten; may
 * alias cot_final); dparams accumulated.  Synchronises. */
int dh_run_vjp(dh_ctx* ctx, const dh_cot* cot_final, dh_cot* cot_initial, dh_dparams* dparams);

/* Optional: allocate now everything a dh_run(n_steps, checkpoint_stride) + dh_run_vjp pair will need (snapshot pool,
 * in-segment states, adjoint scratch, CFL log, and -- each only if the device can hold it, see dh_tune -- the tapes of
 * one segment, the per-step g' store and the per-step particle store), so that neither call allocates.  Invalidates the
 * last run (dh_run_vjp then needs a new dh_run).  Errors: DH_ERR_OOM. */
int dh_reserve(dh_ctx* ctx, int n_steps, int checkpoint_stride);

/* ---- host-buffer variants (end-to-end path: host <-> device copies inside the call) ------------------------- */

/* gas_host: 5 N^3 floats (6 N^3 with dual_energy: q last), part_host: 6 N_p floats (HOST, pinned or pageable), updated in
 * place with the final state.
 * a, dt_prev, step: host scalars of the state, updated. */
int dh_run_host(dh_ctx* ctx, float* gas_host, float* part_host, double* a, double* dt_prev, int64_t* step,
                const double* a_sched, const double* dt_sched, int n_steps, int checkpoint_stride);
/* cot_gas_host / cot_part_host: cotangent of the final state on entry, of the initial state on exit (HOST). */
int dh_run_vjp_host(dh_ctx* ctx, float* cot_gas_host, float* cot_part_host, dh_dparams* dparams);

/* ---- helpers ------------------------------------------------------------------------------------------------ */
const char* dh_last_error(void);
/* out (HOST): 3 * n floats, the CFL maxima of the last dh_run's first n steps. */
int dh_get_cmax(dh_ctx* ctx, float* out, int n);
/* Uniform-in-ln(a) schedule: a_out[0..n] = a0 exp(k r), dt_out[k] = t(a_{k+1}) - t(a_k); EdS closed form, else
 * Simpson quadrature of dt = da / (a H(a)).  HOST arrays. */
int dh_schedule_lna(const dh_cosmology* cosmo, double a0, double a1, int n, double* a_out, double* dt_out);
/* Per-step factors of reading R15: out[4] = (Dtau, kappa, K, A).  HOST. */
int dh_step_scalars(const dh_cosmology* cosmo, double a_i, double a_next, double dt, double dt_prev, double* out);
/* CIC cell indices of n fp32 positions (DEVICE in, DEVICE out): i0 = floor(x - 1/2) mod N, i1 = (i0 + 1) mod N, the
 * very function the deposit / gather kernels use (bit-exact test, reading R22). */
int dh_debug_cell_index(dh_ctx* ctx, const float* x_dev, int64_t n, int32_t* i0_dev, int32_t* i1_dev);
/* Bytes of device memory the context currently holds (scratch + snapshots). */
int64_t dh_device_bytes(dh_ctx* ctx);
/* Number of kernels this library has launched on the context since dh_init (the gpu_launches count of bench.py);
 * cuFFT's internal kernels are not counted. */
int64_t dh_launch_count(dh_ctx* ctx);
int dh_sync(dh_ctx* ctx);
/* Conserved sums of a state (the per-step diagnostics of a run: they are what the scheme keeps to round-off without
 * gravity, Eq. 8): out (HOST, 8 doubles) = (sum rho, sum m_x, sum m_y, sum m_z, sum eps, m_p sum w_x, m_p sum w_y,
 * m_p sum w_z), fp64 accumulation on the device.  Synchronises the stream. */
int dh_conserved_sums(dh_ctx* ctx, const dh_state* state, double* out);
/* The same eight sums for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): no context (dh_init allocates), no cudaMalloc / cudaFree / allocating library routine, no synchronisation.
 *   gas[5]   DEVICE, n_cells floats each: rho, m_x, m_y, m_z, eps;   w[3]  DEVICE, n_part floats each (may be NULL when
 *   n_part = 0);   m_p  particle mass;   out  DEVICE, 8 doubles, written by the kernel (same order as dh_conserved_sums);
 *   cuda_stream  a cudaStream_t or NULL: one memset node + one kernel are enqueued on it, nothing else happens.
 * The per-block partial sums live in a static device array of 512 KiB + 8 B (csrc/noalloc.cu) that every GPU which loads
 * the library holds until the process exits; it serves at most DH_NOALLOC_MAX_ELEMS cells and as many particles (512^3,
 * the largest configuration of BASELINE.json): more is DH_ERR_INVALID with a message naming the limit, as are null
 * pointers and n_cells <= 0.  The first call on each device looks the array's address up (cudaGetSymbolAddress, with that
 * device current): make it outside a stream capture.  Every call on a device shares the array: calls that overlap on the
 * GPU (different streams, or graphs replayed concurrently) race -- serialise them.  The additions are done in an order
 * fixed by the sizes alone (block partials, then the last block adds them in block order): bit-identical from call to
 * call, unlike dh_conserved_sums, whose blocks meet in fp64 atomics. */
#define DH_NOALLOC_MAX_ELEMS 134217728LL
int dh_conserved_sums_noalloc(const float* const gas[5], int64_t n_cells, const float* const w[3], int64_t n_part, double m_p,
                              double* out, void* cuda_stream);
/* Debug aid (compute-sanitizer's initcheck is not available everywhere): fill the context's device buffers with NaN
 * (all-ones bytes).  level 0: pure scratch only (Poisson source and spectra, g' scratch, sweep ping-pong sets, adjoint
 * scratch, the in-segment states and tapes of the reverse pass) -- safe between dh_run and dh_run_vjp; level 1: also what
 * dh_run keeps for dh_run_vjp (snapshots, per-step g', CFL log), which invalidates the last run.  A path that reads a
 * buffer before writing it then returns NaN instead of stale numbers.  Asynchronous on the context's stream. */
int dh_debug_poison(dh_ctx* ctx, int level);
/* Launch-geometry knobs (performance only; results stay within the parity tolerances).  key (HOST string):
 *   "march_s_fwd", "march_s_adj": cells per thread segment of the marching y/z sweeps (0 = built-in choice);
 *   "tape": 0 makes dh_run_vjp recompute g' and the sweep inputs inside every step VJP instead of keeping them for
 *           the steps of the segment being reversed (13 N^3 floats per step of a segment; default 1, falls back to
 *           recomputation by itself when the device cannot hold them);
 *   "gstore": 0 makes a checkpointed dh_run NOT keep every step's g' (3 N^3 floats per step of the run) for
 *           dh_run_vjp, which then repeats deposit + Poisson solve in the segment re-run (default 1, same fallback);
 *   "pstore": 0 makes a checkpointed dh_run NOT keep the particles entering every step (6 n_part floats per step of the
 *           run; its kick + drift then writes the next step's slot directly, no copy) for dh_run_vjp, whose segment re-run
 *           then repeats the particle update (default 1; taken only while the device keeps room for the snapshots,
 *           in-segment states, tapes and adjoint scratch the reverse pass still has to allocate, else the same fallback);
 *   "own_fft": 0 routes the Poisson solve through cuFFT (1 R2C + multiply kernel + 3 C2R) instead of the library's own
 *           FFT passes fused with the Green multiply (default 1 when grid_n is a power of two); the cuFFT plans are
 *           made by this call when they do not exist yet (DH_ERR_CUFFT / DH_ERR_OOM);
 *   "overlap": 0 keeps the particle update of a step on the caller's stream, before the sweeps, instead of forking it
 *           onto the context's side stream beside them (default 1);
 *   "prime": 0 makes every step of dh_run initialise its own Poisson source instead of letting the previous step's last
 *           sweep write it (default 1; bit-identical either way);
 *   "de_march": 0 routes the y/z sweeps of the dual-energy variant (forward; adjoint when want_dsched = 0) through the
 *           chain tile kernels instead of the marching pipelines (default 1; 2.0 - 2.6 times slower per sweep, same
 *           numbers to rounding);
 *   "deposit_tile": 1 routes the deposit through a shared-memory tile per brick of 32 x 8 x 8 lattice sites (the A/B of
 *           profiles/r02.md: three times slower than the default run-aggregated RED; 2: the same tile in 32-bit fixed
 *           point; default 0).
 * Unknown key: DH_ERR_INVALID. */
int dh_tune(dh_ctx* ctx, const char* key, int value);
/* Optional per-kernel timing: while enabled, every kernel / cuFFT / copy the library issues is bracketed by a pair of
 * CUDA events on the context's stream.  dh_profile_read synchronises, adds the elapsed milliseconds and launch counts
 * per category into ms_out / count_out (HOST arrays of dh_profile_categories() entries, overwritten) and clears the
 * record.  dh_profile_name(i): static string, NULL when i is out of range. */
int dh_profile_enable(dh_ctx* ctx, int on);
int dh_profile_categories(void);
const char* dh_profile_name(int i);
int dh_profile_read(dh_ctx* ctx, double* ms_out, int64_t* count_out);

/* ---- single kernels of the path (same kernels dh_step / dh_step_vjp launch; for parity tests and profiling) --
 * All pointers DEVICE.  d = sweep axis 0/1/2 = x/y/z.  lam = Dtau/dx, kap = kappa. */
/* SWEEP_d: gas_out = sweep(gas_in, g) (g may be NULL: no source); cmax_out: 1 float, max-combined (caller zeroes). */
int dh_sweep(dh_ctx* ctx, int d, float* const gas_in[5], const float* g, double lam, double kap, float* const gas_out[5],
             float* cmax_out);
/* Adjoint of SWEEP_d: cot_in overwritten, g_bar overwritten (may be NULL iff g is NULL);
 * scal_bar: DEVICE double[3] += (lam_bar, kap_bar, gamma_bar). */
int dh_sweep_vjp(dh_ctx* ctx, int d, float* const gas_in[5], const float* g, double lam, double kap,
                 float* const cot_out[5], float* const cot_in[5], float* g_bar, double* scal_bar);
/* The same two calls for a context with dual_energy = 1: six fields (rho, m_x, m_y, m_z, eps, q) in and out. */
int dh_sweep_de(dh_ctx* ctx, int d, float* const gas_in[6], const float* g, double lam, double kap,
                float* const gas_out[6], float* cmax_out);
int dh_sweep_de_vjp(dh_ctx* ctx, int d, float* const gas_in[6], const float* g, double lam, double kap,
                    float* const cot_out[6], float* const cot_in[6], float* g_bar, double* scal_bar);
/* delta_tot = [gas_sources_gravity] rho_gas - rho_bar + m_p CIC(pos) (rho_gas may be NULL). */
int dh_deposit(dh_ctx* ctx, const float* rho_gas, float* const pos[3], float* delta_out);
/* g'_d (3 meshes) from delta (delta is not modified). */
int dh_poisson(dh_ctx* ctx, const float* delta, double A, float* const g_out[3]);
/* delta_bar = sum_d G_d^T g_bar_d. */
int dh_poisson_vjp(dh_ctx* ctx, float* const g_bar[3], double A, float* delta_bar_out);
/* S3 in place on part[6]. */
int dh_kick_drift(dh_ctx* ctx, float* const g[3], float* const part[6], double K, double dtau_over_dx);

/* ---- the step on the input side of the path: initial-condition map and its transpose ----
 * PAPER.md:49 (section 2.1): initial conditions by Lagrangian perturbation theory; reading R19 of DESIGN.md: first
 * order (the Zel'dovich map) of a density contrast delta_init given at scale factor a0, one particle per cell:
 *   psi^_d = i k~_d delta^ / k^2;  x = wrap(q + psi/dx), w = vel_factor psi;
 *   rho = f_b (1 + delta), m = rho w, eps = rho (e_tilde0 + |w|^2 / 2),   f_b = Omega_b / Omega_m of dh_init.
 * delta_init: DEVICE, N^3 floats, [z][y][x], not modified.  vel_factor = a0^2 H(a0) f(a0) (EdS: H0 sqrt(a0)), km/s per
 * h^-1 Mpc; e_tilde0 = a0^2 times the initial thermal energy per unit mass.  state_out: caller-owned DEVICE arrays,
 * overwritten; its scalars are set to (a0, dt_prev = 0, step = 0).  Needs gravity_on and n_part_side == grid_n, else
 * DH_ERR_INVALID.  Asynchronous on the context's stream. */
int dh_ic_zeldovich(dh_ctx* ctx, const float* delta_init, double a0, double vel_factor, double e_tilde0,
                    dh_state* state_out);
/* The two scalar arguments above from physical inputs (HOST only, fp64, no device work; readings R18, R19, R27):
 *   *vel_factor = a0^2 H(a0) f(a0), f = dlnD/dlna the linear growth rate of the matter + curvature + Lambda background of
 *                 `cosmo` (Einstein-de Sitter: H0 sqrt(a0));
 *   *e_tilde0   = a0^2 k_B T0 / ((gamma - 1) mu m_p) in (km/s)^2, T0 in K, mu the mean molecular weight (0.59 ionised).
 * Either output may be NULL.  Errors: DH_ERR_INVALID. */
int dh_ic_factors(const dh_cosmology* cosmo, double a0, double T0, double gamma, double mu, double* vel_factor,
                  double* e_tilde0);
/* Transpose of the Jacobian of dh_ic_zeldovich at delta_init applied to cot_state (gas cotangents required, particle
 * cotangent pointers may be NULL = zero): grad_delta (DEVICE, N^3 floats) is OVERWRITTEN with dL/d delta_init.
 * Together with dh_run_vjp this is "gradient w.r.t. the initial density field" in device memory. */
int dh_ic_zeldovich_vjp(dh_ctx* ctx, const float* delta_init, double vel_factor, double e_tilde0,
                        const dh_cot* cot_state, float* grad_delta);

/* ---- the step on the output side: the data term of Eq. 27 and its cotangent ----
 *   L = weight * sum_i (scale * O_i - data_i)^2 / noise_var_i        (Eq. 27: weight = 1/2)
 * observable 0: O = rho_gas (the loss of BASELINE.json's configs, reading R21); 1: O = eps - |m|^2 / (2 rho), the
 * internal energy density the paper's mock observable delta_b T is proportional to.
 * gas, data, noise_var (NULL = 1 everywhere), cot_gas: DEVICE, N^3 floats each.  cot_gas (may be NULL) is OVERWRITTEN
 * with dL/d(gas) -- the cot_final of dh_run_vjp (its particle cotangent is zero).  loss_out: HOST double, may be NULL;
 * when given the call synchronises the stream, otherwise it is asynchronous. */
int dh_data_term(dh_ctx* ctx, int observable, float* const gas[5], const float* data, const float* noise_var,
                 double scale, double weight, float* const cot_gas[5], double* loss_out);

/* Binned power spectrum of a real mesh field and its transpose ("power spectra of the baryon density
 * using a differentiable routine").  With F = FFT3(field), n the integer wave vector and
 * bin b = round(|n|), b = 1 .. N/2:   P_b = (box^3 / N^6) sum_{k in b} |F_k|^2 / count_b   (sums over the full spectrum),
 * k_b = 2 pi b / box.  field: DEVICE, N^3 floats, not modified.  power_out, count_out (may be NULL), power_bar: HOST,
 * N/2 doubles, index b - 1.  field_bar: DEVICE, N^3 floats, OVERWRITTEN with sum_b power_bar_b dP_b/dfield.
 * Both calls synchronise the stream.  Need gravity_on and a power-of-two grid, else DH_ERR_INVALID. */
int dh_power_spectrum(dh_ctx* ctx, const float* field, double* power_out, double* count_out);
int dh_power_spectrum_vjp(dh_ctx* ctx, const float* field, const double* power_bar, float* field_bar);

/* ---- sub-grid star formation and energy injection (section 2.4, :226-283) ----
 * Applied to the gas state between coupled steps.  Per cell, with delta = rho/rho_mean - 1 and T = t_per_e * e~
 * (e~ = eps/rho - |m|^2/(2 rho^2); the caller folds (gamma-1) mu m_p / (k_B a^2) into t_per_e, reading R27):
 *   pi0 = Pi0 sigma((delta - delta_c)/a_width) sigma((T_c - T)/b_width)                        Eq. 25
 *   z   = relaxed Bernoulli of Eq. 24 with temperature tau and the caller's Gumbel(0,1) draws g0, g1 (inputs: Eq. 22-23)
 *   eps += e_inject * rho * z                   (E_0 per unit star-forming gas mass; the caller folds a^2 and units in)
 * Requires 0 < Pi0 < 1, a_width, b_width, tau, rho_mean > 0. */
typedef struct {
    double rho_mean;   /* mean gas density in the state's units (f_b in the configs' units) */
    double t_per_e;    /* temperature per unit e~ */
    double T_c, delta_c, Pi0, e_inject;   /* the model's parameters (T_c, rho_c as delta_c, Pi_0, E_0), :242 */
    double a_width, b_width, tau;         /* hyper-parameters: sigmoid widths of Eq. 25, Gumbel-softmax temperature (0.1, :273) */
} dh_subgrid_params;
/* gas: DEVICE, eps (gas[4]) updated in place, the other fields read only.  g0, g1: DEVICE, N^3 floats.  z_out (may be
 * NULL): DEVICE N^3 floats, the star-forming field of this step.  If aux and pos are given (DEVICE, N_p floats each) the
 * cloud-in-cell readout of z at the particle positions is ADDED to aux (:244, diagnostic; needs z_out). */
int dh_subgrid_step(dh_ctx* ctx, float* const gas[5], const float* g0, const float* g1, const dh_subgrid_params* par,
                    float* z_out, float* const pos[3], float* aux);
/* Transpose at gas_in = the state BEFORE the injection.  cot_gas: in = cotangent of the step's output, out (in place) =
 * cotangent of gas_in.  cot_z (may be NULL): cotangent of z_out.  dpar_out: HOST double[4] += (dT_c, ddelta_c, dPi0,
 * de_inject); synchronises the stream. */
int dh_subgrid_step_vjp(dh_ctx* ctx, float* const gas_in[5], const float* g0, const float* g1,
                        const dh_subgrid_params* par, float* const cot_gas[5], const float* cot_z, double* dpar_out);

/* ---- the whole chain with HOST buffers (the call of a field-level inference loop) ----
 *   delta_init --dh_ic_zeldovich--> state --dh_run(n_steps, stride)--> final gas --dh_data_term--> L
 * and back: dL/d delta_init through dh_run_vjp and dh_ic_zeldovich_vjp.  delta_init_host, data_host, noise_var_host (may be
 * NULL = 1), grad_delta_host: HOST, N^3 floats each (pinned memory makes the copies asynchronous); only these meshes cross
 * the bus (12 or 16 B/cell up, 4 B/cell down), the 44 B/cell state never leaves the device.  loss_out: HOST double (may be
 * NULL).  dparams: accumulated as in dh_run_vjp (may be NULL).  Synchronises the stream.  Needs gravity_on and one
 * particle per cell; observable, scale, weight as in dh_data_term; a0, vel_factor, e_tilde0 as in dh_ic_zeldovich. */
int dh_value_and_grad_host(dh_ctx* ctx, const float* delta_init_host, const float* data_host, const float* noise_var_host,
                           int observable, double scale, double weight, double a0, double vel_factor, double e_tilde0,
                           const double* a_sched, const double* dt_sched, int n_steps, int checkpoint_stride,
                           float* grad_delta_host, double* loss_out, dh_dparams* dparams);

/* ---- cosmological-parameter gradients through the step scalars (sigma_8, Omega_m) --
 * Every step has its own Dtau, kappa, K, A (reading R15), so chaining to a cosmological parameter needs the cotangents
 * step by step, not their sums.  After a dh_run_vjp with dh_options.want_dsched = 1, dh_get_step_dparams copies them:
 * out: HOST double[n_steps][5] = (dgamma, dDtau, dkappa, dK, dA) of steps 0 .. n_steps-1 of the last run (DH_ERR_STATE if
 * the last dh_run_vjp did not keep them).  dh_chain_cosmology (host only, fp64): for the ln-a schedule of dh_schedule_lna
 * it returns sum_steps sum_s dL/ds * ds/dtheta for theta = Omega_m (Omega_L fixed) and H0, ds/dtheta by central differences
 * of the host's closed-form schedule and step factors; the initial state and the baryon fraction are held fixed (its own dependence on cosmology
 * goes through dh_ic_zeldovich_vjp and the caller's transfer function).  Either output may be NULL.
 * sigma_8: the state depends on it only through delta_init, dL/dsigma_8 = <dL/d delta_init, delta_init> / sigma_8. */
int dh_get_step_dparams(dh_ctx* ctx, double* out, int n_steps);
int dh_chain_cosmology(const dh_cosmology* cosmo, double a0, double a1, int n_steps, const double* step_dparams,
                       double* dOmega_m, double* dH0);

#ifdef __cplusplus
}
#endif
#endif /* DIFFHYDRO_H */
