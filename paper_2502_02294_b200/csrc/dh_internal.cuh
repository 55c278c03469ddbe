// dh_internal.cuh -- context, error plumbing and launch declarations shared by the .cu files of libdiffhydro.
// Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <vector>

#include "../../include/diffhydro.h"

namespace dh {

void set_error(const char* fmt, ...);

#define DH_CUDA(call)                                                                          \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            dh::set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return (e_ == cudaErrorMemoryAllocation) ? DH_ERR_OOM : DH_ERR_CUDA;               \
        }                                                                                      \
    } while (0)

#define DH_CUFFT(call)                                                              \
    do {                                                                            \
        cufftResult r_ = (call);                                                    \
        if (r_ != CUFFT_SUCCESS) {                                                  \
            dh::set_error("%s:%d: %s -> cufft error %d", __FILE__, __LINE__, #call, (int)r_); \
            return DH_ERR_CUFFT;                                                    \
        }                                                                           \
    } while (0)

#define DH_TRY(call)            \
    do {                        \
        int rc_ = (call);       \
        if (rc_ != DH_OK) return rc_; \
    } while (0)

// Strang table (reading R9): step n uses STRANG[n mod 6].
static const int STRANG[6][3] = {{0, 1, 2}, {2, 1, 0}, {2, 0, 1}, {1, 0, 2}, {1, 2, 0}, {0, 2, 1}};

struct StepScalars { double dtau, kappa, K, A; };

// Per-kernel timing categories of dh_profile_* (names in api.cu, same order).
enum ProfCat {
    PROF_SOURCE_INIT = 0, PROF_DEPOSIT, PROF_FFT_R2C, PROF_GREEN, PROF_FFT_C2R, PROF_KICK_DRIFT,
    PROF_SWEEP_X, PROF_SWEEP_Y, PROF_SWEEP_Z, PROF_SWEEP_X_ADJ, PROF_SWEEP_Y_ADJ, PROF_SWEEP_Z_ADJ,
    PROF_KICK_DRIFT_ADJ, PROF_GREEN_ADJ, PROF_DEPOSIT_ADJ, PROF_AXPY, PROF_DOT3, PROF_FILL, PROF_COPY,
    PROF_FFT_X1, PROF_FFT_X3, PROF_FFT_Y1, PROF_FFT_Y3, PROF_N
};

struct Snapshot {
    float* buf = nullptr;   // 5 N^3 + 6 N_p floats
    double a = 0, dt_prev = 0;
    int64_t step = 0;
};

// What the VJP of one step needs besides the step's input state: g' of the start-of-step state and the inputs of
// sweeps 2 and 3.  Kept per step of a segment by the reverse pass when memory allows (13 N^3 floats), else recomputed.
struct StepTape {
    float* buf = nullptr;   // (3 + 2 nc) N^3 floats: g'_x, g'_y, g'_z, sweep-2 input (nc), sweep-3 input (nc)
    float* gp[3] = {nullptr, nullptr, nullptr};
    float* sw[2][6] = {};
};

// g' of one step of a checkpointed run, kept from the forward pass for the reverse pass.
struct GravStore {
    float* buf = nullptr;   // 3 N^3 floats
    float* gp[3] = {nullptr, nullptr, nullptr};
};

// The particles entering one step of a checkpointed run, kept from the forward pass for the reverse pass.
struct PartStore {
    float* buf = nullptr;   // 6 n_part floats
    float* p[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
};

}  // namespace dh

struct dh_ctx {
    int N = 0;
    int nc = 5;                    // gas fields per cell: 5, or 6 with dh_options.dual_energy (the sixth is q = a^2 rho e)
    int64_t n3 = 0, np = 0;
    int nps = 0;
    double box = 0, gamma = 0, dx = 0;
    dh_cosmology cosmo{};
    dh_options opt{};
    double f_b = 0, m_p = 0, rho_bar = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    // Side stream: the particle update of a step shares only the read-only g' with the step's three sweeps (reading
    // R16), so it runs beside them; forked from and joined back into `stream` with events inside every step, so callers
    // still see one stream.
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    int sm_count = 148;
    int64_t launches = 0;
    int64_t bytes = 0;
    // tuning knobs (dh_tune): 0 = built-in choice
    int tune_march_s_fwd = 0, tune_march_s_adj = 0;   // segment length of the marching y/z sweeps
    int tune_prime = 1;                               // 0: every step of dh_run initialises its Poisson source itself
    int tune_overlap = 1;                             // 0: kick_drift on the main stream, after which the sweeps start
    int tune_de_march = 1;                            // 0: dual-energy y/z forward sweeps on the chain tile kernels
    int tune_deposit_tile = 0;                        // 1: shared-memory tile deposit (the A/B of profiles/r02.md)

    cufftHandle plan_r2c = 0, plan_c2r = 0;
    bool plans = false;
    void* fft_work = nullptr;
    size_t fft_work_bytes = 0;
    float2* fft_tw = nullptr;      // own FFT passes (fft.cu): (cos, sin)(2 pi j / N)
    bool own_fft = false;          // grid side is a power of two in [32, 1024]
    int tune_own_fft = 1;          // 0: Poisson solve through cuFFT + green kernels (pm.cu)

    // scratch
    float* delta = nullptr;        // N^3 real (Poisson source / delta_bar)
    float2* spec[4] = {nullptr, nullptr, nullptr, nullptr};   // half spectra: [0] delta^, [1..3] g^_d
    float* gp[3] = {nullptr, nullptr, nullptr};               // g'_d
    float* gas_tmp[6] = {};        // output of sweep 1
    float* gas_tmp2[6] = {};       // output of sweep 2 (sweep 3 writes the state)
    float* cmax_step = nullptr;    // 3 floats (device) for dh_step when the caller passes NULL
    float* cmax_log = nullptr;     // 3 * cmax_cap floats
    int cmax_cap = 0;
    int cmax_n = 0;
    std::vector<double> ps_count;  // modes per bin (a property of the grid), filled by the first power-spectrum call
    double* scal_log = nullptr;    // per-step copies of scal_dev (8 doubles each) of the last dh_run_vjp with want_dsched
    int scal_log_cap = 0;
    std::vector<double> step_dp;   // host: per step (dgamma, dDtau, dkappa, dK, dA) of the last dh_run_vjp with want_dsched
    double* sg_scal = nullptr;     // 4 doubles: parameter cotangents of the sub-grid step
    double* ps_bins = nullptr;     // power spectrum: [2][N/2+1] doubles + (behind them) N/2+1 floats of the transpose's table
    double* scal_dev = nullptr;    // 8 doubles: (lam_b, kap_b, gamma_b, K_b, dtau_drift_b, A_b, spare, spare)

    // adjoint scratch (allocated on first use)
    float* sw_in[2][6] = {};       // inputs of sweeps 2 and 3
    float* gpb[3] = {nullptr, nullptr, nullptr};   // cotangent of g'
    float* cot_tmp[6] = {};        // cotangent ping-pong
    float* part_tmp[6] = {};       // particle scratch for the recompute
    bool adj_alloc = false;

    // checkpoints of the last dh_run
    std::vector<dh::Snapshot> snaps;     // segment snapshots
    std::vector<dh::Snapshot> seg;       // per-step inputs inside one segment (reverse pass)
    std::vector<dh::StepTape> tapes;     // per-step intermediates inside one segment (reverse pass)
    int tune_tape = 1;                   // 0: always recompute g' and the sweep inputs in the step VJP
    std::vector<dh::GravStore> gstore;   // per-step g' of the last checkpointed dh_run
    int tune_gstore = 1;                 // 0: never keep g' from the forward pass
    bool run_gstore = false;             // the last dh_run filled gstore[0 .. run_n)
    std::vector<dh::PartStore> pstore;   // particles entering step k = 1 .. run_n - 1 of the last checkpointed dh_run
    int tune_pstore = 1;                 // 0: never keep them (the segment re-run repeats kick + drift)
    bool run_pstore = false;             // the last dh_run filled pstore[1 .. run_n)
    std::vector<double> run_a, run_dt;
    int run_n = 0, run_stride = 0;
    double run_a0 = 0, run_dtprev0 = 0;
    int64_t run_step0 = 0;
    bool run_valid = false;

    // optional per-kernel CUDA-event timing (dh_profile_enable): pairs of events around every launch
    bool prof_on = false;
    std::vector<cudaEvent_t> prof_ev;    // 2 per recorded launch
    std::vector<int> prof_cat;
    size_t prof_used = 0;                // launches recorded since the last read

    // host-variant device buffers
    float* hv_state = nullptr;     // 5 N^3 + 6 N_p
    float* hv_cot = nullptr;
    float* hv_mesh = nullptr;      // 3 N^3: delta_init, data (then the gradient), noise variance of dh_value_and_grad_host
};

namespace dh {

// RAII timing scope: records an event pair on the context's stream around whatever is launched inside it.
struct Prof {
    dh_ctx* c; size_t slot; bool on;
    Prof(dh_ctx* ctx, int cat) : c(ctx), slot(0), on(ctx->prof_on) {
        if (!on) return;
        slot = c->prof_used;
        if (c->prof_ev.size() < 2 * (slot + 1)) {
            cudaEvent_t a, b;
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { on = false; return; }
            c->prof_ev.push_back(a); c->prof_ev.push_back(b);
            c->prof_cat.push_back(cat);
        }
        c->prof_cat[slot] = cat;
        c->prof_used = slot + 1;
        cudaEventRecord(c->prof_ev[2 * slot], c->stream);
    }
    ~Prof() { if (on) cudaEventRecord(c->prof_ev[2 * slot + 1], c->stream); }
};

int dev_alloc(dh_ctx* c, void** p, size_t bytes);
void dev_free(dh_ctx* c, void* p, size_t bytes);

StepScalars step_scalars(const dh_cosmology& co, double a_i, double a_next, double dt, double dt_prev);

// ---- kernels (sweep.cu) ----
// delta_out (may be NULL): also write delta = [gas] rho' - rho_bar, the next step's Poisson source
// (with dh_options.dual_energy the arrays hold six pointers and the calls go to the kernels of sweep_de.cu)
int launch_sweep(dh_ctx* c, int d, float* const* in, const float* g, float lam, float kap, float* const* out,
                 float* cmax, float* delta_out = nullptr);
int launch_sweep_vjp(dh_ctx* c, int d, float* const* in, const float* g, float lam, float kap,
                     float* const* cot_out, float* const* cot_in, float* g_bar, double* scal_bar);
// ---- kernels (pm.cu) ----
// primed: delta already holds [gas] rho_gas - rho_bar (written by the previous step's last sweep): deposit only
int launch_deposit(dh_ctx* c, const float* rho_gas, const float* x, const float* y, const float* z, float* delta,
                   bool primed = false);
int launch_green(dh_ctx* c, const float2* dhat, float A, float2* const ghat[3]);
int launch_green_adj(dh_ctx* c, float2* const gbhat[3], float A, float2* dbhat);
int launch_kick_drift(dh_ctx* c, float* const g[3], float* const part[6], float* const part_out[6], float K,
                      float dtau_dx);
int launch_kick_drift_vjp(dh_ctx* c, float* const g[3], float* const part_in[6], float* const cot_out[6],
                          float* const cot_in[6], float* const gbar[3], float K, float dtau_dx, double* scal_bar);
int launch_deposit_vjp(dh_ctx* c, const float* delta_bar, float* const part_in[6], float* rho_bar_gas,
                       float* const xbar[3]);
int launch_dot3(dh_ctx* c, float* const a[3], float* const b[3], double scale, double* out);
int launch_cell_index(dh_ctx* c, const float* x, int64_t n, int32_t* i0, int32_t* i1);
int launch_fill(dh_ctx* c, float* p, int64_t n, float v);
int launch_axpy(dh_ctx* c, const float* x, float* y, float a);
// ---- initial-condition map (ic.cu) ----
int launch_ic_state(dh_ctx* c, const float* delta, float* const psi[3], float* const gas[5], float* const part[6],
                    float vf, float e0);
int launch_ic_state_vjp(dh_ctx* c, const float* delta, float* const psi[3], const float* const cot_gas[5],
                        const float* const cot_part[6], float* grad, float* const psi_b[3], float vf, float e0);

int launch_data_term(dh_ctx* c, int observable, const float* const gas[5], const float* data, const float* noise_var,
                     float scale, float weight, float* const cot[5], double* loss_dev);

int launch_sum_arrays(dh_ctx* c, const float* const* arrays, int na, int64_t n, double* out_dev);

// ---- sub-grid step (subgrid.cu) ----
int launch_subgrid(dh_ctx* c, float* const gas[5], const float* g0, const float* g1, const dh_subgrid_params& q,
                   float* zout);
int launch_subgrid_vjp(dh_ctx* c, float* const gas_in[5], const float* g0, const float* g1, const dh_subgrid_params& q,
                       float* const cot[5], const float* cot_z, double* scal4_dev);
int launch_cic_readout(dh_ctx* c, const float* mesh, float* const pos[3], float* aux);

// ---- own FFT passes fused with the Green multiply (fft.cu) ----
bool own_fft_supported(int N);
int own_fft_init(dh_ctx* c);
int own_poisson_forward(dh_ctx* c, const float* delta, float A, float* const g_out[3]);
int own_poisson_adjoint(dh_ctx* c, float* const g_bar[3], float A, float* delta_bar);
int own_power_spectrum(dh_ctx* c, const float* field, double* bins_dev /* [2][N/2+1]: sum w |F|^2, sum w */);
int own_power_spectrum_adjoint(dh_ctx* c, const float* field, const float* gtab_dev /* [N/2+1] */, float* field_bar);

int poisson_forward(dh_ctx* c, const float* delta, float A, float* const g_out[3]);
int poisson_adjoint(dh_ctx* c, float* const g_bar[3], float A, float* delta_bar);

}  // namespace dh
