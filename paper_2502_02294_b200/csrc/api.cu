// api.cu -- the C ABI of libdiffhydro (include/diffhydro.h): context, step scheduler, step VJP, checkpointed run.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "dh_internal.cuh"

namespace dh {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int dev_alloc(dh_ctx* c, void** p, size_t bytes) {
    *p = nullptr;
    if (bytes == 0) return DH_OK;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        set_error("cudaMalloc(%zu bytes) failed: %s", bytes, cudaGetErrorString(e));
        return DH_ERR_OOM;
    }
    c->bytes += (int64_t)bytes;
    return DH_OK;
}

void dev_free(dh_ctx* c, void* p, size_t bytes) {
    if (p) {
        cudaFree(p);
        c->bytes -= (int64_t)bytes;
    }
}

// Per-step factors (reading R15): midpoint rule at a_h = sqrt(a_i a_next) for drift int dt/a^2 and kick int dt/a of
// Eq. 2-3; K is centred on a_i (staggered leapfrog, the first step is the opening half kick).
StepScalars step_scalars(const dh_cosmology& co, double a_i, double a_next, double dt, double dt_prev) {
    StepScalars s;
    if (co.static_mode) {
        s.dtau = dt; s.kappa = dt; s.K = 0.5 * (dt_prev + dt);
    } else {
        const double ah = std::sqrt(a_i * a_next);
        s.dtau = dt / (ah * ah);
        s.kappa = dt / ah;
        s.K = (dt_prev + dt) / (2.0 * a_i);
    }
    s.A = 1.5 * co.Omega_m * co.H0 * co.H0;
    return s;
}

// The gas arrays of a state / cotangent as one list of c->nc pointers (the sixth is q with dual energy).
struct G6 {
    float* p[6];
    G6(const dh_state& s) { for (int k = 0; k < 5; ++k) p[k] = s.gas[k]; p[5] = s.eint; }
    G6(const dh_cot& s) { for (int k = 0; k < 5; ++k) p[k] = s.gas[k]; p[5] = s.eint; }
};

static int alloc_fields(dh_ctx* c, float** arr, int n, size_t count) {
    for (int i = 0; i < n; ++i) DH_TRY(dev_alloc(c, (void**)&arr[i], count * sizeof(float)));
    return DH_OK;
}

static int ensure_adjoint_scratch(dh_ctx* c) {
    if (c->adj_alloc) return DH_OK;
    if (c->opt.hydro_on) {
        DH_TRY(alloc_fields(c, c->sw_in[0], c->nc, c->n3));
        DH_TRY(alloc_fields(c, c->sw_in[1], c->nc, c->n3));
        DH_TRY(alloc_fields(c, c->cot_tmp, c->nc, c->n3));
    }
    if (c->opt.gravity_on) DH_TRY(alloc_fields(c, c->gpb, 3, c->n3));
    c->adj_alloc = true;
    return DH_OK;
}

static size_t state_floats(const dh_ctx* c) { return (size_t)(c->nc * c->n3 + 6 * c->np); }

static int snapshot_store(dh_ctx* c, Snapshot& s, const dh_state* st, float* const* part_src = nullptr) {
    if (!s.buf) DH_TRY(dev_alloc(c, (void**)&s.buf, state_floats(c) * sizeof(float)));
    Prof prof(c, PROF_COPY);
    const G6 g(*st);
    for (int k = 0; k < c->nc; ++k)
        DH_CUDA(cudaMemcpyAsync(s.buf + (size_t)k * c->n3, g.p[k], c->n3 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    for (int k = 0; k < 6 && c->np > 0; ++k)
        DH_CUDA(cudaMemcpyAsync(s.buf + (size_t)c->nc * c->n3 + (size_t)k * c->np, part_src ? part_src[k] : st->part[k], c->np * sizeof(float),
                                cudaMemcpyDeviceToDevice, c->stream));
    s.a = st->a; s.dt_prev = st->dt_prev; s.step = st->step;
    return DH_OK;
}

static void snapshot_view(const dh_ctx* c, const Snapshot& s, dh_state* st) {
    for (int k = 0; k < 5; ++k) st->gas[k] = s.buf + (size_t)k * c->n3;
    st->eint = c->nc == 6 ? s.buf + (size_t)5 * c->n3 : nullptr;
    for (int k = 0; k < 6; ++k) st->part[k] = s.buf + (size_t)c->nc * c->n3 + (size_t)k * c->np;
    st->a = s.a; st->dt_prev = s.dt_prev; st->step = s.step;
}

static void tape_view(const dh_ctx* c, StepTape& t) {
    for (int d = 0; d < 3; ++d) t.gp[d] = t.buf + (size_t)d * c->n3;
    for (int i = 0; i < 2; ++i)
        for (int k = 0; k < c->nc; ++k) t.sw[i][k] = t.buf + (size_t)(3 + c->nc * i + k) * c->n3;
}

// Tapes for the steps of one segment.  All or nothing: if the device cannot hold them the reverse pass falls back to
// recomputing g' and the sweep inputs inside every step VJP (same results, more work).
static bool ensure_tapes(dh_ctx* c, int in_seg) {
    if (!c->tune_tape) return false;
    if ((int)c->tapes.size() < in_seg) c->tapes.resize(in_seg);
    const size_t bytes = (size_t)(3 + 2 * c->nc) * c->n3 * sizeof(float);
    for (int i = 0; i < in_seg; ++i) {
        if (c->tapes[i].buf) continue;
        if (dev_alloc(c, (void**)&c->tapes[i].buf, bytes) != DH_OK) {
            for (auto& t : c->tapes) { dev_free(c, t.buf, bytes); t.buf = nullptr; }
            set_error("");
            return false;
        }
        tape_view(c, c->tapes[i]);
    }
    return true;
}

// Per-step store of g' for a checkpointed run (3 N^3 floats per step): the forward pass writes each step's g' there
// instead of into scratch, so neither the segment re-run nor the step VJP repeats the deposit and the Poisson solve.
// All or nothing, like the tapes: when the device cannot hold n_steps of them the reverse pass recomputes g'.
static bool ensure_gstore(dh_ctx* c, int n_steps) {
    if (!c->tune_gstore || !c->opt.gravity_on) return false;
    const size_t bytes = (size_t)3 * c->n3 * sizeof(float);
    if ((int)c->gstore.size() < n_steps) c->gstore.resize(n_steps);
    for (int i = 0; i < n_steps; ++i) {
        GravStore& g = c->gstore[i];
        if (g.buf) continue;
        if (dev_alloc(c, (void**)&g.buf, bytes) != DH_OK) {
            for (auto& t : c->gstore) { dev_free(c, t.buf, bytes); t.buf = nullptr; }
            c->gstore.clear();
            set_error("");
            return false;
        }
        for (int d = 0; d < 3; ++d) g.gp[d] = g.buf + (size_t)d * c->n3;
    }
    return true;
}

// Per-step store of the particles (6 n_part floats per step of the run): dh_run's kick + drift of step k writes straight
// into the slot of step k + 1 (no copy; the caller's arrays get the final particles from the last step), so the segment
// re-run of the reverse pass has no particle update left to repeat.  All or nothing, and only when the device keeps room
// for what the reverse pass still has to allocate (snapshots, in-segment states, tapes, adjoint scratch): losing the
// tapes to this store would cost more than it saves.
static bool ensure_pstore(dh_ctx* c, int n_steps, int stride) {
    if (!c->tune_pstore || c->np <= 0 || n_steps < 2 || stride <= 0) return false;
    const size_t bytes = (size_t)6 * c->np * sizeof(float);
    if ((int)c->pstore.size() < n_steps) c->pstore.resize(n_steps);
    size_t missing = 0;
    for (int i = 1; i < n_steps; ++i) missing += c->pstore[i].buf ? 0 : 1;
    if (missing > 0) {
        const size_t mesh = (size_t)c->n3 * sizeof(float), state = state_floats(c) * sizeof(float);
        const int in_seg = stride < n_steps ? stride : n_steps, nseg = (n_steps + stride - 1) / stride;
        size_t later = c->adj_alloc ? 0 : (size_t)(3 * c->nc + 3) * mesh;
        for (int i = 0; i < nseg; ++i) later += (i < (int)c->snaps.size() && c->snaps[i].buf) ? 0 : state;
        for (int i = 1; i < in_seg; ++i) later += (i < (int)c->seg.size() && c->seg[i].buf) ? 0 : state;
        if (c->tune_tape)
            for (int i = 0; i < in_seg; ++i) later += (i < (int)c->tapes.size() && c->tapes[i].buf) ? 0 : (size_t)(3 + 2 * c->nc) * mesh;
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); return false; }
        if (free_b < missing * bytes + later + ((size_t)1 << 30)) return false;
    }
    for (int i = 1; i < n_steps; ++i) {
        PartStore& ps = c->pstore[i];
        if (ps.buf) continue;
        if (dev_alloc(c, (void**)&ps.buf, bytes) != DH_OK) {
            for (auto& t : c->pstore) { dev_free(c, t.buf, bytes); t.buf = nullptr; }
            c->pstore.clear();
            set_error("");
            return false;
        }
        for (int k = 0; k < 6; ++k) ps.p[k] = ps.buf + (size_t)k * c->np;
    }
    return true;
}

static void free_snaps(dh_ctx* c, std::vector<Snapshot>& v) {
    for (auto& s : v) dev_free(c, s.buf, state_floats(c) * sizeof(float));
    v.clear();
}

// S1 + S2: delta_tot and g' from the state's gas density and particle positions.
static int compute_gravity(dh_ctx* c, float* const* gas, float* const part[6], float A, float* const gp[3],
                           bool delta_primed = false) {
    DH_TRY(launch_deposit(c, gas[0], part[0], part[1], part[2], c->delta, delta_primed));
    DH_TRY(poisson_forward(c, c->delta, A, gp));
    return DH_OK;
}

// The forward step from (gas, part) to (gas_out, part_out); out may alias in (in-place update: the sweeps go
// gas -> A -> B -> gas_out, every field read and written once per sweep, no copy).  With a tape, g' and the two
// intermediate gas states A, B are written into it (and survive the step); otherwise they live in the context's
// scratch.  gp_keep: where g' of this step goes (the run's per-step g' store); gp_ready: it already holds g' of this
// step, so deposit and Poisson solve are skipped.  part_out == nullptr skips the particle update, last_sweep == false stops after sweep 2 (the reverse pass
// needs nothing more of a segment's last step).
static int step_arrays(dh_ctx* c, float* const* gas, float* const part[6], float* const* gas_out,
                       float* const part_out[6], const StepScalars& s, int64_t step, float* cmax3, StepTape* tape,
                       bool last_sweep, float* const* gp_keep = nullptr, bool gp_ready = false,
                       bool delta_primed = false, bool prime_next = false) {
    // delta_primed: c->delta already holds [gas] rho - rho_bar of this state (the previous step's last sweep wrote it);
    // prime_next: this step's last sweep writes it for the next step (dh_run's loop only: nobody can touch the state
    // in between), which takes the source-init pass (8 B/cell) off every step but a run's first.
    const bool grav = c->opt.gravity_on != 0;
    float* const* gp = gp_keep ? gp_keep : (tape ? tape->gp : c->gp);
    if (grav && !gp_ready) DH_TRY(compute_gravity(c, gas, part, (float)s.A, gp, delta_primed));
    // S3 beside S4: fork the particle update onto the side stream (not while per-kernel events are being recorded)
    const bool particles = c->np > 0 && part_out;
    const bool beside = particles && c->opt.hydro_on && c->tune_overlap && c->side && !c->prof_on;
    if (beside) {
        DH_CUDA(cudaEventRecord(c->ev_fork, c->stream));
        DH_CUDA(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
        cudaStream_t main_stream = c->stream;
        c->stream = c->side;
        const int rc = launch_kick_drift(c, grav ? gp : nullptr, part, part_out, (float)s.K, (float)(s.dtau / c->dx));
        c->stream = main_stream;
        DH_TRY(rc);
        DH_CUDA(cudaEventRecord(c->ev_join, c->side));
    } else if (particles) {
        DH_TRY(launch_kick_drift(c, grav ? gp : nullptr, part, part_out, (float)s.K, (float)(s.dtau / c->dx)));
    }
    if (c->opt.hydro_on) {
        const int* order = STRANG[((step % 6) + 6) % 6];
        const float lam = (float)(s.dtau / c->dx), kap = (float)s.kappa;
        const int nc = c->nc;
        float* cur[6]; float* nxt[6];
        for (int k = 0; k < nc; ++k) cur[k] = gas[k];
        for (int sidx = 0; sidx < 3; ++sidx) {
            if (sidx == 2 && !last_sweep) break;
            const int d = order[sidx];
            for (int k = 0; k < nc; ++k)
                nxt[k] = sidx == 2 ? gas_out[k] : (tape ? tape->sw[sidx][k] : (sidx == 0 ? c->gas_tmp[k] : c->gas_tmp2[k]));
            const int rc = launch_sweep(c, d, cur, grav ? gp[d] : nullptr, lam, kap, nxt, cmax3 ? cmax3 + sidx : nullptr,
                                        (sidx == 2 && prime_next) ? c->delta : nullptr);
            if (rc != DH_OK) {                         // join the side stream before reporting: callers see one stream
                if (beside) cudaStreamWaitEvent(c->stream, c->ev_join, 0);
                return rc;
            }
            for (int k = 0; k < nc; ++k) cur[k] = nxt[k];
        }
        if (beside) DH_CUDA(cudaStreamWaitEvent(c->stream, c->ev_join, 0));
    } else if (gas_out[0] != gas[0]) {
        for (int k = 0; k < c->nc; ++k)
            DH_CUDA(cudaMemcpyAsync(gas_out[k], gas[k], c->n3 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    }
    return DH_OK;
}

// The step VJP.  tape == nullptr: g' and the inputs of sweeps 2 and 3 are recomputed from the step's input state
// into the context's scratch first; otherwise they are taken from the tape the reverse pass recorded.
static int step_vjp_arrays(dh_ctx* c, float* const* gas_in, float* const part_in[6], const StepScalars& s, int64_t step,
                           float* const* cot_gas_out, float* const cot_part_out[6], float* const* cot_gas_in,
                           float* const cot_part_in[6], StepTape* tape, float* const* gp_kept = nullptr) {
    DH_TRY(ensure_adjoint_scratch(c));
    const bool grav = c->opt.gravity_on != 0;
    const float lam = (float)(s.dtau / c->dx), kap = (float)s.kappa;
    StepTape local;
    if (!tape) {
        for (int d = 0; d < 3; ++d) local.gp[d] = c->gp[d];
        for (int i = 0; i < 2; ++i) for (int k = 0; k < c->nc; ++k) local.sw[i][k] = c->sw_in[i][k];
        DH_TRY(step_arrays(c, gas_in, part_in, gas_in, nullptr, s, step, nullptr, &local, false, gp_kept, gp_kept != nullptr));
        tape = &local;
    }
    float* const* gp = gp_kept ? gp_kept : tape->gp;
    // ---- S4 reversed
    if (c->opt.hydro_on) {
        const int* order = STRANG[((step % 6) + 6) % 6];
        const int nc = c->nc;
        float* cur[6]; float* nxt[6];
        for (int k = 0; k < nc; ++k) cur[k] = cot_gas_out[k];
        for (int sidx = 2; sidx >= 0; --sidx) {
            const int d = order[sidx];
            float* const* src = (sidx == 0) ? gas_in : tape->sw[sidx - 1];
            // the last adjoint sweep writes the caller's cot_gas_in; the others alternate between the two scratch sets
            if (sidx == 0) for (int k = 0; k < nc; ++k) nxt[k] = cot_gas_in[k];
            else if (sidx == 2) for (int k = 0; k < nc; ++k) nxt[k] = c->cot_tmp[k];
            else for (int k = 0; k < nc; ++k) nxt[k] = c->gas_tmp[k];
            DH_TRY(launch_sweep_vjp(c, d, src, grav ? gp[d] : nullptr, lam, kap, cur, nxt, grav ? c->gpb[d] : nullptr,
                                    c->scal_dev));
            for (int k = 0; k < nc; ++k) cur[k] = nxt[k];
        }
    } else {
        for (int k = 0; k < c->nc; ++k)
            if (cot_gas_in[k] != cot_gas_out[k])
                DH_CUDA(cudaMemcpyAsync(cot_gas_in[k], cot_gas_out[k], c->n3 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
        if (grav) for (int d = 0; d < 3; ++d) DH_TRY(launch_fill(c, c->gpb[d], c->n3, 0.f));
    }
    // ---- S3 reversed (vector deposit adds to the g'_bar the sweeps wrote)
    if (c->np > 0) {
        DH_TRY(launch_kick_drift_vjp(c, grav ? const_cast<float* const*>(gp) : nullptr, part_in, cot_part_out, cot_part_in,
                                     c->gpb, (float)s.K, (float)(s.dtau / c->dx), c->scal_dev));
    }
    // ---- S2, S1 reversed
    if (grav) {
        if (c->opt.want_dA) DH_TRY(launch_dot3(c, c->gpb, const_cast<float* const*>(gp), 1.0 / s.A, c->scal_dev + 5));
        DH_TRY(poisson_adjoint(c, c->gpb, (float)s.A, c->delta));
        DH_TRY(launch_deposit_vjp(c, c->delta, part_in, cot_gas_in[0], cot_part_in));
    }
    return DH_OK;
}

// fold the device scalar accumulators into dparams: scal = (lam_b, kap_b, gamma_b, K_b, (dtau/dx)_b, A_b)
static int harvest_scalars(dh_ctx* c, dh_dparams* dp) {
    double h[8];
    DH_CUDA(cudaMemcpyAsync(h, c->scal_dev, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    if (dp) {
        dp->dgamma += h[2];
        if (c->opt.want_dsched || !c->opt.hydro_on) {
            dp->dDtau += (h[0] + h[4]) / c->dx;
            dp->dkappa += h[1];
        } else {                                   // not computed by the sweep adjoints (dh_options.want_dsched = 0): say so
            dp->dDtau = nan("");
            dp->dkappa = nan("");
        }
        dp->dK += h[3];
        dp->dA += h[5];
    }
    DH_CUDA(cudaMemsetAsync(c->scal_dev, 0, 8 * sizeof(double), c->stream));
    return DH_OK;
}

// cuFFT R2C / C2R plans sharing one work area, on the context's stream; made on first need.
static int ensure_cufft_plans(dh_ctx* c) {
    if (c->plans) return DH_OK;
    const int n = c->N;
    size_t w1 = 0, w2 = 0;
    if (cufftCreate(&c->plan_r2c) != CUFFT_SUCCESS) { set_error("cufftCreate failed"); return DH_ERR_CUFFT; }
    if (cufftCreate(&c->plan_c2r) != CUFFT_SUCCESS) {
        cufftDestroy(c->plan_r2c);
        set_error("cufftCreate failed"); return DH_ERR_CUFFT;
    }
    c->plans = true;
    cufftSetAutoAllocation(c->plan_r2c, 0);
    cufftSetAutoAllocation(c->plan_c2r, 0);
    if (cufftMakePlan3d(c->plan_r2c, n, n, n, CUFFT_R2C, &w1) != CUFFT_SUCCESS ||
        cufftMakePlan3d(c->plan_c2r, n, n, n, CUFFT_C2R, &w2) != CUFFT_SUCCESS) {
        set_error("cufftMakePlan3d(%d^3) failed", n); return DH_ERR_CUFFT;
    }
    c->fft_work_bytes = w1 > w2 ? w1 : w2;
    if (c->fft_work_bytes > 0) {
        DH_TRY(dev_alloc(c, &c->fft_work, c->fft_work_bytes));
        cufftSetWorkArea(c->plan_r2c, c->fft_work);
        cufftSetWorkArea(c->plan_c2r, c->fft_work);
    }
    if (cufftSetStream(c->plan_r2c, c->stream) != CUFFT_SUCCESS || cufftSetStream(c->plan_c2r, c->stream) != CUFFT_SUCCESS) {
        set_error("cufftSetStream failed"); return DH_ERR_CUFFT;
    }
    return DH_OK;
}

static int check_state(const dh_ctx* c, const float* const gas[5], const float* const part[6], const float* eint) {
    for (int k = 0; k < 5; ++k) if (!gas[k]) { set_error("null gas pointer %d", k); return DH_ERR_INVALID; }
    if (c->nc == 6 && !eint) { set_error("dual_energy = 1 needs the eint pointer of the state / cotangent"); return DH_ERR_INVALID; }
    if (c->np > 0) for (int k = 0; k < 6; ++k) if (!part[k]) { set_error("null particle pointer %d", k); return DH_ERR_INVALID; }
    return DH_OK;
}

}  // namespace dh

using namespace dh;

extern "C" {

const char* dh_last_error(void) { return g_err; }

int dh_init(dh_ctx** out, int grid_n, double box, double gamma, const dh_cosmology* cosmo, const dh_options* opt) {
    if (!out || !cosmo || !opt) { set_error("dh_init: null argument"); return DH_ERR_INVALID; }
    *out = nullptr;
    if (grid_n < 32 || grid_n > 1024 || grid_n % 32 != 0) {
        set_error("dh_init: grid_n must be a multiple of 32 in [32, 1024], got %d", grid_n);
        return DH_ERR_INVALID;
    }
    if (opt->dual_energy && !(opt->dual_eta >= 0.0)) {
        set_error("dh_init: dual_energy needs dual_eta >= 0 (customary 1e-3)");
        return DH_ERR_INVALID;
    }
    if (!(box > 0) || !(gamma > 1.0) || !(opt->e_floor > 0) || opt->n_part_side < 0) {
        set_error("dh_init: need box > 0, gamma > 1, e_floor > 0, n_part_side >= 0");
        return DH_ERR_INVALID;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        set_error("dh_init: no CUDA device (this library has no CPU fallback)");
        return DH_ERR_NO_DEVICE;
    }
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceProp prop;
    DH_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) {
        set_error("dh_init: device %s is sm_%d%d; this library is built for sm_100a only", prop.name, prop.major, prop.minor);
        return DH_ERR_NO_DEVICE;
    }
    dh_ctx* c = new (std::nothrow) dh_ctx();
    if (!c) return DH_ERR_OOM;
    c->N = grid_n;
    c->n3 = (int64_t)grid_n * grid_n * grid_n;
    c->nps = opt->n_part_side;
    c->np = (int64_t)c->nps * c->nps * c->nps;
    c->box = box; c->gamma = gamma; c->dx = box / grid_n;
    c->cosmo = *cosmo; c->opt = *opt;
    c->nc = opt->dual_energy ? 6 : 5;
    c->f_b = cosmo->Omega_m > 0 ? cosmo->Omega_b / cosmo->Omega_m : 0.0;
    c->m_p = c->np > 0 ? (1.0 - c->f_b) * (double)c->n3 / (double)c->np : 0.0;
    c->rho_bar = (c->np > 0 ? 1.0 - c->f_b : 0.0) + (opt->gas_sources_gravity ? c->f_b : 0.0);
    c->sm_count = prop.multiProcessorCount;
    // NULL = the legacy default stream, which orders with the caller's default-stream work (torch's current stream is
    // stream 0 unless the caller changed it); a private non-blocking stream would race with it.
    c->stream = (cudaStream_t)opt->cuda_stream;
    int rc = DH_OK;
    auto fail = [&](int code) { dh_free(c); return code; };
    if (opt->gravity_on) {
        const size_t nspec = (size_t)grid_n * grid_n * (grid_n / 2 + 1);
        if ((rc = dev_alloc(c, (void**)&c->delta, c->n3 * sizeof(float))) != DH_OK) return fail(rc);
        for (int i = 0; i < 4; ++i)
            if ((rc = dev_alloc(c, (void**)&c->spec[i], nspec * sizeof(float2))) != DH_OK) return fail(rc);
        if ((rc = alloc_fields(c, c->gp, 3, c->n3)) != DH_OK) return fail(rc);
        // cuFFT plans (transforms only) are needed by the route for sides that are not a power of two; a power-of-two side
        // makes them only when dh_tune("own_fft", 0) asks for that route (at 512^3 their work area is ~0.5 GB)
        if (!own_fft_supported(grid_n) && (rc = ensure_cufft_plans(c)) != DH_OK) return fail(rc);
        if (own_fft_supported(grid_n)) {
            if ((rc = own_fft_init(c)) != DH_OK) return fail(rc);
            c->own_fft = true;
        }
    }
    if (opt->hydro_on && (rc = alloc_fields(c, c->gas_tmp, c->nc, c->n3)) != DH_OK) return fail(rc);
    if (opt->hydro_on && (rc = alloc_fields(c, c->gas_tmp2, c->nc, c->n3)) != DH_OK) return fail(rc);
    if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        set_error("dh_init: side stream / events: %s", cudaGetErrorString(cudaGetLastError()));
        return fail(DH_ERR_CUDA);
    }
    if ((rc = dev_alloc(c, (void**)&c->cmax_step, 3 * sizeof(float))) != DH_OK) return fail(rc);
    if ((rc = dev_alloc(c, (void**)&c->scal_dev, 8 * sizeof(double))) != DH_OK) return fail(rc);
    if (cudaMemsetAsync(c->scal_dev, 0, 8 * sizeof(double), c->stream) != cudaSuccess) return fail(DH_ERR_CUDA);
    *out = c;
    return DH_OK;
}

int dh_free(dh_ctx* c) {
    if (!c) return DH_OK;
    if (c->stream) cudaStreamSynchronize(c->stream);
    if (c->plans) { cufftDestroy(c->plan_r2c); cufftDestroy(c->plan_c2r); }
    cudaFree(c->fft_work);
    cudaFree(c->fft_tw);
    cudaFree(c->delta);
    for (auto p : c->spec) cudaFree(p);
    for (auto p : c->gp) cudaFree(p);
    for (auto p : c->gas_tmp) cudaFree(p);
    for (auto p : c->gas_tmp2) cudaFree(p);
    for (int i = 0; i < 2; ++i) for (auto p : c->sw_in[i]) cudaFree(p);
    for (auto p : c->gpb) cudaFree(p);
    for (auto p : c->cot_tmp) cudaFree(p);
    for (auto p : c->part_tmp) cudaFree(p);
    cudaFree(c->cmax_step); cudaFree(c->cmax_log); cudaFree(c->scal_dev); cudaFree(c->ps_bins); cudaFree(c->sg_scal); cudaFree(c->scal_log);
    cudaFree(c->hv_state); cudaFree(c->hv_cot); cudaFree(c->hv_mesh);
    for (auto& s : c->snaps) cudaFree(s.buf);
    for (auto& s : c->seg) cudaFree(s.buf);
    for (auto& t : c->tapes) cudaFree(t.buf);
    for (auto& t : c->gstore) cudaFree(t.buf);
    for (auto& t : c->pstore) cudaFree(t.buf);
    for (auto e : c->prof_ev) cudaEventDestroy(e);
    if (c->side) { cudaStreamSynchronize(c->side); cudaStreamDestroy(c->side); }
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->own_stream) cudaStreamDestroy(c->stream);
    cudaGetLastError();
    delete c;
    return DH_OK;
}

int dh_sync(dh_ctx* c) {
    if (!c) return DH_ERR_INVALID;
    DH_CUDA(cudaStreamSynchronize(c->stream));
    return DH_OK;
}

static const char* const PROF_NAMES[PROF_N] = {
    "source_init", "deposit", "fft_r2c", "green", "fft_c2r", "kick_drift", "sweep_x", "sweep_y", "sweep_z",
    "sweep_x_adj", "sweep_y_adj", "sweep_z_adj", "kick_drift_adj", "green_adj", "deposit_adj", "axpy", "dot3", "fill",
    "copy", "fft_x1", "fft_x3", "fft_y1", "fft_y3"};

int dh_profile_enable(dh_ctx* c, int on) {
    if (!c) return DH_ERR_INVALID;
    DH_CUDA(cudaStreamSynchronize(c->stream));
    c->prof_on = on != 0;
    c->prof_used = 0;
    return DH_OK;
}
int dh_profile_categories(void) { return PROF_N; }
const char* dh_profile_name(int i) { return (i >= 0 && i < PROF_N) ? PROF_NAMES[i] : nullptr; }
int dh_profile_read(dh_ctx* c, double* ms_out, int64_t* count_out) {
    if (!c || !ms_out || !count_out) { set_error("dh_profile_read: null argument"); return DH_ERR_INVALID; }
    DH_CUDA(cudaStreamSynchronize(c->stream));
    for (int i = 0; i < PROF_N; ++i) { ms_out[i] = 0.0; count_out[i] = 0; }
    for (size_t s = 0; s < c->prof_used; ++s) {
        float ms = 0.f;
        DH_CUDA(cudaEventElapsedTime(&ms, c->prof_ev[2 * s], c->prof_ev[2 * s + 1]));
        ms_out[c->prof_cat[s]] += ms;
        count_out[c->prof_cat[s]] += 1;
    }
    c->prof_used = 0;
    return DH_OK;
}

int dh_tune(dh_ctx* c, const char* key, int value) {
    if (!c || !key) { set_error("dh_tune: null argument"); return DH_ERR_INVALID; }
    if (!strcmp(key, "march_s_fwd")) c->tune_march_s_fwd = value;
    else if (!strcmp(key, "march_s_adj")) c->tune_march_s_adj = value;
    else if (!strcmp(key, "tape")) c->tune_tape = value;
    else if (!strcmp(key, "gstore")) c->tune_gstore = value;
    else if (!strcmp(key, "pstore")) c->tune_pstore = value;
    else if (!strcmp(key, "own_fft")) {
        if (!value && c->opt.gravity_on) DH_TRY(ensure_cufft_plans(c));
        c->tune_own_fft = value;
    }
    else if (!strcmp(key, "overlap")) c->tune_overlap = value;
    else if (!strcmp(key, "prime")) c->tune_prime = value;
    else if (!strcmp(key, "deposit_tile")) c->tune_deposit_tile = value;
    else if (!strcmp(key, "de_march")) c->tune_de_march = value;
    else { set_error("dh_tune: unknown key %s", key); return DH_ERR_INVALID; }
    return DH_OK;
}

int dh_conserved_sums(dh_ctx* c, const dh_state* st, double* out) {
    if (!c || !st || !out) { set_error("dh_conserved_sums: null argument"); return DH_ERR_INVALID; }
    DH_TRY(check_state(c, st->gas, st->part, st->eint));
    double* acc = nullptr;
    DH_TRY(dev_alloc(c, (void**)&acc, 8 * sizeof(double)));
    int rc = DH_OK;
    if (cudaMemsetAsync(acc, 0, 8 * sizeof(double), c->stream) != cudaSuccess) rc = DH_ERR_CUDA;
    const float* g[5] = {st->gas[0], st->gas[1], st->gas[2], st->gas[3], st->gas[4]};
    if (rc == DH_OK) rc = launch_sum_arrays(c, g, 5, c->n3, acc);
    if (rc == DH_OK && c->np > 0) {
        const float* w[3] = {st->part[3], st->part[4], st->part[5]};
        rc = launch_sum_arrays(c, w, 3, c->np, acc + 5);
    }
    if (rc == DH_OK && (cudaMemcpyAsync(out, acc, 8 * sizeof(double), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
                        cudaStreamSynchronize(c->stream) != cudaSuccess)) rc = DH_ERR_CUDA;
    dev_free(c, acc, 8 * sizeof(double));
    if (rc != DH_OK) { if (rc == DH_ERR_CUDA) set_error("dh_conserved_sums: CUDA error"); return rc; }
    for (int d = 0; d < 3; ++d) out[5 + d] *= c->m_p;
    return DH_OK;
}

int dh_debug_poison(dh_ctx* c, int level) {
    if (!c) { set_error("dh_debug_poison: null context"); return DH_ERR_INVALID; }
    const size_t mesh = (size_t)c->n3 * sizeof(float);
    const size_t nspec = (size_t)c->N * c->N * (c->N / 2 + 1) * sizeof(float2);
    auto fill = [&](void* p, size_t bytes) -> int {
        if (p && bytes) DH_CUDA(cudaMemsetAsync(p, 0xff, bytes, c->stream));
        return DH_OK;
    };
    DH_TRY(fill(c->delta, mesh));
    for (auto p : c->spec) DH_TRY(fill(p, nspec));
    for (auto p : c->gp) DH_TRY(fill(p, mesh));
    for (auto p : c->gas_tmp) DH_TRY(fill(p, mesh));
    for (auto p : c->gas_tmp2) DH_TRY(fill(p, mesh));
    for (int i = 0; i < 2; ++i) for (auto p : c->sw_in[i]) DH_TRY(fill(p, mesh));
    for (auto p : c->gpb) DH_TRY(fill(p, mesh));
    for (auto p : c->cot_tmp) DH_TRY(fill(p, mesh));
    const size_t state_bytes = state_floats(c) * sizeof(float);
    for (size_t i = 1; i < c->seg.size(); ++i) DH_TRY(fill(c->seg[i].buf, state_bytes));
    for (auto& t : c->tapes) DH_TRY(fill(t.buf, (size_t)(3 + 2 * c->nc) * mesh));
    if (level >= 1) {
        for (auto& s : c->snaps) DH_TRY(fill(s.buf, state_bytes));
        for (auto& g : c->gstore) DH_TRY(fill(g.buf, 3 * mesh));
        for (auto& t : c->pstore) DH_TRY(fill(t.buf, (size_t)6 * c->np * sizeof(float)));
        DH_TRY(fill(c->cmax_log, (size_t)3 * c->cmax_cap * sizeof(float)));
        c->run_valid = false;
    }
    return DH_OK;
}

int64_t dh_device_bytes(dh_ctx* c) { return c ? c->bytes : 0; }
int64_t dh_launch_count(dh_ctx* c) { return c ? c->launches : 0; }

int dh_step_scalars(const dh_cosmology* cosmo, double a_i, double a_next, double dt, double dt_prev, double* out) {
    if (!cosmo || !out) return DH_ERR_INVALID;
    StepScalars s = step_scalars(*cosmo, a_i, a_next, dt, dt_prev);
    out[0] = s.dtau; out[1] = s.kappa; out[2] = s.K; out[3] = s.A;
    return DH_OK;
}

int dh_schedule_lna(const dh_cosmology* co, double a0, double a1, int n, double* a_out, double* dt_out) {
    if (!co || !a_out || !dt_out || n <= 0 || !(a0 > 0) || !(a1 > a0)) { set_error("dh_schedule_lna: bad argument"); return DH_ERR_INVALID; }
    const double r = std::log(a1 / a0) / n;
    for (int k = 0; k <= n; ++k) a_out[k] = a0 * std::exp(k * r);
    a_out[n] = a1;
    const bool eds = co->Omega_L == 0.0 && std::fabs(co->Omega_m - 1.0) < 1e-15;
    for (int k = 0; k < n; ++k) {
        const double lo = a_out[k], hi = a_out[k + 1];
        if (eds) {
            // t = 2 / (3 H0) a^{3/2}
            dt_out[k] = (2.0 / (3.0 * co->H0)) * (hi * std::sqrt(hi) - lo * std::sqrt(lo));
        } else {
            // dt = d ln a / H(a): composite Simpson in ln a
            const int M = 2048;
            const double h = std::log(hi / lo) / M, Ok = 1.0 - co->Omega_m - co->Omega_L;
            double acc = 0.0;
            for (int j = 0; j <= M; ++j) {
                const double a = lo * std::exp(j * h);
                const double H = co->H0 * std::sqrt(co->Omega_m / (a * a * a) + Ok / (a * a) + co->Omega_L);
                acc += ((j == 0 || j == M) ? 1.0 : ((j & 1) ? 4.0 : 2.0)) / H;
            }
            dt_out[k] = acc * h / 3.0;
        }
    }
    return DH_OK;
}

int dh_step(dh_ctx* c, dh_state* st, double dt, double a, float* cfl_cmax_out) {
    if (!c || !st) { set_error("dh_step: null argument"); return DH_ERR_INVALID; }
    DH_TRY(check_state(c, st->gas, st->part, st->eint));
    const StepScalars s = step_scalars(c->cosmo, st->a, a, dt, st->dt_prev);
    float* cm = cfl_cmax_out ? cfl_cmax_out : c->cmax_step;
    DH_CUDA(cudaMemsetAsync(cm, 0, 3 * sizeof(float), c->stream));
    const G6 g(*st);
    DH_TRY(step_arrays(c, g.p, st->part, g.p, st->part, s, st->step, cm, nullptr, true));
    st->a = c->cosmo.static_mode ? 1.0 : a;
    st->dt_prev = dt;
    st->step += 1;
    return DH_OK;
}

int dh_step_vjp(dh_ctx* c, const dh_state* st, double dt, double a, const dh_cot* cot_out, dh_cot* cot_in, dh_dparams* dp) {
    if (!c || !st || !cot_out || !cot_in) { set_error("dh_step_vjp: null argument"); return DH_ERR_INVALID; }
    DH_TRY(check_state(c, st->gas, st->part, st->eint));
    DH_TRY(check_state(c, cot_out->gas, cot_out->part, cot_out->eint));
    DH_TRY(check_state(c, cot_in->gas, cot_in->part, cot_in->eint));
    const StepScalars s = step_scalars(c->cosmo, st->a, a, dt, st->dt_prev);
    const G6 g(*st), co(*cot_out), ci(*cot_in);
    DH_TRY(step_vjp_arrays(c, g.p, st->part, s, st->step, co.p, cot_out->part, ci.p, cot_in->part, nullptr));
    return harvest_scalars(c, dp);
}

int dh_run(dh_ctx* c, dh_state* st, const double* a_sched, const double* dt_sched, int n_steps, int stride) {
    if (!c || !st || !a_sched || !dt_sched || n_steps < 0) { set_error("dh_run: bad argument"); return DH_ERR_INVALID; }
    DH_TRY(check_state(c, st->gas, st->part, st->eint));
    if (n_steps > c->cmax_cap) {
        dev_free(c, c->cmax_log, (size_t)3 * c->cmax_cap * sizeof(float));
        c->cmax_log = nullptr; c->cmax_cap = 0;
        DH_TRY(dev_alloc(c, (void**)&c->cmax_log, (size_t)3 * n_steps * sizeof(float)));
        c->cmax_cap = n_steps;
    }
    if (n_steps > 0) DH_CUDA(cudaMemsetAsync(c->cmax_log, 0, (size_t)3 * n_steps * sizeof(float), c->stream));
    c->cmax_n = n_steps;
    c->run_valid = false;
    const int nseg = stride > 0 ? (n_steps + stride - 1) / stride : 0;
    if ((int)c->snaps.size() < nseg) c->snaps.resize(nseg);     // the pool only grows (dh_free releases it)
    c->run_a.assign(a_sched, a_sched + n_steps);
    c->run_dt.assign(dt_sched, dt_sched + n_steps);
    c->run_n = n_steps; c->run_stride = stride;
    c->run_gstore = stride > 0 && ensure_gstore(c, n_steps);
    c->run_pstore = ensure_pstore(c, n_steps, stride);
    for (int k = 0; k < n_steps; ++k) {
        // with the particle store, step k reads the slot of step k and writes the slot of step k + 1; the first step reads
        // the caller's arrays and the last one writes them
        float* const* pin = (c->run_pstore && k > 0) ? c->pstore[k].p : st->part;
        float* const* pout = (c->run_pstore && k + 1 < n_steps) ? c->pstore[k + 1].p : st->part;
        if (stride > 0 && k % stride == 0) DH_TRY(snapshot_store(c, c->snaps[k / stride], st, pin));
        const StepScalars s = step_scalars(c->cosmo, st->a, a_sched[k], dt_sched[k], st->dt_prev);
        const bool can_prime = c->opt.gravity_on && c->opt.hydro_on && c->tune_prime && c->nc == 5;
        const G6 g(*st);
        DH_TRY(step_arrays(c, g.p, pin, g.p, pout, s, st->step, c->cmax_log + 3 * k, nullptr, true,
                           c->run_gstore ? c->gstore[k].gp : nullptr, false, can_prime && k > 0,
                           can_prime && k + 1 < n_steps));
        st->a = c->cosmo.static_mode ? 1.0 : a_sched[k];
        st->dt_prev = dt_sched[k];
        st->step += 1;
    }
    // one synchronisation per run: fetch the CFL log and look for NaN/Inf
    if (n_steps > 0) {
        std::vector<float> h((size_t)3 * n_steps);
        DH_CUDA(cudaMemcpyAsync(h.data(), c->cmax_log, h.size() * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
        DH_CUDA(cudaStreamSynchronize(c->stream));
        for (size_t i = 0; i < h.size(); ++i)
            if (!std::isfinite(h[i])) {
                set_error("dh_run: non-finite CFL maximum at step %zu, sweep %zu", i / 3, i % 3);
                return DH_ERR_NONFINITE;
            }
    }
    c->run_valid = stride > 0;
    return DH_OK;
}

int dh_reserve(dh_ctx* c, int n_steps, int stride) {
    if (!c || n_steps < 0) { set_error("dh_reserve: bad argument"); return DH_ERR_INVALID; }
    if (n_steps > c->cmax_cap) {
        dev_free(c, c->cmax_log, (size_t)3 * c->cmax_cap * sizeof(float));
        c->cmax_log = nullptr; c->cmax_cap = 0;
        DH_TRY(dev_alloc(c, (void**)&c->cmax_log, (size_t)3 * n_steps * sizeof(float)));
        c->cmax_cap = n_steps;
    }
    if (stride <= 0) return DH_OK;
    const size_t bytes = state_floats(c) * sizeof(float);
    const int nseg = (n_steps + stride - 1) / stride;
    if ((int)c->snaps.size() < nseg) c->snaps.resize(nseg);
    for (int i = 0; i < nseg; ++i)
        if (!c->snaps[i].buf) DH_TRY(dev_alloc(c, (void**)&c->snaps[i].buf, bytes));
    const int in_seg = stride < n_steps ? stride : n_steps;
    if ((int)c->seg.size() < in_seg) c->seg.resize(in_seg);
    for (int i = 1; i < in_seg; ++i)
        if (!c->seg[i].buf) DH_TRY(dev_alloc(c, (void**)&c->seg[i].buf, bytes));
    DH_TRY(ensure_adjoint_scratch(c));
    ensure_tapes(c, in_seg);
    ensure_gstore(c, n_steps);
    ensure_pstore(c, n_steps, stride);
    c->run_valid = false;
    return DH_OK;
}

int dh_get_cmax(dh_ctx* c, float* out, int n) {
    if (!c || !out || n < 0 || n > c->cmax_n) { set_error("dh_get_cmax: bad argument"); return DH_ERR_INVALID; }
    if (n == 0) return DH_OK;
    DH_CUDA(cudaMemcpyAsync(out, c->cmax_log, (size_t)3 * n * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    return DH_OK;
}

int dh_run_vjp(dh_ctx* c, const dh_cot* cot_final, dh_cot* cot_initial, dh_dparams* dp) {
    if (!c || !cot_final || !cot_initial) { set_error("dh_run_vjp: null argument"); return DH_ERR_INVALID; }
    if (!c->run_valid) { set_error("dh_run_vjp: no checkpointed dh_run to differentiate"); return DH_ERR_STATE; }
    DH_TRY(check_state(c, cot_final->gas, cot_final->part, cot_final->eint));
    DH_TRY(check_state(c, cot_initial->gas, cot_initial->part, cot_initial->eint));
    const int n = c->run_n, stride = c->run_stride;
    const int nseg = (n + stride - 1) / stride;
    // cot_initial doubles as the running cotangent
    const G6 cf(*cot_final), cini(*cot_initial);
    for (int k = 0; k < c->nc; ++k)
        if (cini.p[k] != cf.p[k])
            DH_CUDA(cudaMemcpyAsync(cini.p[k], cf.p[k], c->n3 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    for (int k = 0; k < 6 && c->np > 0; ++k)
        if (cot_initial->part[k] != cot_final->part[k])
            DH_CUDA(cudaMemcpyAsync(cot_initial->part[k], cot_final->part[k], c->np * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    if ((int)c->seg.size() < stride) c->seg.resize(stride);
    const int in_seg = stride < n ? stride : n;
    const bool taped = ensure_tapes(c, in_seg);
    // per-step scalar cotangents (needed to chain to cosmological parameters: every step has its own d(scalars)/d(theta))
    const bool per_step = c->opt.want_dsched != 0;
    if (per_step && c->scal_log_cap < n) {
        if (c->scal_log) dev_free(c, c->scal_log, (size_t)c->scal_log_cap * 8 * sizeof(double));
        c->scal_log = nullptr; c->scal_log_cap = 0;
        DH_TRY(dev_alloc(c, (void**)&c->scal_log, (size_t)n * 8 * sizeof(double)));
        c->scal_log_cap = n;
    }
    c->step_dp.clear();
    for (int sgi = nseg - 1; sgi >= 0; --sgi) {
        const int k0 = sgi * stride, k1 = (k0 + stride < n) ? k0 + stride : n;
        // ---- re-run the segment from its snapshot: step k goes from seg[k - k0] (seg[0] is the snapshot itself) to
        // seg[k - k0 + 1] out of place, so every step's input survives; with tapes each step also leaves its g' and
        // sweep inputs behind, and the segment's last step runs only that far
        for (int k = k0; k < k1; ++k) {
            const bool last = (k == k1 - 1);
            if (last && !taped) break;
            dh_state in;
            snapshot_view(c, k == k0 ? c->snaps[sgi] : c->seg[k - k0], &in);
            const StepScalars s = step_scalars(c->cosmo, in.a, c->run_a[k], c->run_dt[k], in.dt_prev);
            StepTape* tape = taped ? &c->tapes[k - k0] : nullptr;
            float* const* gk = c->run_gstore ? c->gstore[k].gp : nullptr;
            const G6 gin(in);
            // the particles entering step k: kept by dh_run (then the re-run has no particle update to repeat), else the
            // in-segment state's own
            float* const* pin = (c->run_pstore && k > k0) ? c->pstore[k].p : in.part;
            if (last) {
                DH_TRY(step_arrays(c, gin.p, pin, gin.p, nullptr, s, in.step, nullptr, tape, false, gk, gk != nullptr));
            } else {
                Snapshot& nx = c->seg[k - k0 + 1];
                if (!nx.buf) DH_TRY(dev_alloc(c, (void**)&nx.buf, state_floats(c) * sizeof(float)));
                dh_state out;
                snapshot_view(c, nx, &out);
                const G6 gout(out);
                DH_TRY(step_arrays(c, gin.p, pin, gout.p, c->run_pstore ? nullptr : out.part, s, in.step, nullptr, tape, true, gk,
                                   gk != nullptr));
                nx.a = c->cosmo.static_mode ? 1.0 : c->run_a[k];
                nx.dt_prev = c->run_dt[k];
                nx.step = in.step + 1;
            }
        }
        // ---- step VJPs, last step of the segment first
        for (int k = k1 - 1; k >= k0; --k) {
            dh_state in;
            snapshot_view(c, k == k0 ? c->snaps[sgi] : c->seg[k - k0], &in);
            const StepScalars s = step_scalars(c->cosmo, in.a, c->run_a[k], c->run_dt[k], in.dt_prev);
            const G6 gin(in);
            float* const* pin = (c->run_pstore && k > k0) ? c->pstore[k].p : in.part;
            DH_TRY(step_vjp_arrays(c, gin.p, pin, s, in.step, cini.p, cot_initial->part, cini.p,
                                   cot_initial->part, taped ? &c->tapes[k - k0] : nullptr,
                                   c->run_gstore ? c->gstore[k].gp : nullptr));
            if (per_step) {
                DH_CUDA(cudaMemcpyAsync(c->scal_log + (size_t)8 * k, c->scal_dev, 8 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
                DH_CUDA(cudaMemsetAsync(c->scal_dev, 0, 8 * sizeof(double), c->stream));
            }
        }
    }
    if (!per_step) return harvest_scalars(c, dp);
    std::vector<double> h((size_t)8 * n);
    DH_CUDA(cudaMemcpyAsync(h.data(), c->scal_log, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    c->step_dp.resize((size_t)5 * n);
    for (int k = 0; k < n; ++k) {
        const double* q = &h[(size_t)8 * k];
        double* o = &c->step_dp[(size_t)5 * k];
        o[0] = q[2]; o[1] = (q[0] + q[4]) / c->dx; o[2] = q[1]; o[3] = q[3]; o[4] = q[5];
        if (dp) { dp->dgamma += o[0]; dp->dDtau += o[1]; dp->dkappa += o[2]; dp->dK += o[3]; dp->dA += o[4]; }
    }
    return DH_OK;
}

int dh_get_step_dparams(dh_ctx* c, double* out, int n_steps) {
    if (!c || !out || n_steps <= 0) { set_error("dh_get_step_dparams: bad argument"); return DH_ERR_INVALID; }
    if ((int)c->step_dp.size() < 5 * n_steps) {
        set_error("dh_get_step_dparams: the last dh_run_vjp kept %d steps (needs dh_options.want_dsched = 1)", (int)c->step_dp.size() / 5);
        return DH_ERR_STATE;
    }
    for (int i = 0; i < 5 * n_steps; ++i) out[i] = c->step_dp[i];
    return DH_OK;
}

// dL/dOmega_m and dL/dH0 through the step scalars of an ln-a schedule (initial state held fixed): central differences, in
// fp64 on the host, of the closed-form host functions dh_schedule_lna and step_scalars -- no device work.
int dh_chain_cosmology(const dh_cosmology* co, double a0, double a1, int n, const double* step_dparams, double* dOmega_m,
                       double* dH0) {
    if (!co || !step_dparams || n <= 0 || co->static_mode) { set_error("dh_chain_cosmology: bad argument"); return DH_ERR_INVALID; }
    auto scalars = [&](const dh_cosmology& q, std::vector<StepScalars>& out) -> int {
        std::vector<double> a(n + 1), dt(n);
        DH_TRY(dh_schedule_lna(&q, a0, a1, n, a.data(), dt.data()));
        out.resize(n);
        for (int k = 0; k < n; ++k) out[k] = step_scalars(q, a[k], a[k + 1], dt[k], k == 0 ? 0.0 : dt[k - 1]);
        return DH_OK;
    };
    double* outs[2] = {dOmega_m, dH0};
    for (int which = 0; which < 2; ++which) {
        if (!outs[which]) continue;
        dh_cosmology p = *co, m = *co;
        const double h = which == 0 ? 1e-5 : 1e-5 * co->H0;
        if (which == 0) { p.Omega_m += h; m.Omega_m -= h; } else { p.H0 += h; m.H0 -= h; }
        std::vector<StepScalars> sp, sm;
        DH_TRY(scalars(p, sp)); DH_TRY(scalars(m, sm));
        double acc = 0.0;
        for (int k = 0; k < n; ++k) {
            const double* d = step_dparams + (size_t)5 * k;        // (dgamma, dDtau, dkappa, dK, dA)
            acc += (d[1] * (sp[k].dtau - sm[k].dtau) + d[2] * (sp[k].kappa - sm[k].kappa) + d[3] * (sp[k].K - sm[k].K) +
                    d[4] * (sp[k].A - sm[k].A)) / (2.0 * h);
        }
        *outs[which] = acc;
    }
    return DH_OK;
}

// ---------------------------------------------------------------------------------------------- host variants ----
static int hv_ensure(dh_ctx* c, float** buf) {
    if (!*buf) DH_TRY(dev_alloc(c, (void**)buf, state_floats(c) * sizeof(float)));
    return DH_OK;
}

int dh_run_host(dh_ctx* c, float* gas_host, float* part_host, double* a, double* dt_prev, int64_t* step,
                const double* a_sched, const double* dt_sched, int n_steps, int stride) {
    if (!c || !gas_host || !a || !dt_prev || !step || (c->np > 0 && !part_host)) { set_error("dh_run_host: null argument"); return DH_ERR_INVALID; }
    DH_TRY(hv_ensure(c, &c->hv_state));
    dh_state st;
    for (int k = 0; k < 5; ++k) st.gas[k] = c->hv_state + (size_t)k * c->n3;
    st.eint = c->nc == 6 ? c->hv_state + (size_t)5 * c->n3 : nullptr;
    for (int k = 0; k < 6; ++k) st.part[k] = c->hv_state + (size_t)c->nc * c->n3 + (size_t)k * c->np;
    st.a = *a; st.dt_prev = *dt_prev; st.step = *step;
    DH_CUDA(cudaMemcpyAsync(st.gas[0], gas_host, (size_t)c->nc * c->n3 * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    if (c->np > 0) DH_CUDA(cudaMemcpyAsync(st.part[0], part_host, (size_t)6 * c->np * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    DH_TRY(dh_run(c, &st, a_sched, dt_sched, n_steps, stride));
    DH_CUDA(cudaMemcpyAsync(gas_host, st.gas[0], (size_t)c->nc * c->n3 * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    if (c->np > 0) DH_CUDA(cudaMemcpyAsync(part_host, st.part[0], (size_t)6 * c->np * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    *a = st.a; *dt_prev = st.dt_prev; *step = st.step;
    return DH_OK;
}

int dh_run_vjp_host(dh_ctx* c, float* cot_gas_host, float* cot_part_host, dh_dparams* dp) {
    if (!c || !cot_gas_host || (c->np > 0 && !cot_part_host)) { set_error("dh_run_vjp_host: null argument"); return DH_ERR_INVALID; }
    DH_TRY(hv_ensure(c, &c->hv_cot));
    dh_cot ct;
    for (int k = 0; k < 5; ++k) ct.gas[k] = c->hv_cot + (size_t)k * c->n3;
    ct.eint = c->nc == 6 ? c->hv_cot + (size_t)5 * c->n3 : nullptr;
    for (int k = 0; k < 6; ++k) ct.part[k] = c->hv_cot + (size_t)c->nc * c->n3 + (size_t)k * c->np;
    DH_CUDA(cudaMemcpyAsync(ct.gas[0], cot_gas_host, (size_t)c->nc * c->n3 * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    if (c->np > 0) DH_CUDA(cudaMemcpyAsync(ct.part[0], cot_part_host, (size_t)6 * c->np * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    DH_TRY(dh_run_vjp(c, &ct, &ct, dp));
    DH_CUDA(cudaMemcpyAsync(cot_gas_host, ct.gas[0], (size_t)c->nc * c->n3 * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    if (c->np > 0) DH_CUDA(cudaMemcpyAsync(cot_part_host, ct.part[0], (size_t)6 * c->np * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    return DH_OK;
}

// The whole chain of field-level inference with host buffers: delta_init -> state -> n steps -> data term, and back.
int dh_value_and_grad_host(dh_ctx* c, const float* delta_init_host, const float* data_host, const float* noise_var_host,
                           int observable, double scale, double weight, double a0, double vel_factor, double e_tilde0,
                           const double* a_sched, const double* dt_sched, int n_steps, int stride, float* grad_delta_host,
                           double* loss_out, dh_dparams* dp) {
    if (!c || !delta_init_host || !data_host || !a_sched || !dt_sched || !grad_delta_host || n_steps <= 0 || stride <= 0) {
        set_error("dh_value_and_grad_host: bad argument (needs n_steps > 0 and a checkpoint stride > 0)");
        return DH_ERR_INVALID;
    }
    DH_TRY(hv_ensure(c, &c->hv_state));
    DH_TRY(hv_ensure(c, &c->hv_cot));
    if (!c->hv_mesh) DH_TRY(dev_alloc(c, (void**)&c->hv_mesh, (size_t)3 * c->n3 * sizeof(float)));
    float* delta_d = c->hv_mesh;
    float* data_d = c->hv_mesh + c->n3;                    // becomes the gradient once the data term has read it
    float* noise_d = noise_var_host ? c->hv_mesh + 2 * c->n3 : nullptr;
    const size_t mesh_bytes = (size_t)c->n3 * sizeof(float);
    DH_CUDA(cudaMemcpyAsync(delta_d, delta_init_host, mesh_bytes, cudaMemcpyHostToDevice, c->stream));
    DH_CUDA(cudaMemcpyAsync(data_d, data_host, mesh_bytes, cudaMemcpyHostToDevice, c->stream));
    if (noise_d) DH_CUDA(cudaMemcpyAsync(noise_d, noise_var_host, mesh_bytes, cudaMemcpyHostToDevice, c->stream));
    dh_state st;
    dh_cot ct;
    for (int k = 0; k < 5; ++k) { st.gas[k] = c->hv_state + (size_t)k * c->n3; ct.gas[k] = c->hv_cot + (size_t)k * c->n3; }
    st.eint = c->nc == 6 ? c->hv_state + (size_t)5 * c->n3 : nullptr;
    ct.eint = c->nc == 6 ? c->hv_cot + (size_t)5 * c->n3 : nullptr;
    for (int k = 0; k < 6; ++k) {
        st.part[k] = c->hv_state + (size_t)c->nc * c->n3 + (size_t)k * c->np;
        ct.part[k] = c->hv_cot + (size_t)c->nc * c->n3 + (size_t)k * c->np;
    }
    DH_TRY(dh_ic_zeldovich(c, delta_d, a0, vel_factor, e_tilde0, &st));
    DH_TRY(dh_run(c, &st, a_sched, dt_sched, n_steps, stride));
    DH_CUDA(cudaMemsetAsync(ct.part[0], 0, (size_t)6 * c->np * sizeof(float), c->stream));   // the loss does not see particles
    if (ct.eint) DH_CUDA(cudaMemsetAsync(ct.eint, 0, (size_t)c->n3 * sizeof(float), c->stream));   // nor q
    DH_TRY(dh_data_term(c, observable, st.gas, data_d, noise_d, scale, weight, ct.gas, loss_out));
    DH_TRY(dh_run_vjp(c, &ct, &ct, dp));
    DH_TRY(dh_ic_zeldovich_vjp(c, delta_d, vel_factor, e_tilde0, &ct, data_d));
    DH_CUDA(cudaMemcpyAsync(grad_delta_host, data_d, mesh_bytes, cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    return DH_OK;
}

// ---------------------------------------------------------------------------------------------- single kernels ----
int dh_debug_cell_index(dh_ctx* c, const float* x_dev, int64_t n, int32_t* i0_dev, int32_t* i1_dev) {
    if (!c || !x_dev || !i0_dev || !i1_dev || n < 0) { set_error("dh_debug_cell_index: bad argument"); return DH_ERR_INVALID; }
    return launch_cell_index(c, x_dev, n, i0_dev, i1_dev);
}

int dh_sweep(dh_ctx* c, int d, float* const gas_in[5], const float* g, double lam, double kap, float* const gas_out[5],
             float* cmax_out) {
    if (!c || d < 0 || d > 2 || !gas_in || !gas_out) { set_error("dh_sweep: bad argument"); return DH_ERR_INVALID; }
    if (c->nc != 5) { set_error("dh_sweep: this context has dual_energy = 1, call dh_sweep_de"); return DH_ERR_INVALID; }
    return launch_sweep(c, d, gas_in, g, (float)lam, (float)kap, gas_out, cmax_out);
}

int dh_sweep_de(dh_ctx* c, int d, float* const gas_in[6], const float* g, double lam, double kap, float* const gas_out[6],
                float* cmax_out) {
    if (!c || d < 0 || d > 2 || !gas_in || !gas_out) { set_error("dh_sweep_de: bad argument"); return DH_ERR_INVALID; }
    if (c->nc != 6) { set_error("dh_sweep_de: needs a context with dual_energy = 1"); return DH_ERR_INVALID; }
    return launch_sweep(c, d, gas_in, g, (float)lam, (float)kap, gas_out, cmax_out);
}

int dh_sweep_de_vjp(dh_ctx* c, int d, float* const gas_in[6], const float* g, double lam, double kap,
                    float* const cot_out[6], float* const cot_in[6], float* g_bar, double* scal_bar) {
    if (!c || d < 0 || d > 2 || !gas_in || !cot_out || !cot_in || !scal_bar || (g && !g_bar)) {
        set_error("dh_sweep_de_vjp: bad argument"); return DH_ERR_INVALID;
    }
    if (c->nc != 6) { set_error("dh_sweep_de_vjp: needs a context with dual_energy = 1"); return DH_ERR_INVALID; }
    return launch_sweep_vjp(c, d, gas_in, g, (float)lam, (float)kap, cot_out, cot_in, g_bar, scal_bar);
}

int dh_sweep_vjp(dh_ctx* c, int d, float* const gas_in[5], const float* g, double lam, double kap,
                 float* const cot_out[5], float* const cot_in[5], float* g_bar, double* scal_bar) {
    if (!c || d < 0 || d > 2 || !gas_in || !cot_out || !cot_in || !scal_bar || (g && !g_bar)) {
        set_error("dh_sweep_vjp: bad argument"); return DH_ERR_INVALID;
    }
    if (c->nc != 5) { set_error("dh_sweep_vjp: this context has dual_energy = 1, call dh_sweep_de_vjp"); return DH_ERR_INVALID; }
    return launch_sweep_vjp(c, d, gas_in, g, (float)lam, (float)kap, cot_out, cot_in, g_bar, scal_bar);
}

int dh_deposit(dh_ctx* c, const float* rho_gas, float* const pos[3], float* delta_out) {
    if (!c || !delta_out || (c->np > 0 && !pos)) { set_error("dh_deposit: bad argument"); return DH_ERR_INVALID; }
    return launch_deposit(c, rho_gas, pos ? pos[0] : nullptr, pos ? pos[1] : nullptr, pos ? pos[2] : nullptr, delta_out);
}

int dh_poisson(dh_ctx* c, const float* delta, double A, float* const g_out[3]) {
    if (!c || !delta || !g_out || !c->opt.gravity_on) { set_error("dh_poisson: bad argument or gravity off"); return DH_ERR_INVALID; }
    return poisson_forward(c, delta, (float)A, g_out);
}

int dh_poisson_vjp(dh_ctx* c, float* const g_bar[3], double A, float* delta_bar_out) {
    if (!c || !g_bar || !delta_bar_out || !c->opt.gravity_on) { set_error("dh_poisson_vjp: bad argument or gravity off"); return DH_ERR_INVALID; }
    return poisson_adjoint(c, g_bar, (float)A, delta_bar_out);
}

// The two scalar arguments of the Zel'dovich map from physical inputs (host only, fp64).  vel_factor = a^2 H(a) f(a) with
// the linear growth rate f = dlnD/dlna of a matter + curvature + Lambda background, D ~ H int_0^a da'/(a'H)^3:
//   f = dlnH/dlna + a / ((aE)^3 I),  E = H/H0,  I = int_0^a da'/(a'E)^3   (Simpson in s = sqrt(a'/a): smooth integrand);
// e_tilde0 = a0^2 k_B T0 / ((gamma-1) mu m_p) in (km/s)^2 (readings R18, R27).
int dh_ic_factors(const dh_cosmology* co, double a0, double T0, double gamma, double mu, double* vel_factor,
                  double* e_tilde0) {
    if (!co || !(a0 > 0) || !(gamma > 1.0) || !(mu > 0) || !(T0 >= 0) || !(co->Omega_m > 0)) {
        set_error("dh_ic_factors: need a0 > 0, gamma > 1, mu > 0, T0 >= 0, Omega_m > 0");
        return DH_ERR_INVALID;
    }
    const double Om = co->Omega_m, OL = co->Omega_L, Ok = 1.0 - Om - OL;
    auto E2 = [&](double a) { return Om / (a * a * a) + Ok / (a * a) + OL; };
    if (vel_factor) {
        const int M = 4096;
        double acc = 0.0;
        for (int j = 0; j <= M; ++j) {
            const double s = (double)j / M, ap = a0 * s * s;
            // da' = 2 a0 s ds;  1/(a'E)^3 = (a'^2 E2)^-3/2 with a'^2 E2 = Om/a' + Ok + OL a'^2
            const double q = j == 0 ? 0.0 : 2.0 * a0 * s / std::pow(Om / ap + Ok + OL * ap * ap, 1.5);
            acc += ((j == 0 || j == M) ? 1.0 : ((j & 1) ? 4.0 : 2.0)) * q;
        }
        const double I = acc / (3.0 * M);
        const double e2 = E2(a0), E = std::sqrt(e2);
        const double dlnH = (-3.0 * Om / (a0 * a0 * a0) - 2.0 * Ok / (a0 * a0)) / (2.0 * e2);
        const double aE = a0 * E;
        const double f = dlnH + a0 / (aE * aE * aE * I);
        *vel_factor = a0 * a0 * co->H0 * E * f;
    }
    if (e_tilde0) {
        const double kB = 1.380649e-23, mp = 1.67262192369e-27;     // J/K (SI), kg (CODATA 2018)
        *e_tilde0 = a0 * a0 * (kB * T0 / ((gamma - 1.0) * mu * mp)) * 1e-6;
    }
    return DH_OK;
}

static int check_ic(const dh_ctx* c, const float* delta_init, const char* who) {
    if (!c || !delta_init) { set_error("%s: null argument", who); return DH_ERR_INVALID; }
    if (!c->opt.gravity_on || c->nps != c->N) {
        set_error("%s: needs gravity_on and one particle per cell (n_part_side == grid_n)", who);
        return DH_ERR_INVALID;
    }
    return DH_OK;
}

int dh_ic_zeldovich(dh_ctx* c, const float* delta_init, double a0, double vel_factor, double e_tilde0, dh_state* out) {
    DH_TRY(check_ic(c, delta_init, "dh_ic_zeldovich"));
    if (!out) { set_error("dh_ic_zeldovich: null state"); return DH_ERR_INVALID; }
    DH_TRY(check_state(c, out->gas, out->part, out->eint));
    DH_TRY(poisson_forward(c, delta_init, 1.f, c->gp));                    // psi = grad^-1 of -delta: the A = 1 solve
    DH_TRY(launch_ic_state(c, delta_init, c->gp, out->gas, out->part, (float)vel_factor, (float)e_tilde0));
    if (c->nc == 6) {                                                      // q = rho e~_0 (reading R33)
        DH_TRY(launch_fill(c, out->eint, c->n3, 0.f));
        DH_TRY(launch_axpy(c, out->gas[0], out->eint, (float)e_tilde0));
    }
    out->a = a0; out->dt_prev = 0.0; out->step = 0;
    return DH_OK;
}

int dh_ic_zeldovich_vjp(dh_ctx* c, const float* delta_init, double vel_factor, double e_tilde0, const dh_cot* cot_state,
                        float* grad_delta) {
    DH_TRY(check_ic(c, delta_init, "dh_ic_zeldovich_vjp"));
    if (!cot_state || !grad_delta) { set_error("dh_ic_zeldovich_vjp: null argument"); return DH_ERR_INVALID; }
    for (int k = 0; k < 5; ++k) if (!cot_state->gas[k]) { set_error("dh_ic_zeldovich_vjp: null gas cotangent %d", k); return DH_ERR_INVALID; }
    DH_TRY(ensure_adjoint_scratch(c));
    DH_TRY(poisson_forward(c, delta_init, 1.f, c->gp));
    const float* cg[5] = {cot_state->gas[0], cot_state->gas[1], cot_state->gas[2], cot_state->gas[3], cot_state->gas[4]};
    if (c->nc == 6 && cot_state->eint) {                                   // q = rho e~_0: rho_b += e~_0 q_b, in scratch
        DH_CUDA(cudaMemcpyAsync(c->delta, cot_state->gas[0], c->n3 * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
        DH_TRY(launch_axpy(c, cot_state->eint, c->delta, (float)e_tilde0));
        cg[0] = c->delta;                                                  // consumed before the Poisson adjoint reuses it
    }
    DH_TRY(launch_ic_state_vjp(c, delta_init, c->gp, cg, cot_state->part, grad_delta, c->gpb,
                               (float)vel_factor, (float)e_tilde0));
    DH_TRY(poisson_adjoint(c, c->gpb, 1.f, c->delta));
    DH_TRY(launch_axpy(c, c->delta, grad_delta, 1.f));
    return DH_OK;
}

static int ps_scratch(dh_ctx* c, const char* who) {
    if (!c->opt.gravity_on || !c->own_fft) {
        set_error("%s: needs gravity_on and a power-of-two grid in [32, 1024] (the own FFT passes)", who);
        return DH_ERR_INVALID;
    }
    const int nb1 = c->N / 2 + 1;
    if (!c->ps_bins) DH_TRY(dev_alloc(c, (void**)&c->ps_bins, (size_t)nb1 * (2 * sizeof(double) + sizeof(float))));
    return DH_OK;
}

int dh_power_spectrum(dh_ctx* c, const float* field, double* power_out, double* count_out) {
    if (!c || !field || !power_out) { set_error("dh_power_spectrum: null argument"); return DH_ERR_INVALID; }
    DH_TRY(ps_scratch(c, "dh_power_spectrum"));
    const int nb1 = c->N / 2 + 1;
    DH_CUDA(cudaMemsetAsync(c->ps_bins, 0, (size_t)2 * nb1 * sizeof(double), c->stream));
    DH_TRY(own_power_spectrum(c, field, c->ps_bins));
    std::vector<double> h(2 * nb1);
    DH_CUDA(cudaMemcpyAsync(h.data(), c->ps_bins, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    const double norm = c->box * c->box * c->box / ((double)c->n3 * (double)c->n3);
    c->ps_count.assign(h.begin() + nb1, h.end());
    for (int b = 1; b < nb1; ++b) {
        power_out[b - 1] = h[nb1 + b] > 0 ? norm * h[b] / h[nb1 + b] : 0.0;
        if (count_out) count_out[b - 1] = h[nb1 + b];
    }
    return DH_OK;
}

int dh_power_spectrum_vjp(dh_ctx* c, const float* field, const double* power_bar, float* field_bar) {
    if (!c || !field || !power_bar || !field_bar) { set_error("dh_power_spectrum_vjp: null argument"); return DH_ERR_INVALID; }
    DH_TRY(ps_scratch(c, "dh_power_spectrum_vjp"));
    const int nb1 = c->N / 2 + 1;
    // mode counts per bin are a property of the grid: one pass of the forward kernel gives them, once per context
    if ((int)c->ps_count.size() != nb1) {
        DH_CUDA(cudaMemsetAsync(c->ps_bins, 0, (size_t)2 * nb1 * sizeof(double), c->stream));
        DH_TRY(own_power_spectrum(c, field, c->ps_bins));
        std::vector<double> h(2 * nb1);
        DH_CUDA(cudaMemcpyAsync(h.data(), c->ps_bins, h.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        DH_CUDA(cudaStreamSynchronize(c->stream));
        c->ps_count.assign(h.begin() + nb1, h.end());
    }
    const std::vector<double>& cnt = c->ps_count;
    const double norm = c->box * c->box * c->box / ((double)c->n3 * (double)c->n3);
    std::vector<float> g(nb1, 0.f);
    for (int b = 1; b < nb1; ++b) g[b] = cnt[b] > 0 ? (float)(2.0 * norm * power_bar[b - 1] / cnt[b]) : 0.f;
    float* gtab = reinterpret_cast<float*>(c->ps_bins + 2 * nb1);
    DH_CUDA(cudaMemcpyAsync(gtab, g.data(), nb1 * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));             // g is a local: the copy must finish before it goes away
    DH_TRY(own_power_spectrum_adjoint(c, field, gtab, field_bar));
    return DH_OK;
}

static int check_subgrid(const dh_ctx* c, float* const gas[5], const float* g0, const float* g1, const dh_subgrid_params* q,
                         const char* who) {
    if (!c || !gas || !g0 || !g1 || !q) { set_error("%s: null argument", who); return DH_ERR_INVALID; }
    for (int k = 0; k < 5; ++k) if (!gas[k]) { set_error("%s: null gas pointer %d", who, k); return DH_ERR_INVALID; }
    if (!(q->Pi0 > 0 && q->Pi0 < 1) || !(q->a_width > 0) || !(q->b_width > 0) || !(q->tau > 0) || !(q->rho_mean > 0)) {
        set_error("%s: need 0 < Pi0 < 1 and a_width, b_width, tau, rho_mean > 0", who);
        return DH_ERR_INVALID;
    }
    return DH_OK;
}

int dh_subgrid_step(dh_ctx* c, float* const gas[5], const float* g0, const float* g1, const dh_subgrid_params* par,
                    float* z_out, float* const pos[3], float* aux) {
    DH_TRY(check_subgrid(c, gas, g0, g1, par, "dh_subgrid_step"));
    if (aux && (!z_out || !pos || !pos[0] || !pos[1] || !pos[2])) {
        set_error("dh_subgrid_step: the particle readout needs z_out and the three position arrays");
        return DH_ERR_INVALID;
    }
    DH_TRY(launch_subgrid(c, gas, g0, g1, *par, z_out));
    if (aux) DH_TRY(launch_cic_readout(c, z_out, pos, aux));
    return DH_OK;
}

int dh_subgrid_step_vjp(dh_ctx* c, float* const gas_in[5], const float* g0, const float* g1, const dh_subgrid_params* par,
                        float* const cot_gas[5], const float* cot_z, double* dpar_out) {
    DH_TRY(check_subgrid(c, gas_in, g0, g1, par, "dh_subgrid_step_vjp"));
    if (!cot_gas) { set_error("dh_subgrid_step_vjp: null cotangent"); return DH_ERR_INVALID; }
    for (int k = 0; k < 5; ++k) if (!cot_gas[k]) { set_error("dh_subgrid_step_vjp: null cotangent %d", k); return DH_ERR_INVALID; }
    if (!c->sg_scal) DH_TRY(dev_alloc(c, (void**)&c->sg_scal, 4 * sizeof(double)));
    double h[4] = {0, 0, 0, 0};
    DH_CUDA(cudaMemsetAsync(c->sg_scal, 0, 4 * sizeof(double), c->stream));
    DH_TRY(launch_subgrid_vjp(c, gas_in, g0, g1, *par, cot_gas, cot_z, c->sg_scal));
    DH_CUDA(cudaMemcpyAsync(h, c->sg_scal, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    DH_CUDA(cudaStreamSynchronize(c->stream));
    if (dpar_out) for (int j = 0; j < 4; ++j) dpar_out[j] += h[j];
    return DH_OK;
}

int dh_data_term(dh_ctx* c, int observable, float* const gas[5], const float* data, const float* noise_var, double scale,
                 double weight, float* const cot_gas[5], double* loss_out) {
    if (!c || !gas || !data || (observable != 0 && observable != 1)) {
        set_error("dh_data_term: bad argument (observable is 0 = rho or 1 = internal energy density)");
        return DH_ERR_INVALID;
    }
    for (int k = 0; k < 5; ++k)
        if (!gas[k] || (cot_gas && !cot_gas[k])) { set_error("dh_data_term: null array %d", k); return DH_ERR_INVALID; }
    double* loss_dev = c->scal_dev + 6;                                    // spare slot of the scalar accumulators
    DH_CUDA(cudaMemsetAsync(loss_dev, 0, sizeof(double), c->stream));
    DH_TRY(launch_data_term(c, observable, gas, data, noise_var, (float)scale, (float)weight, cot_gas, loss_dev));
    if (loss_out) {
        DH_CUDA(cudaMemcpyAsync(loss_out, loss_dev, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        DH_CUDA(cudaStreamSynchronize(c->stream));
    }
    return DH_OK;
}

int dh_kick_drift(dh_ctx* c, float* const g[3], float* const part[6], double K, double dtau_over_dx) {
    if (!c || !part) { set_error("dh_kick_drift: bad argument"); return DH_ERR_INVALID; }
    return launch_kick_drift(c, g, part, part, (float)K, (float)dtau_over_dx);
}

}  // extern "C"
