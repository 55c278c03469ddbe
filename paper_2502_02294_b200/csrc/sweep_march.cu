// sweep_march.cu -- y and z sweeps of the relaxing-TVD scheme (forward and adjoint) as register-streaming
// ("marching") kernels for sm_100a.
//
// The scheme is the one stated at the top of sweep.cu (section 2.3.1-2.3.2, Eq. 9-18, :105-150; readings
// R3-R8, R11, R17 of DESIGN.md).  Layout: a warp's 32 lanes are 32 consecutive x (every load and store is one
// coalesced 128-byte row segment); a thread owns ONE pencil segment of `S` cells along the sweep axis and marches
// along it.  Everything the two Runge-Kutta stages need from neighbouring cells is carried in registers from one
// iteration to the next, so there is no shared-memory exchange, no barrier, and nothing is computed twice except the
// HALO cells at the two ends of a segment (3 forward, 4 adjoint).
//
// Forward pipeline, iteration that loads cell q (delay 3: it finishes cell q-3):
//   P(u_q) -> G_q, H_q ; D_{q-1} = G_{q-1} - H_q ; u*_{q-1} ; P(u*_{q-1}) -> G*_{q-1}, H*_{q-1}
//   PsiG_{q-2} = G*_{q-2} + L(dG_{q-3}, dG_{q-2})        dG_n = G*_{n+1} - G*_n
//   PsiH_{q-3} = H*_{q-2} - L(dH_{q-3}, dH_{q-2})        dH_n = H*_{n+1} - H*_n
//   Psi_{q-3}  = PsiG_{q-3} - PsiH_{q-3} ;  u'_{q-3} = R_{q-3} - (lam/2)(Psi_{q-3} - Psi_{q-4}),  R_n = u_n + kap S(u*_n, g_n)
// Adjoint pipeline (delay 4: the iteration that loads u_q, g_q and the output cotangent ob_{q-1} finishes u_b of cell
// q-4 and g_b of cell q-3): the forward recompute above, then with Psi_b_n = -(lam/2)(ob_n - ob_{n+1})
//   G-limiter of interface q-2 and H-limiter of interface q-3 -> G*_b, H*_b of cell q-3 complete
//   u*_b_{q-3} = P^T(u*_{q-3})(G*_b, H*_b) + source terms ;  D_b_{q-4} = -(lam/4)(u*_b_{q-4} - u*_b_{q-3})
//   u_b_{q-4} = ob + u*_b + (kap/2) source^T + P^T(u_{q-4})(D_b_{q-4}, -D_b_{q-5})
// lam_b is formed without carrying D or Psi:  stage B by summation by parts, sum_n Psi_n Psi_b_n / lam; stage A from
// u*_n - u_n - (kap/2) S = -(lam/4)(D_n - D_{n-1}).
#include "sweep_common.cuh"
#include "async_copy.cuh"

namespace dh {

// wrapped running offset along the sweep axis: off = base + p * stride, p in [0, N)
struct AxisPos {
    int p, off;
    __device__ __forceinline__ void set(int p_unwrapped, int N, int base, int stride) {
        p = p_unwrapped < 0 ? p_unwrapped + N : (p_unwrapped >= N ? p_unwrapped - N : p_unwrapped);
        off = base + p * stride;
    }
    __device__ __forceinline__ void next(int N, int base, int stride) {
        ++p; off += stride;
        if (p == N) { p = 0; off = base; }
    }
};

// ------------------------------------------------------------------------------------------------- forward ----
template <bool HAS_G, bool EPS>
struct FwdPipe {
    float u1[5], g1, G1[5], D2[5];       // u_{q-1}, g_{q-1}, G_{q-1}, D_{q-2}
    float R1[5], R2[5];                  // R_{q-2}, R_{q-3}
    float Gs[5], dGs[5], Hs[5], dHs[5];  // G*_{q-2}, dG_{q-3}, H*_{q-2}, dH_{q-3}
    float PG[5], Psi[5];                 // PsiG_{q-3}, Psi_{q-4}

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            u1[k] = 1.f; G1[k] = 0.f; D2[k] = 0.f; R1[k] = 0.f; R2[k] = 0.f; Gs[k] = 0.f; dGs[k] = 0.f; Hs[k] = 0.f;
            dHs[k] = 0.f; PG[k] = 0.f; Psi[k] = 0.f;
        }
        g1 = 0.f;
    }

    // take cell q; out = u'_{q-3}; c0 = freezing speed of cell q
    __device__ __forceinline__ void push(const float (&u0)[5], float g0, const SweepConst& sc, float (&out)[5], float& c0) {
        float G0[5], H0[5];
        prim_GH(u0, sc, G0, H0, c0);
        float us[5], D1[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            D1[k] = G1[k] - H0[k];
            us[k] = fmaf(-0.25f * sc.lam, D1[k] - D2[k], u1[k]);
        }
        float R0[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) R0[k] = u1[k];
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g1;
            us[1] = fmaf(hk, u1[0], us[1]);
            us[4] = fmaf(hk, u1[1], us[4]);
            const float kg = sc.kap * g1;
            R0[1] = fmaf(kg, us[0], R0[1]);
            R0[4] = fmaf(kg, us[1], R0[4]);
        }
        float Gs0[5], Hs0[5], cdummy;
        prim_GH(us, sc, Gs0, Hs0, cdummy);
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float dG0 = Gs0[k] - Gs[k];
            const float dH0 = Hs0[k] - Hs[k];
            const float PG0 = Gs[k] + limM<EPS>(dGs[k], dG0, sc.eps4);
            const float PH = Hs[k] - limM<EPS>(dHs[k], dH0, sc.eps4);
            const float Psi0 = PG[k] - PH;
            out[k] = fmaf(-0.5f * sc.lam, Psi0 - Psi[k], R2[k]);
            // rotate
            Psi[k] = Psi0; PG[k] = PG0;
            Gs[k] = Gs0[k]; dGs[k] = dG0; Hs[k] = Hs0[k]; dHs[k] = dH0;
            R2[k] = R1[k]; R1[k] = R0[k];
            u1[k] = u0[k]; G1[k] = G0[k]; D2[k] = D1[k];
        }
        g1 = g0;
    }
};

// Asynchronous staging ring.  Every thread copies the cells of ITS OWN pencil a few iterations ahead of their use with
// 4-byte cp.async (a warp's 32 copies are one coalesced 128-byte row segment) into ring[stage][field][thread] and reads
// them back with conflict-free LDS; since a thread only ever reads what it copied itself, cp.async.wait_group is the
// only synchronisation -- no barrier.  The ring hides the HBM latency that 12-16 resident warps of a register-heavy
// kernel cannot, and in the adjoint doubles as the window of already-visited cells (re-read instead of carried).
constexpr int RING = 8;          // stages (power of two)
constexpr int NTHR = 128;        // threads per block, fixed: ring offsets are immediates
constexpr int PF_FWD = 3;        // iterations of prefetch, forward
constexpr int PF_ADJ = 2;
constexpr int ADJ_UNROLL = 2;       // loop unrolling of the adjoint: 1 -> 404 us, 2 -> 366 us at 256^3
constexpr int ADJ_BLOCKS = 3;        // resident blocks per SM of the adjoint (168 registers)

// block = (BX lanes along x, BY pencils); grid = (N / BX, N / BY, segments along the sweep axis)
template <int DIR, bool HAS_G, bool EPS>
__global__ void __launch_bounds__(128, 4) sweep_march_fwd_kernel(Ptr5 in, const float* __restrict__ gfield, MPtr5 outp,
                                                                 float* cmax, SweepConst sc, int S,
                                                                 float* __restrict__ delta_out) {
    constexpr int HALO = 3, NF = HAS_G ? 6 : 5;
    extern __shared__ float ring[];              // [RING][NF][nthr]
    __shared__ int s_max;
    constexpr int nthr = NTHR;
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    if (tid == 0) s_max = 0;
    __syncthreads();
    const int N = sc.N;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int o = blockIdx.y * blockDim.y + threadIdx.y;
    const int p0 = blockIdx.z * S;
    const int len = min(S, N - p0);
    const int stride = DIR == 1 ? N : N * N;
    const int base = DIR == 1 ? o * N * N + x : o * N + x;
    const int niter = len + 2 * HALO;
    AxisPos ld;
    ld.set(p0 - HALO, N, base, stride);
    int off_out = base + p0 * stride;
    float* const my = ring + tid;
    auto issue = [&](int it) {
        float* dst = my + (it & (RING - 1)) * NF * nthr;
#pragma unroll
        for (int k = 0; k < 5; ++k) cp_async4(dst + k * nthr, in.p[k] + ld.off);
        if (HAS_G) cp_async4(dst + 5 * nthr, gfield + ld.off);
        ld.next(N, base, stride);
    };
#pragma unroll
    for (int it = 0; it < PF_FWD; ++it) {
        if (it < niter) issue(it);
        cp_async_commit();
    }
    FwdPipe<HAS_G, EPS> pipe;
    pipe.init();
    float cm = 0.f;
#pragma unroll 2
    for (int i = 0; i < niter; ++i) {
        if (i + PF_FWD < niter) issue(i + PF_FWD);
        cp_async_commit();
        cp_async_wait<PF_FWD>();
        const float* src = my + (i & (RING - 1)) * NF * nthr;
        float u0[5], g0 = 0.f;
#pragma unroll
        for (int k = 0; k < 5; ++k) u0[k] = src[k * nthr];
        if (HAS_G) g0 = src[5 * nthr];
        float out[5], c0;
        pipe.push(u0, g0, sc, out, c0);
        cm = (c0 > cm || c0 != c0) ? c0 : cm;
        if (i >= 2 * HALO) {
#pragma unroll
            for (int k = 0; k < 5; ++k) outp.p[k][off_out] = out[k];
            if (delta_out) delta_out[off_out] = fmaf(sc.src_flag, out[0], -sc.src_rho_bar);   // replaces source_init
            off_out += stride;
        }
    }
    if (cmax) block_max_to_global(cm, cmax, &s_max);
}

// --------------------------------------------------------------------------- forward, dual-energy variant ----
// The same pipeline with the sixth component q (sweep_de.cu states the scheme; readings R33-R36): P selects the thermal
// energy, the sixth flux component is q_s v, and the source -p dv/dx enters stage A for cell q-1 with v_q - v_{q-2} and
// stage B for cell q-3 with v*_{q-2} - v*_{q-4}: four more carried velocities and two pressures, no extra delay.
struct Ptr6m { const float* p[6]; };
struct MPtr6m { float* p[6]; };

template <bool HAS_G, bool EPS>
struct FwdPipeDE {
    float U1[6], g1, G1[6], D2[6];       // (u, q_s)_{q-1}, g_{q-1}, G_{q-1}, D_{q-2}
    float R1[6], R2[6];                  // R_{q-2}, R_{q-3}
    float Gs[6], dGs[6], Hs[6], dHs[6];  // G*_{q-2}, dG_{q-3}, H*_{q-2}, dH_{q-3}
    float PG[6], Psi[6];                 // PsiG_{q-3}, Psi_{q-4}
    float v1, v2, p1;                    // v_{q-1}, v_{q-2}, p_{q-1}
    float vsA, vsB, vsC, psA, psB;       // v*_{q-2}, v*_{q-3}, v*_{q-4}, p*_{q-2}, p*_{q-3}

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            U1[k] = 1.f; G1[k] = 0.f; D2[k] = 0.f; R1[k] = 0.f; R2[k] = 0.f; Gs[k] = 0.f; dGs[k] = 0.f; Hs[k] = 0.f;
            dHs[k] = 0.f; PG[k] = 0.f; Psi[k] = 0.f;
        }
        g1 = 0.f; v1 = v2 = p1 = 0.f; vsA = vsB = vsC = psA = psB = 0.f;
    }

    // take cell q; out = (u', q')_{q-3}; c0 = freezing speed of cell q
    __device__ __forceinline__ void push(const float (&u0)[6], float g0, const SweepConst& sc, float (&out)[6], float& c0) {
        float G0[6], H0[6], v0, p0, qs0;
        prim_de(u0, sc, G0, H0, c0, v0, p0, qs0);
        float us[6], D1[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            D1[k] = G1[k] - H0[k];
            us[k] = fmaf(-0.25f * sc.lam, D1[k] - D2[k], U1[k]);
        }
        us[5] = fmaf(-0.25f * sc.lam * p1, v0 - v2, us[5]);
        float R0[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) R0[k] = U1[k];
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g1;
            us[1] = fmaf(hk, U1[0], us[1]);
            us[4] = fmaf(hk, U1[1], us[4]);
            const float kg = sc.kap * g1;
            R0[1] = fmaf(kg, us[0], R0[1]);
            R0[4] = fmaf(kg, us[1], R0[4]);
        }
        float Gs0[6], Hs0[6], cdummy, vs0, ps0, qdummy;
        prim_de(us, sc, Gs0, Hs0, cdummy, vs0, ps0, qdummy);
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float dG0 = Gs0[k] - Gs[k];
            const float dH0 = Hs0[k] - Hs[k];
            const float PG0 = Gs[k] + limM<EPS>(dGs[k], dG0, sc.eps4);
            const float PH = Hs[k] - limM<EPS>(dHs[k], dH0, sc.eps4);
            const float Psi0 = PG[k] - PH;
            out[k] = fmaf(-0.5f * sc.lam, Psi0 - Psi[k], R2[k]);
            Psi[k] = Psi0; PG[k] = PG0;
            Gs[k] = Gs0[k]; dGs[k] = dG0; Hs[k] = Hs0[k]; dHs[k] = dH0;
            R2[k] = R1[k]; R1[k] = R0[k];
            G1[k] = G0[k]; D2[k] = D1[k];
        }
        out[5] = fmaf(-0.5f * sc.lam * psB, vsA - vsC, out[5]);
#pragma unroll
        for (int k = 0; k < 5; ++k) U1[k] = u0[k];
        U1[5] = qs0;
        g1 = g0;
        v2 = v1; v1 = v0; p1 = p0;
        vsC = vsB; vsB = vsA; vsA = vs0;
        psB = psA; psA = ps0;
    }
};

template <int DIR, bool HAS_G, bool EPS>
__global__ void __launch_bounds__(128, 3) sweep_march_fwd_de_kernel(Ptr6m in, const float* __restrict__ gfield, MPtr6m outp,
                                                                    float* cmax, SweepConst sc, int S) {
    constexpr int HALO = 3, NF = HAS_G ? 7 : 6;
    extern __shared__ float ring[];              // [RING][NF][nthr]
    __shared__ int s_max;
    constexpr int nthr = NTHR;
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    if (tid == 0) s_max = 0;
    __syncthreads();
    const int N = sc.N;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int o = blockIdx.y * blockDim.y + threadIdx.y;
    const int p0 = blockIdx.z * S;
    const int len = min(S, N - p0);
    const int stride = DIR == 1 ? N : N * N;
    const int base = DIR == 1 ? o * N * N + x : o * N + x;
    const int niter = len + 2 * HALO;
    AxisPos ld;
    ld.set(p0 - HALO, N, base, stride);
    int off_out = base + p0 * stride;
    float* const my = ring + tid;
    auto issue = [&](int it) {
        float* dst = my + (it & (RING - 1)) * NF * nthr;
#pragma unroll
        for (int k = 0; k < 6; ++k) cp_async4(dst + k * nthr, in.p[k] + ld.off);
        if (HAS_G) cp_async4(dst + 6 * nthr, gfield + ld.off);
        ld.next(N, base, stride);
    };
#pragma unroll
    for (int it = 0; it < PF_FWD; ++it) {
        if (it < niter) issue(it);
        cp_async_commit();
    }
    FwdPipeDE<HAS_G, EPS> pipe;
    pipe.init();
    float cm = 0.f;
#pragma unroll 2
    for (int i = 0; i < niter; ++i) {
        if (i + PF_FWD < niter) issue(i + PF_FWD);
        cp_async_commit();
        cp_async_wait<PF_FWD>();
        const float* src = my + (i & (RING - 1)) * NF * nthr;
        float u0[6], g0 = 0.f;
#pragma unroll
        for (int k = 0; k < 6; ++k) u0[k] = src[k * nthr];
        if (HAS_G) g0 = src[6 * nthr];
        float out[6], c0;
        pipe.push(u0, g0, sc, out, c0);
        // the CFL maximum is over the sweep's own cells (the halo cells belong to the neighbouring segments)
        if (i >= HALO && i < len + HALO) cm = (c0 > cm || c0 != c0) ? c0 : cm;
        if (i >= 2 * HALO) {
#pragma unroll
            for (int k = 0; k < 6; ++k) outp.p[k][off_out] = out[k];
            off_out += stride;
        }
    }
    if (cmax) block_max_to_global(cm, cmax, &s_max);
}

// ------------------------------------------------------------------------------------------------- adjoint ----
// LK = false drops the cotangents of lam and kap (dh_options.want_dsched = 0): gamma_b only.
template <bool HAS_G, int EPS, bool LK>
struct AdjPipe {
    // forward recompute
    float u1[5], g1, G1[5], D2[5];         // u_{q-1}, g_{q-1}, G_{q-1}, D_{q-2}
    float us1[5], us2[5];                  // u*_{q-2}, u*_{q-3}
    float Gs[5], dGs[5], Hs[5], dHs[5];    // G*_{q-2}, dG_{q-3}, H*_{q-2}, dH_{q-3}
    // cotangents in flight
    float GB0[5], GB1[5];                  // partial G*_b of cells q-3 (interfaces q-4, q-3) and q-2 (interface q-3)
    float HB0[5], HB1[5];                  // partial H*_b of cells q-3 (interfaces q-5, q-4) and q-2 (interface q-4)
    float accR[5], usbR[5], DbR[5];        // ob + u*_b + source^T of cell q-4, u*_b_{q-4}, D_b_{q-5}

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            u1[k] = 1.f; G1[k] = 0.f; D2[k] = 0.f; us1[k] = 1.f; us2[k] = 1.f; Gs[k] = 0.f; dGs[k] = 0.f; Hs[k] = 0.f;
            dHs[k] = 0.f; GB0[k] = 0.f; GB1[k] = 0.f; HB0[k] = 0.f; HB1[k] = 0.f;
            accR[k] = 0.f; usbR[k] = 0.f; DbR[k] = 0.f;
        }
        g1 = 0.f;
    }

    // Takes u_q, g_q and, re-read from the ring, ob_{q-1}, ob_{q-2}, ob_{q-3}, u_{q-3}, g_{q-3}, u_{q-4}.  Returns
    // ub = u_b of cell q-4, gb = g_b of cell q-3, and the scalar-cotangent terms of this iteration split by the cell /
    // interface they belong to so the caller can count each once: lamG (interface q-2), lamH (interface q-3), and
    // for cell q-3: lamA, kapM, gamM; for cell q-4: gamR.
    __device__ __forceinline__ void push(const float (&u0)[5], float g0, const float (&ob0)[5], const float (&ob1)[5],
                                         const float (&ob2)[5], const float (&uM)[5], float gM, const float (&uR)[5],
                                         const SweepConst& sc, float (&ub)[5], float& gb, float& lamG, float& lamH,
                                         float& lamA, float& kapM, float& gamM, float& gamR) {
        // ---- forward recompute: P(u_q), u*_{q-1}, P(u*_{q-1})
        float G0[5], H0[5], cdummy;
        prim_GH(u0, sc, G0, H0, cdummy);
        float us0[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float D1 = G1[k] - H0[k];
            us0[k] = fmaf(-0.25f * sc.lam, D1 - D2[k], u1[k]);
            D2[k] = D1;
        }
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g1;
            us0[1] = fmaf(hk, u1[0], us0[1]);
            us0[4] = fmaf(hk, u1[1], us0[4]);
        }
        float Gs0[5], Hs0[5];
        prim_GH(us0, sc, Gs0, Hs0, cdummy);
        // ---- limiters: G side of interface q-2, H side of interface q-3; G*_b, H*_b of cell q-3 complete
        float GsB[5], HsB[5];
        float lg = 0.f, lh = 0.f;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float dG0 = Gs0[k] - Gs[k];
            const float dH0 = Hs0[k] - Hs[k];
            float LA, LB, MA, MB;
            const float L = limM_grad<EPS>(dGs[k], dG0, sc.eps4, LA, LB);
            const float M = limM_grad<EPS>(dHs[k], dH0, sc.eps4, MA, MB);
            const float dob0 = ob1[k] - ob0[k];           // ob_{q-2} - ob_{q-1}
            const float dob1 = ob2[k] - ob1[k];           // ob_{q-3} - ob_{q-2}
            const float pb0 = -0.5f * sc.lam * dob0;      // Psi_b of interface q-2
            const float pb1 = -0.5f * sc.lam * dob1;      // Psi_b of interface q-3
            if (LK) {
                lg = fmaf(Gs[k] + L, dob0, lg);           // PsiG_{q-2} (ob_{q-2} - ob_{q-1})
                lh = fmaf(Hs[k] - M, dob1, lh);           // PsiH_{q-3} (ob_{q-3} - ob_{q-2})
            }
            GsB[k] = fmaf(-LA, pb0, GB0[k]);
            GB0[k] = fmaf(1.f + LA - LB, pb0, GB1[k]);
            GB1[k] = LB * pb0;
            HsB[k] = fmaf(-MA, pb1, HB0[k]);
            HB0[k] = fmaf(-1.f + MA - MB, pb1, HB1[k]);
            HB1[k] = MB * pb1;
            Gs[k] = Gs0[k]; dGs[k] = dG0; Hs[k] = Hs0[k]; dHs[k] = dH0;
        }
        lamG = -0.5f * lg;
        lamH = 0.5f * lh;
        // ---- cell m = q-3: u*_b, g_b, the additive part of u_b
        float usb[5];
        gamM = 0.f;
        prim_GH_vjp(us2, sc, GsB, HsB, usb, gamM);
        float acc[5];
        gb = 0.f; kapM = 0.f;
        if (HAS_G) {
            const float kg = sc.kap * gM;
            usb[0] = fmaf(kg, ob2[1], usb[0]);
            usb[1] = fmaf(kg, ob2[4], usb[1]);
        }
#pragma unroll
        for (int k = 0; k < 5; ++k) acc[k] = ob2[k] + usb[k];
        float dA = 0.f;                                   // sum_k u*_b (u - u* + (kap/2) g S(u))
        if (LK) {
#pragma unroll
            for (int k = 0; k < 5; ++k) dA = fmaf(usb[k], uM[k] - us2[k], dA);
        }
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * gM;
            acc[0] = fmaf(hk, usb[1], acc[0]);
            acc[1] = fmaf(hk, usb[4], acc[1]);
            const float tB = us2[0] * ob2[1] + us2[1] * ob2[4];
            const float tA = uM[0] * usb[1] + uM[1] * usb[4];
            const float t = fmaf(0.5f, tA, tB);
            gb = sc.kap * t;
            if (LK) { kapM = gM * t; dA = fmaf(hk, tA, dA); }
        }
        lamA = -sc.inv_lam * dA;
        // ---- cell r = q-4: stage-A transpose
        float Gb[5], Hb[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float Db = -0.25f * sc.lam * (usbR[k] - usb[k]);
            Gb[k] = Db;
            Hb[k] = -DbR[k];
            DbR[k] = Db;
            usbR[k] = usb[k];
        }
        gamR = 0.f;
        prim_GH_vjp(uR, sc, Gb, Hb, ub, gamR);
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            ub[k] += accR[k];
            accR[k] = acc[k];
            // rotate the rest
            us2[k] = us1[k]; us1[k] = us0[k];
            u1[k] = u0[k]; G1[k] = G0[k];
        }
        g1 = g0;
    }
};

template <int DIR, bool HAS_G, int EPS, bool LK>
__global__ void __launch_bounds__(128, ADJ_BLOCKS) sweep_march_adj_kernel(Ptr5 in, const float* __restrict__ gfield,
                                                                          Ptr5 cot_out, MPtr5 cot_in,
                                                                          float* __restrict__ gbar, double* scal,
                                                                          SweepConst sc, int S) {
    constexpr int HALO = 4, NF = HAS_G ? 11 : 10, OB = HAS_G ? 6 : 5;
    extern __shared__ float ring[];              // [RING][NF][nthr]: u (5), g, ob (5) of one cell per stage
    __shared__ float s_red[96];
    constexpr int nthr = NTHR;
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int N = sc.N;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int o = blockIdx.y * blockDim.y + threadIdx.y;
    const int p0 = blockIdx.z * S;
    const int len = min(S, N - p0);
    const int stride = DIR == 1 ? N : N * N;
    const int base = DIR == 1 ? o * N * N + x : o * N + x;
    const int niter = len + 2 * HALO;
    AxisPos ld;
    ld.set(p0 - HALO, N, base, stride);
    int off_m = base + (p0 - 1) * stride;         // cell q-3 (g_b store), valid from the first owned cell on
    int off_r = base + (p0 - 1) * stride;         // cell q-4 (u_b store)
    float* const my = ring + tid;
    auto issue = [&](int it) {
        float* dst = my + (it & (RING - 1)) * NF * nthr;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            cp_async4(dst + k * nthr, in.p[k] + ld.off);
            cp_async4(dst + (OB + k) * nthr, cot_out.p[k] + ld.off);
        }
        if (HAS_G) cp_async4(dst + 5 * nthr, gfield + ld.off);
        ld.next(N, base, stride);
    };
    // stages -4 .. -1 are read (as ob / re-read cells) before they were ever filled: give them finite values
#pragma unroll
    for (int st = RING - 4; st < RING; ++st)
#pragma unroll
        for (int k = 0; k < NF; ++k) my[(st * NF + k) * nthr] = k < 5 ? 1.f : 0.f;
#pragma unroll
    for (int it = 0; it < PF_ADJ; ++it) {
        if (it < niter) issue(it);
        cp_async_commit();
    }
    AdjPipe<HAS_G, EPS, LK> pipe;
    pipe.init();
    float lacc = 0.f, kacc = 0.f, gacc = 0.f;
#pragma unroll ADJ_UNROLL
    for (int i = 0; i < niter; ++i) {
        if (i + PF_ADJ < niter) issue(i + PF_ADJ);
        cp_async_commit();
        cp_async_wait<PF_ADJ>();
        const float* s0 = my + (i & (RING - 1)) * NF * nthr;
        const float* s1 = my + ((i - 1) & (RING - 1)) * NF * nthr;
        const float* s2 = my + ((i - 2) & (RING - 1)) * NF * nthr;
        const float* s3 = my + ((i - 3) & (RING - 1)) * NF * nthr;
        const float* s4 = my + ((i - 4) & (RING - 1)) * NF * nthr;
        float u0[5], ob0[5], ob1[5], ob2[5], uM[5], uR[5], g0 = 0.f, gM = 0.f;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            u0[k] = s0[k * nthr];
            ob0[k] = s1[(OB + k) * nthr];
            ob1[k] = s2[(OB + k) * nthr];
            ob2[k] = s3[(OB + k) * nthr];
            uM[k] = s3[k * nthr];
            uR[k] = s4[k * nthr];
        }
        if (HAS_G) { g0 = s0[5 * nthr]; gM = s3[5 * nthr]; }
        float ub[5], gb, lamG, lamH, lamA, kapM, gamM, gamR;
        pipe.push(u0, g0, ob0, ob1, ob2, uM, gM, uR, sc, ub, gb, lamG, lamH, lamA, kapM, gamM, gamR);
        // interface q-2 = p0 + i - 6, cell / interface q-3 = p0 + i - 7, cell q-4 = p0 + i - 8
        if (LK && i >= 6 && i < len + 6) lacc += lamG;
        if (i >= 7) {
            off_m += stride;
            if (i < len + 7) {
                if (LK) { lacc += lamH + lamA; kacc += kapM; }
                gacc += gamM;
                if (HAS_G) gbar[off_m] = gb;
            }
        }
        if (i >= 8) {
            off_r += stride;
            gacc += gamR;
#pragma unroll
            for (int k = 0; k < 5; ++k) cot_in.p[k][off_r] = ub[k];
        }
    }
    block_sum3_to_global(lacc, kacc, gacc, scal, s_red);
}

// --------------------------------------------------------------------------- adjoint, dual-energy variant ----
// AdjPipe with the sixth component and the transposes of the two source terms (gamma_b only: a context that wants the
// cotangents of Dtau and kappa goes through the chain kernels of sweep_de.cu).  With t_n = p*_n q'_b,n and tA_n = p_n q*_b,n:
//   cell m = q-3:  v*_b = -(lam/2)(t_{q-4} - t_{q-2}),   p*_b = -(lam/2) q'_b,m (v*_{q-2} - v*_{q-4})      -> P^T(u*_m, q*_m)
//   cell r = q-4:  v_b  = -(lam/4)(tA_{q-5} - tA_{q-3}), p_b  = -(lam/4) q*_b,r (v_{q-3} - v_{q-5}),  q_s_b = q'_b,r + q*_b,r -> P^T(u_r, q_r)
template <bool HAS_G, int EPS>
struct AdjPipeDE {
    float U1[6], g1, G1[6], D2[6];         // (u, q_s)_{q-1}, g_{q-1}, G_{q-1}, D_{q-2}
    float us1[6], us2[6];                  // (u*, q*)_{q-2}, (u*, q*)_{q-3}
    float Gs[6], dGs[6], Hs[6], dHs[6];    // G*_{q-2}, dG_{q-3}, H*_{q-2}, dH_{q-3}
    float GB0[6], GB1[6], HB0[6], HB1[6];  // partial G*_b, H*_b in flight (as AdjPipe)
    float accR[5], qsbR, usbR[6], DbR[6];  // cell q-4: ob + u*_b + source^T, q'_b + q*_b, (u*, q*)_b; D_b_{q-5}
    float v1, v2, v3, v4, v5, p1, p2, p3;  // v_{q-1 .. q-5}, p_{q-1 .. q-3} of the input cells
    float tA4, tA5;                        // tA_{q-4}, tA_{q-5}
    float vsA, vsB, vsC, psA, psB, psC;    // v*, p* of cells q-2, q-3, q-4
    float obq4;                            // q'_b of cell q-4

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            U1[k] = 1.f; G1[k] = 0.f; D2[k] = 0.f; us1[k] = 1.f; us2[k] = 1.f; Gs[k] = 0.f; dGs[k] = 0.f; Hs[k] = 0.f;
            dHs[k] = 0.f; GB0[k] = 0.f; GB1[k] = 0.f; HB0[k] = 0.f; HB1[k] = 0.f; usbR[k] = 0.f; DbR[k] = 0.f;
        }
#pragma unroll
        for (int k = 0; k < 5; ++k) accR[k] = 0.f;
        qsbR = 0.f; g1 = 0.f;
        v1 = v2 = v3 = v4 = v5 = p1 = p2 = p3 = tA4 = tA5 = 0.f;
        vsA = vsB = vsC = psA = psB = psC = obq4 = 0.f;
    }

    __device__ __forceinline__ void push(const float (&u0)[6], float g0, const float (&ob0)[6], const float (&ob1)[6],
                                         const float (&ob2)[6], const float (&uM)[6], float gM, const float (&uR)[6],
                                         const SweepConst& sc, float (&ub)[6], float& gb, float& gamM, float& gamR) {
        // ---- forward recompute: P(u_q), (u*, q*)_{q-1}, P of it
        float G0[6], H0[6], cdummy, v0, p0, qs0;
        prim_de(u0, sc, G0, H0, cdummy, v0, p0, qs0);
        float us0[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float D1 = G1[k] - H0[k];
            us0[k] = fmaf(-0.25f * sc.lam, D1 - D2[k], U1[k]);
            D2[k] = D1;
        }
        us0[5] = fmaf(-0.25f * sc.lam * p1, v0 - v2, us0[5]);
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g1;
            us0[1] = fmaf(hk, U1[0], us0[1]);
            us0[4] = fmaf(hk, U1[1], us0[4]);
        }
        float Gs0[6], Hs0[6], vs0, ps0, qdummy;
        prim_de(us0, sc, Gs0, Hs0, cdummy, vs0, ps0, qdummy);
        // ---- limiters: G side of interface q-2, H side of interface q-3; G*_b, H*_b of cell q-3 complete
        float GsB[6], HsB[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float dG0 = Gs0[k] - Gs[k];
            const float dH0 = Hs0[k] - Hs[k];
            float LA, LB, MA, MB;
            limM_grad<EPS>(dGs[k], dG0, sc.eps4, LA, LB);
            limM_grad<EPS>(dHs[k], dH0, sc.eps4, MA, MB);
            const float pb0 = -0.5f * sc.lam * (ob1[k] - ob0[k]);      // Psi_b of interface q-2
            const float pb1 = -0.5f * sc.lam * (ob2[k] - ob1[k]);      // Psi_b of interface q-3
            GsB[k] = fmaf(-LA, pb0, GB0[k]);
            GB0[k] = fmaf(1.f + LA - LB, pb0, GB1[k]);
            GB1[k] = LB * pb0;
            HsB[k] = fmaf(-MA, pb1, HB0[k]);
            HB0[k] = fmaf(-1.f + MA - MB, pb1, HB1[k]);
            HB1[k] = MB * pb1;
            Gs[k] = Gs0[k]; dGs[k] = dG0; Hs[k] = Hs0[k]; dHs[k] = dH0;
        }
        // ---- cell m = q-3
        const float vsb = -0.5f * sc.lam * (psC * obq4 - psA * ob1[5]);
        const float psb = -0.5f * sc.lam * ob2[5] * (vsA - vsC);
        float usb[6];
        gamM = 0.f;
        prim_de_vjp(us2, sc, GsB, HsB, vsb, psb, 0.f, usb, gamM);
        gb = 0.f;
        if (HAS_G) {
            const float kg = sc.kap * gM;
            usb[0] = fmaf(kg, ob2[1], usb[0]);
            usb[1] = fmaf(kg, ob2[4], usb[1]);
        }
        float acc[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) acc[k] = ob2[k] + usb[k];
        const float qsb = ob2[5] + usb[5];
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * gM;
            acc[0] = fmaf(hk, usb[1], acc[0]);
            acc[1] = fmaf(hk, usb[4], acc[1]);
            const float tB = us2[0] * ob2[1] + us2[1] * ob2[4];
            const float tAg = uM[0] * usb[1] + uM[1] * usb[4];
            gb = sc.kap * fmaf(0.5f, tAg, tB);
        }
        // ---- cell r = q-4: stage-A transpose
        float Gb[6], Hb[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float Db = -0.25f * sc.lam * (usbR[k] - usb[k]);
            Gb[k] = Db;
            Hb[k] = -DbR[k];
            DbR[k] = Db;
        }
        const float tA3 = p3 * usb[5];
        const float vb = -0.25f * sc.lam * (tA5 - tA3);
        const float pb = -0.25f * sc.lam * usbR[5] * (v3 - v5);
        gamR = 0.f;
        prim_de_vjp(uR, sc, Gb, Hb, vb, pb, qsbR, ub, gamR);
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            ub[k] += accR[k];
            accR[k] = acc[k];
        }
        qsbR = qsb;
        // ---- rotate
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            usbR[k] = usb[k];
            us2[k] = us1[k]; us1[k] = us0[k];
            G1[k] = G0[k];
        }
#pragma unroll
        for (int k = 0; k < 5; ++k) U1[k] = u0[k];
        U1[5] = qs0;
        g1 = g0;
        v5 = v4; v4 = v3; v3 = v2; v2 = v1; v1 = v0;
        p3 = p2; p2 = p1; p1 = p0;
        tA5 = tA4; tA4 = tA3;
        vsC = vsB; vsB = vsA; vsA = vs0;
        psC = psB; psB = psA; psA = ps0;
        obq4 = ob2[5];
    }
};

template <int DIR, bool HAS_G, int EPS>
__global__ void __launch_bounds__(128, 2) sweep_march_adj_de_kernel(Ptr6m in, const float* __restrict__ gfield, Ptr6m cot_out,
                                                                    MPtr6m cot_in, float* __restrict__ gbar, double* scal,
                                                                    SweepConst sc, int S) {
    constexpr int HALO = 4, NF = HAS_G ? 13 : 12, OB = HAS_G ? 7 : 6;
    extern __shared__ float ring[];              // [RING][NF][nthr]: (u, q) (6), g, ob (6) of one cell per stage
    __shared__ float s_red[96];
    constexpr int nthr = NTHR;
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int N = sc.N;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int o = blockIdx.y * blockDim.y + threadIdx.y;
    const int p0 = blockIdx.z * S;
    const int len = min(S, N - p0);
    const int stride = DIR == 1 ? N : N * N;
    const int base = DIR == 1 ? o * N * N + x : o * N + x;
    const int niter = len + 2 * HALO;
    AxisPos ld;
    ld.set(p0 - HALO, N, base, stride);
    int off_m = base + (p0 - 1) * stride;
    int off_r = base + (p0 - 1) * stride;
    float* const my = ring + tid;
    auto issue = [&](int it) {
        float* dst = my + (it & (RING - 1)) * NF * nthr;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            cp_async4(dst + k * nthr, in.p[k] + ld.off);
            cp_async4(dst + (OB + k) * nthr, cot_out.p[k] + ld.off);
        }
        if (HAS_G) cp_async4(dst + 6 * nthr, gfield + ld.off);
        ld.next(N, base, stride);
    };
#pragma unroll
    for (int st = RING - 4; st < RING; ++st)
#pragma unroll
        for (int k = 0; k < NF; ++k) my[(st * NF + k) * nthr] = k < 6 ? 1.f : 0.f;
#pragma unroll
    for (int it = 0; it < PF_ADJ; ++it) {
        if (it < niter) issue(it);
        cp_async_commit();
    }
    AdjPipeDE<HAS_G, EPS> pipe;
    pipe.init();
    float gacc = 0.f;
#pragma unroll 1
    for (int i = 0; i < niter; ++i) {
        if (i + PF_ADJ < niter) issue(i + PF_ADJ);
        cp_async_commit();
        cp_async_wait<PF_ADJ>();
        const float* s0 = my + (i & (RING - 1)) * NF * nthr;
        const float* s1 = my + ((i - 1) & (RING - 1)) * NF * nthr;
        const float* s2 = my + ((i - 2) & (RING - 1)) * NF * nthr;
        const float* s3 = my + ((i - 3) & (RING - 1)) * NF * nthr;
        const float* s4 = my + ((i - 4) & (RING - 1)) * NF * nthr;
        float u0[6], ob0[6], ob1[6], ob2[6], uM[6], uR[6], g0 = 0.f, gM = 0.f;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            u0[k] = s0[k * nthr];
            ob0[k] = s1[(OB + k) * nthr];
            ob1[k] = s2[(OB + k) * nthr];
            ob2[k] = s3[(OB + k) * nthr];
            uM[k] = s3[k * nthr];
            uR[k] = s4[k * nthr];
        }
        if (HAS_G) { g0 = s0[6 * nthr]; gM = s3[6 * nthr]; }
        float ub[6], gb, gamM, gamR;
        pipe.push(u0, g0, ob0, ob1, ob2, uM, gM, uR, sc, ub, gb, gamM, gamR);
        if (i >= 7) {
            off_m += stride;
            if (i < len + 7) {
                gacc += gamM;
                if (HAS_G) gbar[off_m] = gb;
            }
        }
        if (i >= 8) {
            off_r += stride;
            gacc += gamR;
#pragma unroll
            for (int k = 0; k < 6; ++k) cot_in.p[k][off_r] = ub[k];
        }
    }
    block_sum3_to_global(0.f, 0.f, gacc, scal, s_red);
}

// ----------------------------------------------------------------------------------------------- launchers ----
#define MARCH_LAUNCH(kern, grid, block, sm, stream, ...)                                                        \
    do {                                                                                                        \
        if ((sm) + 2048 > 48 * 1024)             /* static shared memory counts against the 48 KB default too */       \
            DH_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sm)));        \
        kern<<<grid, block, sm, stream>>>(__VA_ARGS__);                                                         \
    } while (0)

// NTHR threads: as many lanes along x as divide N, the rest along the pencil index (N is a multiple of 32)
static dim3 march_block(int N) {
    const int bx = N % 128 == 0 ? 128 : (N % 64 == 0 ? 64 : 32);
    return dim3(bx, NTHR / bx, 1);
}

static int march_segment(int N, int tuned, int halo) {
    // segment length: long enough that the 2*halo recomputed cells stay a small fraction, short enough that the grid
    // holds several waves of blocks on 148 SMs
    int S = tuned > 0 ? tuned : (N >= 256 ? 128 : (N >= 128 ? 64 : 32));
    if (S > N) S = N;
    if (S < 2 * halo) S = 2 * halo;
    return S;
}

template <int DIR>
static int march_fwd_dispatch(dh_ctx* c, dim3 grid, dim3 block, const Ptr5& pin, const float* g, const MPtr5& pout,
                              float* cmax, const SweepConst& sc, int S, bool eps, float* delta_out) {
    const size_t sm = (size_t)RING * (g ? 6 : 5) * block.x * block.y * sizeof(float);
    if (g) {
        if (eps) MARCH_LAUNCH((sweep_march_fwd_kernel<DIR, true, true>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S, delta_out);
        else MARCH_LAUNCH((sweep_march_fwd_kernel<DIR, true, false>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S, delta_out);
    } else {
        if (eps) MARCH_LAUNCH((sweep_march_fwd_kernel<DIR, false, true>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S, delta_out);
        else MARCH_LAUNCH((sweep_march_fwd_kernel<DIR, false, false>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S, delta_out);
    }
    return DH_OK;
}

template <int DIR, bool LK, bool HAS_G, int EPS>
static int march_adj_launch(dh_ctx* c, dim3 grid, dim3 block, const Ptr5& pin, const float* g, const Ptr5& pco,
                            const MPtr5& pci, float* gbar, double* scal, const SweepConst& sc, int S) {
    const size_t sm = (size_t)RING * (HAS_G ? 11 : 10) * block.x * block.y * sizeof(float);
    MARCH_LAUNCH((sweep_march_adj_kernel<DIR, HAS_G, EPS, LK>), grid, block, sm, c->stream, pin, g, pco, pci, gbar, scal, sc, S);
    return DH_OK;
}

// eps_mode: 1 = sign(A) 4 eps in denominator and numerators (lim_eps > 1e-18), 2 = denominator only, 0 = lim_eps == 0
template <int DIR, bool LK>
static int march_adj_dispatch(dh_ctx* c, dim3 grid, dim3 block, const Ptr5& pin, const float* g, const Ptr5& pco,
                              const MPtr5& pci, float* gbar, double* scal, const SweepConst& sc, int S, int eps_mode) {
#define DH_ADJ_CASE(G_, E_) return march_adj_launch<DIR, LK, G_, E_>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S)
    if (g) { if (eps_mode == 1) DH_ADJ_CASE(true, 1); if (eps_mode == 2) DH_ADJ_CASE(true, 2); DH_ADJ_CASE(true, 0); }
    if (eps_mode == 1) DH_ADJ_CASE(false, 1);
    if (eps_mode == 2) DH_ADJ_CASE(false, 2);
    DH_ADJ_CASE(false, 0);
#undef DH_ADJ_CASE
}

int launch_sweep_march(dh_ctx* c, int d, const Ptr5& pin, const float* g, const MPtr5& pout, float* cmax,
                       const SweepConst& sc, float* delta_out) {
    const int N = c->N;
    const int S = march_segment(N, c->tune_march_s_fwd, 3);
    const dim3 block = march_block(N);
    const dim3 grid(N / block.x, N / block.y, (N + S - 1) / S);
    const bool eps = c->opt.lim_eps > 1e-18;
    if (d == 1) DH_TRY(march_fwd_dispatch<1>(c, grid, block, pin, g, pout, cmax, sc, S, eps, delta_out));
    else DH_TRY(march_fwd_dispatch<2>(c, grid, block, pin, g, pout, cmax, sc, S, eps, delta_out));
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

template <int DIR>
static int march_fwd_de_dispatch(dh_ctx* c, dim3 grid, dim3 block, const Ptr6m& pin, const float* g, const MPtr6m& pout,
                                 float* cmax, const SweepConst& sc, int S, bool eps) {
    const size_t sm = (size_t)RING * (g ? 7 : 6) * block.x * block.y * sizeof(float);
    if (g) {
        if (eps) MARCH_LAUNCH((sweep_march_fwd_de_kernel<DIR, true, true>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S);
        else MARCH_LAUNCH((sweep_march_fwd_de_kernel<DIR, true, false>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S);
    } else {
        if (eps) MARCH_LAUNCH((sweep_march_fwd_de_kernel<DIR, false, true>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S);
        else MARCH_LAUNCH((sweep_march_fwd_de_kernel<DIR, false, false>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, S);
    }
    return DH_OK;
}

// y / z forward sweep of the dual-energy variant; pointers already permuted to (rho, m_n, m_t1, m_t2, eps, q)
int launch_sweep_march_de(dh_ctx* c, int d, const float* const in[6], const float* g, float* const out[6], float* cmax,
                          const SweepConst& sc) {
    const int N = c->N;
    const int S = march_segment(N, c->tune_march_s_fwd, 3);
    const dim3 block = march_block(N);
    const dim3 grid(N / block.x, N / block.y, (N + S - 1) / S);
    const bool eps = c->opt.lim_eps > 1e-18;
    Ptr6m pin; MPtr6m pout;
    for (int k = 0; k < 6; ++k) { pin.p[k] = in[k]; pout.p[k] = out[k]; }
    if (d == 1) DH_TRY(march_fwd_de_dispatch<1>(c, grid, block, pin, g, pout, cmax, sc, S, eps));
    else DH_TRY(march_fwd_de_dispatch<2>(c, grid, block, pin, g, pout, cmax, sc, S, eps));
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

template <int DIR, bool HAS_G>
static int march_adj_de_dispatch(dh_ctx* c, dim3 grid, dim3 block, const Ptr6m& pin, const float* g, const Ptr6m& pco,
                                 const MPtr6m& pci, float* gbar, double* scal, const SweepConst& sc, int S, int eps_mode) {
    const size_t sm = (size_t)RING * (HAS_G ? 13 : 12) * block.x * block.y * sizeof(float);
    if (eps_mode == 1) MARCH_LAUNCH((sweep_march_adj_de_kernel<DIR, HAS_G, 1>), grid, block, sm, c->stream, pin, g, pco, pci, gbar, scal, sc, S);
    else if (eps_mode == 2) MARCH_LAUNCH((sweep_march_adj_de_kernel<DIR, HAS_G, 2>), grid, block, sm, c->stream, pin, g, pco, pci, gbar, scal, sc, S);
    else MARCH_LAUNCH((sweep_march_adj_de_kernel<DIR, HAS_G, 0>), grid, block, sm, c->stream, pin, g, pco, pci, gbar, scal, sc, S);
    return DH_OK;
}

// y / z adjoint sweep of the dual-energy variant without the cotangents of Dtau and kappa; pointers already permuted
int launch_sweep_march_de_vjp(dh_ctx* c, int d, const float* const in[6], const float* g, const float* const cot_out[6],
                              float* const cot_in[6], float* gbar, double* scal, const SweepConst& sc) {
    const int N = c->N;
    const int S = march_segment(N, c->tune_march_s_adj, 4);
    const dim3 block = march_block(N);
    const dim3 grid(N / block.x, N / block.y, (N + S - 1) / S);
    const int eps = c->opt.lim_eps > 1e-18 ? 1 : (c->opt.lim_eps > 0.0 ? 2 : 0);
    Ptr6m pin, pco; MPtr6m pci;
    for (int k = 0; k < 6; ++k) { pin.p[k] = in[k]; pco.p[k] = cot_out[k]; pci.p[k] = cot_in[k]; }
    int rc;
    if (d == 1) rc = g ? march_adj_de_dispatch<1, true>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps)
                       : march_adj_de_dispatch<1, false>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps);
    else rc = g ? march_adj_de_dispatch<2, true>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps)
                : march_adj_de_dispatch<2, false>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps);
    DH_TRY(rc);
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_sweep_march_vjp(dh_ctx* c, int d, const Ptr5& pin, const float* g, const Ptr5& pco, const MPtr5& pci,
                           float* gbar, double* scal, const SweepConst& sc) {
    const int N = c->N;
    const int S = march_segment(N, c->tune_march_s_adj, 4);
    const dim3 block = march_block(N);
    const dim3 grid(N / block.x, N / block.y, (N + S - 1) / S);
    const int eps = c->opt.lim_eps > 1e-18 ? 1 : (c->opt.lim_eps > 0.0 ? 2 : 0);
    const bool lk = c->opt.want_dsched != 0;
    int rc;
    if (d == 1) rc = lk ? march_adj_dispatch<1, true>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps)
                        : march_adj_dispatch<1, false>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps);
    else rc = lk ? march_adj_dispatch<2, true>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps)
                 : march_adj_dispatch<2, false>(c, grid, block, pin, g, pco, pci, gbar, scal, sc, S, eps);
    DH_TRY(rc);
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

}  // namespace dh
