// sweep_de.cu -- the dual-energy variant of the relaxing-TVD sweep (forward and adjoint) for sm_100a.
//
// PAPER.md:85 ("can straightforwardly be expanded to a dual energy formalism, bringing more accurate solutions in
// low-density, high-velocity regions of the flow") and the internal-energy source S_e = (0, 0, -a p div U) the paper prints
// beside its flux vector; readings R33-R36 of DESIGN.md.  A sixth field q = a^2 rho_b e (internal energy
// density) is carried beside u = (rho, m_n, m_t1, m_t2, eps):
//   P(u, q):  e_T = eps/rho - |m|^2/(2 rho^2);  e = e_T if e_T > eta eps/rho else q/rho;  q_s = rho e;  e+ = max(e, e_floor);
//             p = (gamma-1) rho e+;  c = |v| + sqrt(gamma (gamma-1) e+);  F = (m_n, m_n v + p, m_t1 v, m_t2 v, (eps+p) v, q_s v)
//             G = c (u, q_s) + F,  H = c (u, q_s) - F                                   (six components)
//   stage A:  u*  as in sweep.cu;   q*_n = q_s,n - (lam/4)(D_n - D_{n-1})_q - (lam/4) p_n  (v_{n+1} - v_{n-1})
//   stage B:  u'  as in sweep.cu;   q'_n = q_s,n - (lam/2)(Psi_n - Psi_{n-1})_q - (lam/2) p*_n (v*_{n+1} - v*_{n-1})
// In fp32 e_T is the difference of two numbers 1/(thermal fraction) times larger: at Mach 600 (config 2 / 3 late in the
// run) its rounding error alone is 6e-8 x 2e5 = 1 % per operation; q does not have that cancellation.
//
// Kernel design: the "chain" layout of sweep.cu (each thread owns K = 2 consecutive cells along the sweep axis, neighbours
// exchange flux vectors through a slot-major shared-memory buffer) for all three axes -- the variant is an accuracy
// option, not the headline path, so it reuses one core for x (whole rows per block, float2 I/O) and y/z (32 lanes along x
// times C chain threads, halo recomputed).  The adjoint follows oracle-independent algebra: the transposed statements of
// the forward in gather form, with the extra cotangents of v and p that the source term hands to P^T.
#include "sweep_common.cuh"

namespace dh {

struct Ptr6 { const float* p[6]; };
struct MPtr6s { float* p[6]; };

struct ChainDE {
    float* ex;
    int nthr, tid, ltid, rtid;
};

constexpr int DE_FWD_SLOTS = 14 + 38;    // exchange A: H_0, G_{K-1}, v_0, v_{K-1};  B: 6 flux vectors + v*_0, v*_{K-1}
constexpr int DE_ADJ_SLOTS = 2 * 40;     // two regions of 40 slots, used alternately (A, C | B, D)

// ------------------------------------------------------------------------------------------------- forward core ----
template <int K, bool HAS_G>
__device__ __forceinline__ void de_forward_core(const float (&u)[K][6], const float (&g)[K], const ChainDE& ch,
                                                const SweepConst& sc, float (&out)[K][6], float (&cin)[K]) {
    const int nt = ch.nthr;
    float G[K][6], H[K][6], v[K], p[K], qs[K];
#pragma unroll
    for (int j = 0; j < K; ++j) prim_de(u[j], sc, G[j], H[j], cin[j], v[j], p[j], qs[j]);
    float* exA = ch.ex;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        exA[k * nt + ch.tid] = H[0][k];
        exA[(6 + k) * nt + ch.tid] = G[K - 1][k];
    }
    exA[12 * nt + ch.tid] = v[0];
    exA[13 * nt + ch.tid] = v[K - 1];
    __syncthreads();
    float Gm1[6], HK[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        Gm1[k] = exA[(6 + k) * nt + ch.ltid];
        HK[k] = exA[k * nt + ch.rtid];
    }
    const float vm1 = exA[13 * nt + ch.ltid], vK = exA[12 * nt + ch.rtid];
    float us[K][6], Gs[K][6], Hs[K][6], vs[K], ps[K];
#pragma unroll
    for (int j = 0; j < K; ++j) {
        const float U[6] = {u[j][0], u[j][1], u[j][2], u[j][3], u[j][4], qs[j]};
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float Dn = G[j][k] - (j + 1 < K ? H[j + 1][k] : HK[k]);
            const float Dm = (j > 0 ? G[j - 1][k] : Gm1[k]) - H[j][k];
            us[j][k] = fmaf(-0.25f * sc.lam, Dn - Dm, U[k]);
        }
        const float dv = (j + 1 < K ? v[j + 1] : vK) - (j > 0 ? v[j - 1] : vm1);
        us[j][5] = fmaf(-0.25f * sc.lam * p[j], dv, us[j][5]);
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g[j];
            us[j][1] = fmaf(hk, u[j][0], us[j][1]);
            us[j][4] = fmaf(hk, u[j][1], us[j][4]);
        }
        float cd, qd;
        prim_de(us[j], sc, Gs[j], Hs[j], cd, vs[j], ps[j], qd);
    }
    float* exB = ch.ex + 14 * nt;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        exB[(0 + k) * nt + ch.tid] = Gs[0][k];
        exB[(6 + k) * nt + ch.tid] = Hs[0][k];
        exB[(12 + k) * nt + ch.tid] = Hs[1][k];
        exB[(18 + k) * nt + ch.tid] = Gs[K - 2][k];
        exB[(24 + k) * nt + ch.tid] = Gs[K - 1][k];
        exB[(30 + k) * nt + ch.tid] = Hs[K - 1][k];
    }
    exB[36 * nt + ch.tid] = vs[0];
    exB[37 * nt + ch.tid] = vs[K - 1];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        float g_[K + 3], h_[K + 3];     // g_[i] = G*_{i-2}, h_[i] = H*_{i-1}
        g_[0] = exB[(18 + k) * nt + ch.ltid];
        g_[1] = exB[(24 + k) * nt + ch.ltid];
        h_[0] = exB[(30 + k) * nt + ch.ltid];
#pragma unroll
        for (int j = 0; j < K; ++j) { g_[2 + j] = Gs[j][k]; h_[1 + j] = Hs[j][k]; }
        g_[K + 2] = exB[(0 + k) * nt + ch.rtid];
        h_[K + 1] = exB[(6 + k) * nt + ch.rtid];
        h_[K + 2] = exB[(12 + k) * nt + ch.rtid];
        float psi[K + 1];
#pragma unroll
        for (int i = 0; i <= K; ++i) {
            const int n = i - 1;
            const float LR = limL(g_[n + 2] - g_[n + 1], g_[n + 3] - g_[n + 2], sc.eps4);
            const float LL = limL(h_[n + 2] - h_[n + 1], h_[n + 3] - h_[n + 2], sc.eps4);
            psi[i] = (g_[n + 2] + LR) - (h_[n + 2] - LL);
        }
#pragma unroll
        for (int j = 0; j < K; ++j) out[j][k] = fmaf(-0.5f * sc.lam, psi[j + 1] - psi[j], k < 5 ? u[j][k] : qs[j]);
    }
    const float vsm1 = exB[37 * nt + ch.ltid], vsK = exB[36 * nt + ch.rtid];
#pragma unroll
    for (int j = 0; j < K; ++j) {
        const float dv = (j + 1 < K ? vs[j + 1] : vsK) - (j > 0 ? vs[j - 1] : vsm1);
        out[j][5] = fmaf(-0.5f * sc.lam * ps[j], dv, out[j][5]);
        if (HAS_G) {
            const float kg = sc.kap * g[j];
            out[j][1] = fmaf(kg, us[j][0], out[j][1]);
            out[j][4] = fmaf(kg, us[j][1], out[j][4]);
        }
    }
}

// ------------------------------------------------------------------------------------------------- adjoint core ----
template <int K, bool HAS_G>
__device__ __forceinline__ void de_adjoint_core(const float (&u)[K][6], const float (&g)[K], const float (&ob)[K][6],
                                                const bool (&count)[K], const ChainDE& ch, const SweepConst& sc,
                                                float (&ub)[K][6], float (&gb)[K], float& lam_b, float& kap_b,
                                                float& gamma_b) {
    const int nt = ch.nthr;
    float* const R1 = ch.ex;              // exchanges A and C
    float* const R2 = ch.ex + 40 * nt;    // exchanges B and D
    float dD[K][6], us[K][6], v[K], p[K], qs[K], dvA[K];
    {
        float G[K][6], H[K][6];
#pragma unroll
        for (int j = 0; j < K; ++j) { float c_; prim_de(u[j], sc, G[j], H[j], c_, v[j], p[j], qs[j]); }
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            R1[k * nt + ch.tid] = H[0][k];
            R1[(6 + k) * nt + ch.tid] = G[K - 1][k];
        }
        R1[12 * nt + ch.tid] = v[0];
        R1[13 * nt + ch.tid] = v[K - 1];
        __syncthreads();
        const float vm1 = R1[13 * nt + ch.ltid], vK = R1[12 * nt + ch.rtid];
#pragma unroll
        for (int j = 0; j < K; ++j) {
            const float U[6] = {u[j][0], u[j][1], u[j][2], u[j][3], u[j][4], qs[j]};
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const float Gm1 = R1[(6 + k) * nt + ch.ltid];
                const float HK = R1[k * nt + ch.rtid];
                const float Dn = G[j][k] - (j + 1 < K ? H[j + 1][k] : HK);
                const float Dm = (j > 0 ? G[j - 1][k] : Gm1) - H[j][k];
                dD[j][k] = Dn - Dm;
                us[j][k] = fmaf(-0.25f * sc.lam, dD[j][k], U[k]);
            }
            dvA[j] = (j + 1 < K ? v[j + 1] : vK) - (j > 0 ? v[j - 1] : vm1);
            us[j][5] = fmaf(-0.25f * sc.lam * p[j], dvA[j], us[j][5]);
            if (HAS_G) {
                const float hk = 0.5f * sc.kap * g[j];
                us[j][1] = fmaf(hk, u[j][0], us[j][1]);
                us[j][4] = fmaf(hk, u[j][1], us[j][4]);
            }
        }
    }
    float GsB[K][6], HsB[K][6], dpsi[K][6], vs[K], ps[K], dvB[K];
    {
        float Gs[K][6], Hs[K][6];
#pragma unroll
        for (int j = 0; j < K; ++j) { float c_, q_; prim_de(us[j], sc, Gs[j], Hs[j], c_, vs[j], ps[j], q_); }
        // exchange B: to the left: G*_0, H*_0, H*_1, ob_0, v*_0; to the right: G*_{K-1}, v*_{K-1}
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            R2[(0 + k) * nt + ch.tid] = Gs[0][k];
            R2[(6 + k) * nt + ch.tid] = Hs[0][k];
            R2[(12 + k) * nt + ch.tid] = Hs[1][k];
            R2[(18 + k) * nt + ch.tid] = ob[0][k];
            R2[(24 + k) * nt + ch.tid] = Gs[K - 1][k];
        }
        R2[30 * nt + ch.tid] = vs[0];
        R2[31 * nt + ch.tid] = vs[K - 1];
        __syncthreads();
        const float vsm1 = R2[31 * nt + ch.ltid], vsK = R2[30 * nt + ch.rtid];
#pragma unroll
        for (int j = 0; j < K; ++j) dvB[j] = (j + 1 < K ? vs[j + 1] : vsK) - (j > 0 ? vs[j - 1] : vsm1);
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            float g_[K + 2], h_[K + 2], o_[K + 1];   // g_[i] = G*_{i-1}; h_[i] = H*_i; o_[i] = ob_i
            g_[0] = R2[(24 + k) * nt + ch.ltid];
#pragma unroll
            for (int j = 0; j < K; ++j) { g_[1 + j] = Gs[j][k]; h_[j] = Hs[j][k]; o_[j] = ob[j][k]; }
            g_[K + 1] = R2[(0 + k) * nt + ch.rtid];
            h_[K] = R2[(6 + k) * nt + ch.rtid];
            h_[K + 1] = R2[(12 + k) * nt + ch.rtid];
            o_[K] = R2[(18 + k) * nt + ch.rtid];
            float gB[K + 2], hB[K + 2];
#pragma unroll
            for (int i = 0; i < K + 2; ++i) { gB[i] = 0.f; hB[i] = 0.f; }
            float psi[K];
#pragma unroll
            for (int j = 0; j < K; ++j) {
                const float psib = -0.5f * sc.lam * (o_[j] - o_[j + 1]);
                float LA, LB;
                const float LR = limL_grad(g_[j + 1] - g_[j], g_[j + 2] - g_[j + 1], sc.eps4, LA, LB);
                gB[j + 1] = fmaf(psib, 1.f + LA - LB, gB[j + 1]);
                gB[j] = fmaf(-LA, psib, gB[j]);
                gB[j + 2] = fmaf(LB, psib, gB[j + 2]);
                float MA, MB;
                const float LL = limL_grad(h_[j + 1] - h_[j], h_[j + 2] - h_[j + 1], sc.eps4, MA, MB);
                hB[j + 1] = fmaf(psib, -1.f + MA - MB, hB[j + 1]);
                hB[j] = fmaf(-MA, psib, hB[j]);
                hB[j + 2] = fmaf(MB, psib, hB[j + 2]);
                psi[j] = (g_[j + 1] + LR) - (h_[j + 1] - LL);
            }
            // exchange C (region 1: every thread finished reading A before the B barrier)
            R1[(0 + k) * nt + ch.tid] = gB[0];
            R1[(6 + k) * nt + ch.tid] = gB[K + 1];
            R1[(12 + k) * nt + ch.tid] = hB[K];
            R1[(18 + k) * nt + ch.tid] = hB[K + 1];
            R1[(24 + k) * nt + ch.tid] = psi[K - 1];
#pragma unroll
            for (int j = 0; j < K; ++j) { GsB[j][k] = gB[j + 1]; HsB[j][k] = hB[j]; }
#pragma unroll
            for (int j = 1; j < K; ++j) dpsi[j][k] = psi[j] - psi[j - 1];
            dpsi[0][k] = psi[0];
        }
        // the source of stage B hands t = p* q'_b to the velocity cotangents of the neighbouring cells
        R1[30 * nt + ch.tid] = ps[0] * ob[0][5];
        R1[31 * nt + ch.tid] = ps[K - 1] * ob[K - 1][5];
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            GsB[K - 1][k] += R1[(0 + k) * nt + ch.rtid];
            GsB[0][k] += R1[(6 + k) * nt + ch.ltid];
            HsB[0][k] += R1[(12 + k) * nt + ch.ltid];
            HsB[1][k] += R1[(18 + k) * nt + ch.ltid];
            dpsi[0][k] -= R1[(24 + k) * nt + ch.ltid];
        }
    }
    const float tBm1 = R1[31 * nt + ch.ltid], tBK = R1[30 * nt + ch.rtid];
    // ---- cotangent of (u*, q*): P^T with the source's extra cotangents, stage-B gravity source
    float usb[K][6];
    float gacc = 0.f, lacc = 0.f, kacc = 0.f;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        const float tm = j > 0 ? ps[j - 1] * ob[j - 1][5] : tBm1;
        const float tp = j + 1 < K ? ps[j + 1] * ob[j + 1][5] : tBK;
        const float vsb = -0.5f * sc.lam * (tm - tp);
        const float psb = -0.5f * sc.lam * ob[j][5] * dvB[j];
        float gm_j = 0.f;
        prim_de_vjp(us[j], sc, GsB[j], HsB[j], vsb, psb, 0.f, usb[j], gm_j);
        float l_j = 0.f;
#pragma unroll
        for (int k = 0; k < 6; ++k) l_j = fmaf(ob[j][k], dpsi[j][k], l_j);
        l_j = -0.5f * fmaf(ob[j][5] * ps[j], dvB[j], l_j);
        float k_j = 0.f;
        gb[j] = 0.f;
        if (HAS_G) {
            const float kg = sc.kap * g[j];
            usb[j][0] = fmaf(kg, ob[j][1], usb[j][0]);
            usb[j][1] = fmaf(kg, ob[j][4], usb[j][1]);
            const float t = us[j][0] * ob[j][1] + us[j][1] * ob[j][4];
            gb[j] = sc.kap * t;
            k_j = g[j] * t;
        }
        if (count[j]) { gacc += gm_j; lacc += l_j; kacc += k_j; }
    }
    // ---- exchange D (region 2): (u*, q*)_b of my first and last cell, and tA = p q*_b of both
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        R2[k * nt + ch.tid] = usb[0][k];
        R2[(6 + k) * nt + ch.tid] = usb[K - 1][k];
    }
    R2[12 * nt + ch.tid] = p[0] * usb[0][5];
    R2[13 * nt + ch.tid] = p[K - 1] * usb[K - 1][5];
    __syncthreads();
    float usbK[6], usbM1[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        usbK[k] = R2[k * nt + ch.rtid];
        usbM1[k] = R2[(6 + k) * nt + ch.ltid];
    }
    const float tAm1 = R2[13 * nt + ch.ltid], tAK = R2[12 * nt + ch.rtid];
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float Gb[6], Hb[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            const float nxt = (j + 1 < K) ? usb[j + 1][k] : usbK[k];
            const float prv = (j > 0) ? usb[j - 1][k] : usbM1[k];
            Gb[k] = -0.25f * sc.lam * (usb[j][k] - nxt);
            Hb[k] = 0.25f * sc.lam * (prv - usb[j][k]);
        }
        const float tm = j > 0 ? p[j - 1] * usb[j - 1][5] : tAm1;
        const float tp = j + 1 < K ? p[j + 1] * usb[j + 1][5] : tAK;
        const float vb = -0.25f * sc.lam * (tm - tp);
        const float pb = -0.25f * sc.lam * usb[j][5] * dvA[j];
        const float qsb = ob[j][5] + usb[j][5];          // both stages start from q_s
        float gm_j = 0.f;
        prim_de_vjp(u[j], sc, Gb, Hb, vb, pb, qsb, ub[j], gm_j);
        float l_j = 0.f;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            ub[j][k] += ob[j][k] + usb[j][k];
            l_j = fmaf(usb[j][k], dD[j][k], l_j);
        }
        l_j = fmaf(usb[j][5], dD[j][5], l_j);
        l_j = -0.25f * fmaf(usb[j][5] * p[j], dvA[j], l_j);
        float k_j = 0.f;
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g[j];
            ub[j][0] = fmaf(hk, usb[j][1], ub[j][0]);
            ub[j][1] = fmaf(hk, usb[j][4], ub[j][1]);
            const float t = u[j][0] * usb[j][1] + u[j][1] * usb[j][4];
            gb[j] = fmaf(0.5f * sc.kap, t, gb[j]);
            k_j = 0.5f * g[j] * t;
        }
        if (count[j]) { gacc += gm_j; lacc += l_j; kacc += k_j; }
    }
    lam_b = lacc; kap_b = kacc; gamma_b = gacc;
}

// ------------------------------------------------------------------------------------------------------ kernels ----
constexpr int KD = 2;     // cells per thread (float2 I/O in the x sweep)

__device__ __forceinline__ void ld2(const float* p, float& a, float& b) {
    const float2 t = __ldg(reinterpret_cast<const float2*>(p));
    a = t.x; b = t.y;
}

// K consecutive floats (K = 2 or 4) of one row as one 8 / 16-byte access
template <int K>
__device__ __forceinline__ void ldK(const float* p, float (&v)[K]) {
    if (K == 4) {
        const float4 t = __ldg(reinterpret_cast<const float4*>(p));
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[K - 1] = t.w;
    } else {
        ld2(p, v[0], v[1]);
    }
}
template <int K>
__device__ __forceinline__ void stK(float* p, const float (&v)[K]) {
    if (K == 4) *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[K - 1]);
    else *reinterpret_cast<float2*>(p) = make_float2(v[0], v[1]);
}

// x sweep: block = (N/K chain threads, R rows); grid.x = ceil(N^2 / R).  Forward K = 4 (64 - 77 registers at K = 2 leave the
// room; the exchanges and barriers are per thread, so twice the cells per thread halve them), adjoint K = KD = 2.
constexpr int KDF = 4;
template <bool HAS_G, int K>
__global__ void __launch_bounds__(512) sweep_de_x_fwd_kernel(Ptr6 in, const float* __restrict__ gfield, MPtr6s outp,
                                                             float* cmax, SweepConst sc, long nrows) {
    extern __shared__ float smem[];
    __shared__ int s_max;
    const int Cx = blockDim.x, nthr = blockDim.x * blockDim.y;
    const int cx = threadIdx.x, r = threadIdx.y;
    if (cx == 0 && r == 0) s_max = 0;
    long row = (long)blockIdx.x * blockDim.y + r;
    const bool valid = row < nrows;
    if (!valid) row = nrows - 1;
    const long base = row * sc.N + (long)cx * K;
    float u[K][6], g[K], out[K][6], cin[K];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        float v[K];
        ldK<K>(in.p[k] + base, v);
#pragma unroll
        for (int j = 0; j < K; ++j) u[j][k] = v[j];
    }
    if (HAS_G) ldK<K>(gfield + base, g);
    else {
#pragma unroll
        for (int j = 0; j < K; ++j) g[j] = 0.f;
    }
    ChainDE ch{smem, nthr, r * Cx + cx, r * Cx + (cx == 0 ? Cx - 1 : cx - 1), r * Cx + (cx == Cx - 1 ? 0 : cx + 1)};
    de_forward_core<K, HAS_G>(u, g, ch, sc, out, cin);
    if (valid) {
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            float v[K];
#pragma unroll
            for (int j = 0; j < K; ++j) v[j] = out[j][k];
            stK<K>(outp.p[k] + base, v);
        }
    }
    if (cmax) {
        float cm = cin[0];
#pragma unroll
        for (int j = 1; j < K; ++j) cm = (cin[j] > cm || cin[j] != cin[j]) ? cin[j] : cm;
        block_max_to_global(cm, cmax, &s_max);
    }
}

template <bool HAS_G>
__global__ void __launch_bounds__(512) sweep_de_x_adj_kernel(Ptr6 in, const float* __restrict__ gfield, Ptr6 cot_out,
                                                             MPtr6s cot_in, float* __restrict__ gbar, double* scal,
                                                             SweepConst sc, long nrows) {
    extern __shared__ float smem[];
    __shared__ float s_red[96];
    const int Cx = blockDim.x, nthr = blockDim.x * blockDim.y;
    const int cx = threadIdx.x, r = threadIdx.y;
    long row = (long)blockIdx.x * blockDim.y + r;
    const bool valid = row < nrows;
    if (!valid) row = nrows - 1;
    const long base = row * sc.N + (long)cx * KD;
    float u[KD][6], g[KD] = {0.f, 0.f}, ob[KD][6], ub[KD][6], gb[KD];
    const bool count[KD] = {valid, valid};
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        ld2(in.p[k] + base, u[0][k], u[1][k]);
        ld2(cot_out.p[k] + base, ob[0][k], ob[1][k]);
    }
    if (HAS_G) ld2(gfield + base, g[0], g[1]);
    ChainDE ch{smem, nthr, r * Cx + cx, r * Cx + (cx == 0 ? Cx - 1 : cx - 1), r * Cx + (cx == Cx - 1 ? 0 : cx + 1)};
    float lb, kb, gmb;
    de_adjoint_core<KD, HAS_G>(u, g, ob, count, ch, sc, ub, gb, lb, kb, gmb);
    if (valid) {
#pragma unroll
        for (int k = 0; k < 6; ++k) *reinterpret_cast<float2*>(cot_in.p[k] + base) = make_float2(ub[0][k], ub[1][k]);
        if (HAS_G) *reinterpret_cast<float2*>(gbar + base) = make_float2(gb[0], gb[1]);
    }
    block_sum3_to_global(lb, kb, gmb, scal, s_red);
}

// y/z sweeps: block = (32 lanes along x, C chain threads along the sweep axis); grid = (tiles, N/32, N).
// A tile covers C*KD cells starting HALO cells before its first output cell.
template <bool HAS_G, int DIR>
__global__ void __launch_bounds__(512) sweep_de_yz_fwd_kernel(Ptr6 in, const float* __restrict__ gfield, MPtr6s outp,
                                                              float* cmax, SweepConst sc) {
    constexpr int HALO = 3;
    extern __shared__ float smem[];
    __shared__ int s_max;
    const int C = blockDim.y, nthr = 32 * C;
    const int lane = threadIdx.x, c = threadIdx.y;
    if (lane == 0 && c == 0) s_max = 0;
    const int N = sc.N;
    const int S = C * KD - 2 * HALO;
    const int x = blockIdx.y * 32 + lane;
    const int o = blockIdx.z;
    const int q0 = blockIdx.x * S - HALO + c * KD;
    float u[KD][6], g[KD], out[KD][6], cin[KD];
    long addr[KD];
#pragma unroll
    for (int j = 0; j < KD; ++j) {
        int p = q0 + j;
        p = p < 0 ? p + N : (p >= N ? p - N : p);
        p = p >= N ? p - N : p;
        addr[j] = (DIR == 1) ? ((long)o * N + p) * N + x : ((long)p * N + o) * N + x;
#pragma unroll
        for (int k = 0; k < 6; ++k) u[j][k] = __ldg(in.p[k] + addr[j]);
        g[j] = HAS_G ? __ldg(gfield + addr[j]) : 0.f;
    }
    ChainDE ch{smem, nthr, c * 32 + lane, (c == 0 ? C - 1 : c - 1) * 32 + lane, (c == C - 1 ? 0 : c + 1) * 32 + lane};
    de_forward_core<KD, HAS_G>(u, g, ch, sc, out, cin);
    float cm = 0.f;
#pragma unroll
    for (int j = 0; j < KD; ++j) {
        const int li = c * KD + j;
        const bool ok = li >= HALO && li < HALO + S && (q0 + j) < N;
        if (ok) {
#pragma unroll
            for (int k = 0; k < 6; ++k) outp.p[k][addr[j]] = out[j][k];
            cm = (cin[j] > cm || cin[j] != cin[j]) ? cin[j] : cm;
        }
    }
    if (cmax) block_max_to_global(cm, cmax, &s_max);
}

template <bool HAS_G, int DIR>
__global__ void __launch_bounds__(512) sweep_de_yz_adj_kernel(Ptr6 in, const float* __restrict__ gfield, Ptr6 cot_out,
                                                              MPtr6s cot_in, float* __restrict__ gbar, double* scal,
                                                              SweepConst sc) {
    constexpr int HALO = 4;
    extern __shared__ float smem[];
    __shared__ float s_red[96];
    const int C = blockDim.y, nthr = 32 * C;
    const int lane = threadIdx.x, c = threadIdx.y;
    const int N = sc.N;
    const int S = C * KD - 2 * HALO;
    const int x = blockIdx.y * 32 + lane;
    const int o = blockIdx.z;
    const int q0 = blockIdx.x * S - HALO + c * KD;
    float u[KD][6], g[KD], ob[KD][6], ub[KD][6], gb[KD];
    bool count[KD];
    long addr[KD];
#pragma unroll
    for (int j = 0; j < KD; ++j) {
        int p = q0 + j;
        p = p < 0 ? p + N : (p >= N ? p - N : p);
        p = p >= N ? p - N : p;
        addr[j] = (DIR == 1) ? ((long)o * N + p) * N + x : ((long)p * N + o) * N + x;
#pragma unroll
        for (int k = 0; k < 6; ++k) { u[j][k] = __ldg(in.p[k] + addr[j]); ob[j][k] = __ldg(cot_out.p[k] + addr[j]); }
        g[j] = HAS_G ? __ldg(gfield + addr[j]) : 0.f;
        const int li = c * KD + j;
        count[j] = li >= HALO && li < HALO + S && (q0 + j) < N;
    }
    ChainDE ch{smem, nthr, c * 32 + lane, (c == 0 ? C - 1 : c - 1) * 32 + lane, (c == C - 1 ? 0 : c + 1) * 32 + lane};
    float lb, kb, gmb;
    de_adjoint_core<KD, HAS_G>(u, g, ob, count, ch, sc, ub, gb, lb, kb, gmb);
#pragma unroll
    for (int j = 0; j < KD; ++j) {
        if (count[j]) {
#pragma unroll
            for (int k = 0; k < 6; ++k) cot_in.p[k][addr[j]] = ub[j][k];
            if (HAS_G) gbar[addr[j]] = gb[j];
        }
    }
    block_sum3_to_global(lb, kb, gmb, scal, s_red);
}

// ---------------------------------------------------------------------------------------------------- launchers ----
#define DE_LAUNCH(kern, grid, block, sm, stream, ...)                                                           \
    do {                                                                                                        \
        if ((sm) > 48 * 1024)                                                                                   \
            DH_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sm)));        \
        kern<<<grid, block, sm, stream>>>(__VA_ARGS__);                                                         \
    } while (0)

// (rho, m_normal, m_t1, m_t2, eps, q) for sweep axis d
static void permute6(int d, float* const f[6], const float* out[6]) {
    out[0] = f[0]; out[1] = f[1 + d]; out[2] = f[1 + (d + 1) % 3]; out[3] = f[1 + (d + 2) % 3]; out[4] = f[4]; out[5] = f[5];
}

static void de_x_geometry(int N, int K, dim3& block, unsigned& grid, long nrows) {
    // N/K chain threads per row, rows per block so that blocks are whole warps of about 64 threads (see sweep.cu)
    const int Cx = N / K;
    int g = Cx, b = 32;
    while (b) { int t = g % b; g = b; b = t; }
    const int unit = 32 / g;
    int R = (64 / Cx) / unit * unit;
    if (R < unit) R = unit;
    block = dim3(Cx, R, 1);
    grid = (unsigned)((nrows + R - 1) / R);
}

static int de_yz_chain_threads(int N, int halo) {
    int best = 8; double best_cost = 1e30;
    for (int C = 6; C <= 16; ++C) {
        const int S = C * KD - 2 * halo;
        if (S <= 0 || C * KD > N + 2 * halo) continue;
        const int T = (N + S - 1) / S;
        const double cost = (double)T * C * KD / N;
        if (cost < best_cost - 1e-9) { best_cost = cost; best = C; }
    }
    return best;
}

int launch_sweep_de(dh_ctx* c, int d, float* const in[6], const float* g, float lam, float kap, float* const out[6],
                    float* cmax) {
    const int N = c->N;
    Prof prof(c, PROF_SWEEP_X + d);
    SweepConst sc = make_sweep_const(c, lam, kap);
    Ptr6 pin; MPtr6s pout;
    const float* tmp[6];
    permute6(d, in, tmp);
    for (int k = 0; k < 6; ++k) pin.p[k] = tmp[k];
    permute6(d, out, tmp);
    for (int k = 0; k < 6; ++k) pout.p[k] = const_cast<float*>(tmp[k]);
    if (d == 0) {
        dim3 block; unsigned grid; const long nrows = (long)N * N;
        de_x_geometry(N, KDF, block, grid, nrows);
        const size_t sm = (size_t)DE_FWD_SLOTS * block.x * block.y * sizeof(float);
        if (g) DE_LAUNCH((sweep_de_x_fwd_kernel<true, KDF>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, nrows);
        else DE_LAUNCH((sweep_de_x_fwd_kernel<false, KDF>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, nrows);
    } else if (c->tune_de_march) {
        // y / z forward: the marching pipeline with the sixth component (sweep_march.cu), 3.2 x faster than the chain tile
        float* outm[6];
        for (int k = 0; k < 6; ++k) outm[k] = pout.p[k];
        DH_TRY(launch_sweep_march_de(c, d, pin.p, g, outm, cmax, sc));
    } else {
        const int C = de_yz_chain_threads(N, 3);
        const int S = C * KD - 6;
        const dim3 block(32, C, 1), grid((N + S - 1) / S, N / 32, N);
        const size_t sm = (size_t)DE_FWD_SLOTS * 32 * C * sizeof(float);
        if (d == 1) {
            if (g) DE_LAUNCH((sweep_de_yz_fwd_kernel<true, 1>), grid, block, sm, c->stream, pin, g, pout, cmax, sc);
            else DE_LAUNCH((sweep_de_yz_fwd_kernel<false, 1>), grid, block, sm, c->stream, pin, g, pout, cmax, sc);
        } else {
            if (g) DE_LAUNCH((sweep_de_yz_fwd_kernel<true, 2>), grid, block, sm, c->stream, pin, g, pout, cmax, sc);
            else DE_LAUNCH((sweep_de_yz_fwd_kernel<false, 2>), grid, block, sm, c->stream, pin, g, pout, cmax, sc);
        }
    }
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_sweep_de_vjp(dh_ctx* c, int d, float* const in[6], const float* g, float lam, float kap,
                        float* const cot_out[6], float* const cot_in[6], float* g_bar, double* scal_bar) {
    const int N = c->N;
    Prof prof(c, PROF_SWEEP_X_ADJ + d);
    SweepConst sc = make_sweep_const(c, lam, kap);
    Ptr6 pin, pco; MPtr6s pci;
    const float* tmp[6];
    permute6(d, in, tmp);
    for (int k = 0; k < 6; ++k) pin.p[k] = tmp[k];
    permute6(d, cot_out, tmp);
    for (int k = 0; k < 6; ++k) pco.p[k] = tmp[k];
    permute6(d, cot_in, tmp);
    for (int k = 0; k < 6; ++k) pci.p[k] = const_cast<float*>(tmp[k]);
    if (d == 0) {
        dim3 block; unsigned grid; const long nrows = (long)N * N;
        de_x_geometry(N, KD, block, grid, nrows);
        const size_t sm = (size_t)DE_ADJ_SLOTS * block.x * block.y * sizeof(float);
        if (g) DE_LAUNCH((sweep_de_x_adj_kernel<true>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc, nrows);
        else DE_LAUNCH((sweep_de_x_adj_kernel<false>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc, nrows);
    } else if (c->tune_de_march && !c->opt.want_dsched) {
        // y / z adjoint without the cotangents of Dtau and kappa: the marching pipeline with the sixth component
        float* cim[6];
        for (int k = 0; k < 6; ++k) cim[k] = pci.p[k];
        DH_TRY(launch_sweep_march_de_vjp(c, d, pin.p, g, pco.p, cim, g_bar, scal_bar, sc));
    } else {
        const int C = de_yz_chain_threads(N, 4);
        const int S = C * KD - 8;
        const dim3 block(32, C, 1), grid((N + S - 1) / S, N / 32, N);
        const size_t sm = (size_t)DE_ADJ_SLOTS * 32 * C * sizeof(float);
        if (d == 1) {
            if (g) DE_LAUNCH((sweep_de_yz_adj_kernel<true, 1>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc);
            else DE_LAUNCH((sweep_de_yz_adj_kernel<false, 1>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc);
        } else {
            if (g) DE_LAUNCH((sweep_de_yz_adj_kernel<true, 2>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc);
            else DE_LAUNCH((sweep_de_yz_adj_kernel<false, 2>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc);
        }
    }
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

}  // namespace dh
