// sweep.cu -- dimensionally split relaxing-TVD sweep (forward and adjoint) for sm_100a.
//
// What one sweep computes (section 2.3.1-2.3.2, Eq. 9-18, :105-150; readings R3-R8, R11, R17 in DESIGN.md),
// on every periodic pencil along the sweep axis, with u = (rho, m_n, m_t1, m_t2, eps):
//   (G, H, c) = P(u):   v = m_n/rho, e = eps/rho - |m|^2/(2 rho^2), e+ = max(e, e_floor), p = (gamma-1) rho e+,
//                       c = |v| + sqrt(gamma (gamma-1) e+),  F = (m_n, m_n v + p, m_t1 v, m_t2 v, (eps+p) v),
//                       G = c u + F = 2 F^R,  H = c u - F = 2 F^L                          (Eq. 9-11, :117)
//   stage A (Eq. 12):   D_n = G_n - H_{n+1};  u*_n = u_n - (lam/4)(D_n - D_{n-1}) + (kap/2) S(u_n, g_n)
//   stage B (Eq. 13-18): Psi_n = G*_n + L(G*_n - G*_{n-1}, G*_{n+1} - G*_n) - H*_{n+1} + L(H*_{n+1} - H*_n, H*_{n+2} - H*_{n+1})
//                       u'_n = u_n - (lam/2)(Psi_n - Psi_{n-1}) + kap S(u*_n, g_n)
//   L(A,B) = AB/(A + B + sign(A) 4 eps) if AB > 0 else 0   (= 2 phi(A/4, B/4), phi the altered Van Leer limiter, Eq. 18)
//   S(u, g) = (0, rho g, 0, 0, m_n g)                      (gravity source S_g of Eq. 8, :101)
//   c_max = max c over the sweep's input                    (Eq. 19-20)
// Working with the doubled fluxes G, H removes every factor 1/2 of the paper's form from the inner loops.
//
// Kernel design ("chain" layout).  Each thread owns K consecutive cells ALONG the sweep axis in registers; the few
// flux vectors a neighbouring thread needs (2 per stage-A, 6 per stage-B) go through a slot-major shared-memory
// exchange buffer, so nothing is computed twice inside a block and shared-memory traffic is ~1/K of a
// cell-per-thread stencil.
//   x sweep : a block holds whole rows (N/K threads per row, float4/float2 loads), the periodic wrap happens inside
//             the block -- no halo, each array is read and written exactly once.
//   y,z sweeps: the marching kernels of sweep_march.cu (the chain layout with a recomputed halo is kept only by the
//             dual-energy variant, sweep_de.cu).
// The adjoint kernel recomputes stage A and B from the sweep's input and applies the transposed operations in
// gather form: each thread differentiates its own K interfaces and hands the contributions that cross its boundary
// to the neighbour through the same exchange buffer (4 exchanges in all).
#include "sweep_common.cuh"

namespace dh {

// ---------------------------------------------------------------------------------------------------------------
// Exchange buffer: slot-major, ex[slot * nthr + tid]; a thread publishes into its own column and reads the column of
// its left / right neighbour along the chain (wrapping inside the block).
struct Chain {
    float* ex;
    int nthr, tid, ltid, rtid;
};

template <int K, bool HAS_G>
__device__ __forceinline__ void sweep_forward_core(const float (&u)[K][5], const float (&g)[K], const Chain& ch,
                                                   const SweepConst& sc, float (&out)[K][5], float (&cin)[K]) {
    float G[K][5], H[K][5];
#pragma unroll
    for (int j = 0; j < K; ++j) prim_GH(u[j], sc, G[j], H[j], cin[j]);
    // ---- exchange A: H of my first cell (left neighbour needs H_{n+1}), G of my last cell (right neighbour needs G_{n-1})
    float* exA = ch.ex;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        exA[k * ch.nthr + ch.tid] = H[0][k];
        exA[(5 + k) * ch.nthr + ch.tid] = G[K - 1][k];
    }
    __syncthreads();
    float Gm1[5], HK[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        Gm1[k] = exA[(5 + k) * ch.nthr + ch.ltid];
        HK[k] = exA[k * ch.nthr + ch.rtid];
    }
    // ---- stage A and P(u*)
    float rs[K], ms[K];          // rho*, m_n* for the stage-B source
    float Gs[K][5], Hs[K][5];
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float us[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float Dn = G[j][k] - (j + 1 < K ? H[j + 1][k] : HK[k]);
            const float Dm = (j > 0 ? G[j - 1][k] : Gm1[k]) - H[j][k];
            us[k] = fmaf(-0.25f * sc.lam, Dn - Dm, u[j][k]);
        }
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g[j];
            us[1] = fmaf(hk, u[j][0], us[1]);
            us[4] = fmaf(hk, u[j][1], us[4]);
        }
        rs[j] = us[0];
        ms[j] = us[1];
        float cdummy;
        prim_GH(us, sc, Gs[j], Hs[j], cdummy);
    }
    // ---- exchange B: to the left neighbour G*_0, H*_0, H*_1 (its G*_K, H*_K, H*_{K+1});
    //                  to the right neighbour G*_{K-2}, G*_{K-1}, H*_{K-1} (its G*_{-2}, G*_{-1}, H*_{-1})
    float* exB = ch.ex + 10 * ch.nthr;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        exB[(0 + k) * ch.nthr + ch.tid] = Gs[0][k];
        exB[(5 + k) * ch.nthr + ch.tid] = Hs[0][k];
        exB[(10 + k) * ch.nthr + ch.tid] = Hs[1][k];
        exB[(15 + k) * ch.nthr + ch.tid] = Gs[K - 2][k];
        exB[(20 + k) * ch.nthr + ch.tid] = Gs[K - 1][k];
        exB[(25 + k) * ch.nthr + ch.tid] = Hs[K - 1][k];
    }
    __syncthreads();
    // ---- stage B, component by component (the limiter is component-wise)
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        float g_[K + 3], h_[K + 3];     // g_[i] = G*_{i-2} (i = 0..K+2), h_[i] = H*_{i-1} (i = 0..K+2)
        g_[0] = exB[(15 + k) * ch.nthr + ch.ltid];
        g_[1] = exB[(20 + k) * ch.nthr + ch.ltid];
        h_[0] = exB[(25 + k) * ch.nthr + ch.ltid];
#pragma unroll
        for (int j = 0; j < K; ++j) { g_[2 + j] = Gs[j][k]; h_[1 + j] = Hs[j][k]; }
        g_[K + 2] = exB[(0 + k) * ch.nthr + ch.rtid];
        h_[K + 1] = exB[(5 + k) * ch.nthr + ch.rtid];
        h_[K + 2] = exB[(10 + k) * ch.nthr + ch.rtid];
        // Psi at interfaces n = -1 .. K-1 (right face of cell n)
        float psi[K + 1];
#pragma unroll
        for (int i = 0; i <= K; ++i) {
            const int n = i - 1;
            // G*_n = g_[n+2], H*_{n+1} = h_[n+2]
            const float LR = limL(g_[n + 2] - g_[n + 1], g_[n + 3] - g_[n + 2], sc.eps4);
            const float LL = limL(h_[n + 2] - h_[n + 1], h_[n + 3] - h_[n + 2], sc.eps4);
            psi[i] = (g_[n + 2] + LR) - (h_[n + 2] - LL);
        }
#pragma unroll
        for (int j = 0; j < K; ++j) out[j][k] = fmaf(-0.5f * sc.lam, psi[j + 1] - psi[j], u[j][k]);
    }
    if (HAS_G) {
#pragma unroll
        for (int j = 0; j < K; ++j) {
            const float kg = sc.kap * g[j];
            out[j][1] = fmaf(kg, rs[j], out[j][1]);
            out[j][4] = fmaf(kg, ms[j], out[j][4]);
        }
    }
}

// Adjoint core.  In: u (sweep input), g, ob (cotangent of the sweep output).  Out: ub (cotangent of u), gb (of g) and
// per-thread partial sums of the scalar cotangents over the cells flagged in `count` (each global cell once).
// LK = false drops the cotangents of lam and kap (dh_options.want_dsched = 0) and with them the arrays only they need.
template <int K, bool HAS_G, bool LK = true>
__device__ __forceinline__ void sweep_adjoint_core(const float (&u)[K][5], const float (&g)[K], const float (&ob)[K][5],
                                                   const bool (&count)[K], const Chain& ch, const SweepConst& sc,
                                                   float (&ub)[K][5], float (&gb)[K], float& lam_b, float& kap_b,
                                                   float& gamma_b) {
    const int nt = ch.nthr;
    float dD[K][5];     // D_n - D_{n-1}
    float us[K][5];
    {
        float G[K][5], H[K][5];
#pragma unroll
        for (int j = 0; j < K; ++j) { float c_; prim_GH(u[j], sc, G[j], H[j], c_); }
        float* exA = ch.ex;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            exA[k * nt + ch.tid] = H[0][k];
            exA[(5 + k) * nt + ch.tid] = G[K - 1][k];
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float Gm1 = exA[(5 + k) * nt + ch.ltid];
            const float HK = exA[k * nt + ch.rtid];
#pragma unroll
            for (int j = 0; j < K; ++j) {
                const float Dn = G[j][k] - (j + 1 < K ? H[j + 1][k] : HK);
                const float Dm = (j > 0 ? G[j - 1][k] : Gm1) - H[j][k];
                const float dd = Dn - Dm;
                if (LK) dD[j][k] = dd;
                us[j][k] = fmaf(-0.25f * sc.lam, dd, u[j][k]);
            }
        }
        if (HAS_G) {
#pragma unroll
            for (int j = 0; j < K; ++j) {
                const float hk = 0.5f * sc.kap * g[j];
                us[j][1] = fmaf(hk, u[j][0], us[j][1]);
                us[j][4] = fmaf(hk, u[j][1], us[j][4]);
            }
        }
    }
    float GsB[K][5], HsB[K][5];      // cotangents of G*, H* of my cells
    float dpsi[K][5];                // Psi_j - Psi_{j-1}: only the lam_b sum needs it
    {
        float Gs[K][5], Hs[K][5];
#pragma unroll
        for (int j = 0; j < K; ++j) { float c_; prim_GH(us[j], sc, Gs[j], Hs[j], c_); }
        // ---- exchange B: to the left: G*_0, H*_0, H*_1, ob_0 (its G*_K, H*_K, H*_{K+1}, ob_K); to the right: G*_{K-1}
        float* exB = ch.ex + 25 * nt;     // region 2 (A and C live in region 1, B and D in region 2)
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            exB[(0 + k) * nt + ch.tid] = Gs[0][k];
            exB[(5 + k) * nt + ch.tid] = Hs[0][k];
            exB[(10 + k) * nt + ch.tid] = Hs[K > 1 ? 1 : 0][k];
            exB[(15 + k) * nt + ch.tid] = ob[0][k];
            exB[(20 + k) * nt + ch.tid] = Gs[K - 1][k];
        }
        __syncthreads();
        float* exC = ch.ex;                // region 1: every thread finished reading A before the B barrier
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            float g_[K + 2], h_[K + 2], o_[K + 1];   // g_[i] = G*_{i-1} (i=0..K+1); h_[i] = H*_i (i=0..K+1); o_[i] = ob_i
            g_[0] = exB[(20 + k) * nt + ch.ltid];
#pragma unroll
            for (int j = 0; j < K; ++j) { g_[1 + j] = Gs[j][k]; h_[j] = Hs[j][k]; o_[j] = ob[j][k]; }
            g_[K + 1] = exB[(0 + k) * nt + ch.rtid];
            h_[K] = exB[(5 + k) * nt + ch.rtid];
            h_[K + 1] = exB[(10 + k) * nt + ch.rtid];
            o_[K] = exB[(15 + k) * nt + ch.rtid];
            float gB[K + 2], hB[K + 2];              // same indexing as g_, h_
#pragma unroll
            for (int i = 0; i < K + 2; ++i) { gB[i] = 0.f; hB[i] = 0.f; }
            float psi[K];
#pragma unroll
            for (int j = 0; j < K; ++j) {            // my interface j = right face of my cell j
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
            // ---- exchange C: contributions that cross my boundary, and Psi of my last interface
            exC[(0 + k) * nt + ch.tid] = gB[0];          // -> left neighbour's G*_{K-1}
            exC[(5 + k) * nt + ch.tid] = gB[K + 1];      // -> right neighbour's G*_0
            exC[(10 + k) * nt + ch.tid] = hB[K];         // -> right neighbour's H*_0
            exC[(15 + k) * nt + ch.tid] = hB[K + 1];     // -> right neighbour's H*_1
            exC[(20 + k) * nt + ch.tid] = psi[K - 1];
#pragma unroll
            for (int j = 0; j < K; ++j) { GsB[j][k] = gB[j + 1]; HsB[j][k] = hB[j]; }
            if (LK) {
#pragma unroll
                for (int j = 1; j < K; ++j) dpsi[j][k] = psi[j] - psi[j - 1];
                dpsi[0][k] = psi[0];                      // Psi_{-1} subtracted after the exchange
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            GsB[K - 1][k] += exC[(0 + k) * nt + ch.rtid];
            GsB[0][k] += exC[(5 + k) * nt + ch.ltid];
            HsB[0][k] += exC[(10 + k) * nt + ch.ltid];
            if (K > 1) HsB[1][k] += exC[(15 + k) * nt + ch.ltid];
            if (LK) dpsi[0][k] -= exC[(20 + k) * nt + ch.ltid];
        }
        // K == 1: H*_1 of the left neighbour's view is the cell after me -- not supported (K >= 2 required)
    }
    // ---- cotangent of u*:  P^T, stage-B source, then stage A
    float usb[K][5];
    float gacc = 0.f, lacc = 0.f, kacc = 0.f;
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float gm_j = 0.f;
        prim_GH_vjp(us[j], sc, GsB[j], HsB[j], usb[j], gm_j);
        float l_j = 0.f;
        if (LK) {
#pragma unroll
            for (int k = 0; k < 5; ++k) l_j = fmaf(ob[j][k], dpsi[j][k], l_j);
            l_j *= -0.5f;
        }
        float k_j = 0.f;
        gb[j] = 0.f;
        if (HAS_G) {
            const float kg = sc.kap * g[j];
            usb[j][0] = fmaf(kg, ob[j][1], usb[j][0]);
            usb[j][1] = fmaf(kg, ob[j][4], usb[j][1]);
            const float t = us[j][0] * ob[j][1] + us[j][1] * ob[j][4];
            gb[j] = sc.kap * t;
            if (LK) k_j = g[j] * t;
        }
        if (count[j]) { gacc += gm_j; lacc += l_j; kacc += k_j; }
    }
    // ---- exchange D: u*_b of my first cell (left neighbour's usb_K) and of my last cell (right neighbour's usb_{-1})
    float* exD = ch.ex + 25 * nt;          // region 2: B was consumed before the C barrier
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        exD[k * nt + ch.tid] = usb[0][k];
        exD[(5 + k) * nt + ch.tid] = usb[K - 1][k];
    }
    __syncthreads();
    float usbK[5], usbM1[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        usbK[k] = exD[k * nt + ch.rtid];
        usbM1[k] = exD[(5 + k) * nt + ch.ltid];
    }
#pragma unroll
    for (int j = 0; j < K; ++j) {
        float Gb[5], Hb[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const float nxt = (j + 1 < K) ? usb[j + 1][k] : usbK[k];
            const float prv = (j > 0) ? usb[j - 1][k] : usbM1[k];
            Gb[k] = -0.25f * sc.lam * (usb[j][k] - nxt);        // D_b at my right face
            Hb[k] = 0.25f * sc.lam * (prv - usb[j][k]);         // -D_b at my left face
        }
        float gm_j = 0.f;
        prim_GH_vjp(u[j], sc, Gb, Hb, ub[j], gm_j);
        float l_j = 0.f;
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            ub[j][k] += ob[j][k] + usb[j][k];
            if (LK) l_j = fmaf(usb[j][k], dD[j][k], l_j);
        }
        l_j *= -0.25f;
        float k_j = 0.f;
        if (HAS_G) {
            const float hk = 0.5f * sc.kap * g[j];
            ub[j][0] = fmaf(hk, usb[j][1], ub[j][0]);
            ub[j][1] = fmaf(hk, usb[j][4], ub[j][1]);
            const float t = u[j][0] * usb[j][1] + u[j][1] * usb[j][4];
            gb[j] = fmaf(0.5f * sc.kap, t, gb[j]);
            if (LK) k_j = 0.5f * g[j] * t;
        }
        if (count[j]) { gacc += gm_j; lacc += l_j; kacc += k_j; }
    }
    lam_b = lacc; kap_b = kacc; gamma_b = gacc;
}

// ---------------------------------------------------------------------------------------------------------------
// vector load/store of K consecutive floats (K = 2 or 4), 8/16-byte aligned
template <int K> struct VecT;
template <> struct VecT<2> { using type = float2; };
template <> struct VecT<4> { using type = float4; };

template <int K>
__device__ __forceinline__ void load_vec(const float* p, float (&v)[K]) {
    typename VecT<K>::type t = __ldg(reinterpret_cast<const typename VecT<K>::type*>(p));
    const float* f = reinterpret_cast<const float*>(&t);
#pragma unroll
    for (int j = 0; j < K; ++j) v[j] = f[j];
}
template <int K>
__device__ __forceinline__ void store_vec(float* p, const float (&v)[K]) {
    typename VecT<K>::type t;
    float* f = reinterpret_cast<float*>(&t);
#pragma unroll
    for (int j = 0; j < K; ++j) f[j] = v[j];
    *reinterpret_cast<typename VecT<K>::type*>(p) = t;
}

// ------------------------------------------------------------------------------------------- x sweep kernels ----
// block = (N/K chain threads, R rows); grid.x = ceil(N^2 / R)
template <int K, bool HAS_G>
__global__ void __launch_bounds__(512) sweep_x_fwd_kernel(Ptr5 in, const float* __restrict__ gfield, MPtr5 outp,
                                                          float* cmax, SweepConst sc, long nrows,
                                                          float* __restrict__ delta_out) {
    extern __shared__ float smem[];
    __shared__ int s_max;
    const int Cx = blockDim.x, nthr = blockDim.x * blockDim.y;
    const int cx = threadIdx.x, r = threadIdx.y;
    if (cx == 0 && r == 0) s_max = 0;
    long row = (long)blockIdx.x * blockDim.y + r;
    const bool valid = row < nrows;
    if (!valid) row = nrows - 1;
    const long base = row * sc.N + (long)cx * K;
    float u[K][5], g[K], out[K][5], cin[K];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        float v[K];
        load_vec<K>(in.p[k] + base, v);
#pragma unroll
        for (int j = 0; j < K; ++j) u[j][k] = v[j];
    }
    if (HAS_G) load_vec<K>(gfield + base, g);
    else {
#pragma unroll
        for (int j = 0; j < K; ++j) g[j] = 0.f;
    }
    Chain ch{smem, nthr, r * Cx + cx, r * Cx + (cx == 0 ? Cx - 1 : cx - 1), r * Cx + (cx == Cx - 1 ? 0 : cx + 1)};
    sweep_forward_core<K, HAS_G>(u, g, ch, sc, out, cin);
    if (valid) {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            float v[K];
#pragma unroll
            for (int j = 0; j < K; ++j) v[j] = out[j][k];
            store_vec<K>(outp.p[k] + base, v);
        }
        if (delta_out) {                                   // next step's Poisson source: replaces source_init
            float v[K];
#pragma unroll
            for (int j = 0; j < K; ++j) v[j] = fmaf(sc.src_flag, out[j][0], -sc.src_rho_bar);
            store_vec<K>(delta_out + base, v);
        }
    }
    if (cmax) {
        float cm = cin[0];
#pragma unroll
        for (int j = 1; j < K; ++j) cm = (cin[j] > cm || cin[j] != cin[j]) ? cin[j] : cm;
        block_max_to_global(cm, cmax, &s_max);
    }
}

template <int K, bool HAS_G, bool LK>
__global__ void __launch_bounds__(512) sweep_x_adj_kernel(Ptr5 in, const float* __restrict__ gfield, Ptr5 cot_out,
                                                          MPtr5 cot_in, float* __restrict__ gbar, double* scal,
                                                          SweepConst sc, long nrows) {
    extern __shared__ float smem[];
    __shared__ float s_red[96];
    const int Cx = blockDim.x, nthr = blockDim.x * blockDim.y;
    const int cx = threadIdx.x, r = threadIdx.y;
    long row = (long)blockIdx.x * blockDim.y + r;
    const bool valid = row < nrows;
    if (!valid) row = nrows - 1;
    const long base = row * sc.N + (long)cx * K;
    float u[K][5], g[K], ob[K][5], ub[K][5], gb[K];
    bool count[K];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        float v[K], w[K];
        load_vec<K>(in.p[k] + base, v);
        load_vec<K>(cot_out.p[k] + base, w);
#pragma unroll
        for (int j = 0; j < K; ++j) { u[j][k] = v[j]; ob[j][k] = w[j]; }
    }
    if (HAS_G) load_vec<K>(gfield + base, g);
    else {
#pragma unroll
        for (int j = 0; j < K; ++j) g[j] = 0.f;
    }
#pragma unroll
    for (int j = 0; j < K; ++j) count[j] = valid;
    Chain ch{smem, nthr, r * Cx + cx, r * Cx + (cx == 0 ? Cx - 1 : cx - 1), r * Cx + (cx == Cx - 1 ? 0 : cx + 1)};
    float lb, kb, gmb;
    sweep_adjoint_core<K, HAS_G, LK>(u, g, ob, count, ch, sc, ub, gb, lb, kb, gmb);
    if (valid) {
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            float v[K];
#pragma unroll
            for (int j = 0; j < K; ++j) v[j] = ub[j][k];
            store_vec<K>(cot_in.p[k] + base, v);
        }
        if (HAS_G) store_vec<K>(gbar + base, gb);
    }
    block_sum3_to_global(lb, kb, gmb, scal, s_red);
}

// ------------------------------------------------------------------------------------------------ launchers ----
SweepConst make_sweep_const(const dh_ctx* c, float lam, float kap) {
    SweepConst sc;
    sc.lam = lam; sc.kap = kap;
    sc.gamma = (float)c->gamma;
    sc.gm1 = (float)(c->gamma - 1.0);
    sc.ggm1 = (float)(c->gamma * (c->gamma - 1.0));
    sc.e_floor = (float)c->opt.e_floor;
    sc.eps4 = (float)(4.0 * c->opt.lim_eps);
    sc.inv_lam = lam != 0.f ? 1.f / lam : 0.f;
    sc.N = c->N;
    sc.src_flag = c->opt.gas_sources_gravity ? 1.f : 0.f;
    sc.src_rho_bar = (float)c->rho_bar;
    sc.de_eta = (float)c->opt.dual_eta;
    return sc;
}

// pointer permutation: (rho, m_normal, m_t1, m_t2, eps) for sweep axis d; transverse in cyclic order
static void permute(int d, float* const* f, const float* out[5]) {
    out[0] = f[0]; out[1] = f[1 + d]; out[2] = f[1 + (d + 1) % 3]; out[3] = f[1 + (d + 2) % 3]; out[4] = f[4];
}

template <class Kern>
static cudaError_t allow_smem(Kern kern, size_t bytes) {
    return bytes > 48 * 1024 ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes)
                             : cudaSuccess;
}
#define DH_LAUNCH(kern, grid, block, sm, stream, ...)            \
    do {                                                         \
        DH_CUDA(allow_smem(kern, sm));                           \
        kern<<<grid, block, sm, stream>>>(__VA_ARGS__);          \
    } while (0)

constexpr int KF = 4;   // cells per thread, forward
constexpr int KA = 2;   // cells per thread, adjoint (register budget)
constexpr int FWD_SLOTS = 40, ADJ_SLOTS = 50;

template <int K>
static void x_geometry(int N, dim3& block, unsigned& grid, long nrows) {
    // N/K chain threads per row; as few rows per block as keep whole warps (the block reductions shuffle with a full
    // mask: Cx * R must be a multiple of 32).  Small blocks matter: every exchange is a block-wide barrier, and at
    // 256^3 blocks of 64 / 128 / 256 / 512 threads take 178 / 181 / 197 / 260 us forward (adjoint 501 / 533 / 617 from 128).
    constexpr int X_THREADS = 64;
    const int Cx = N / K;
    int g = Cx, b = 32;
    while (b) { int t = g % b; g = b; b = t; }      // g = gcd(Cx, 32)
    const int unit = 32 / g;
    int R = (X_THREADS / Cx) / unit * unit;
    if (R < unit) R = unit;
    block = dim3(Cx, R, 1);
    grid = (unsigned)((nrows + R - 1) / R);
}

int launch_sweep(dh_ctx* c, int d, float* const* in, const float* g, float lam, float kap, float* const* out,
                 float* cmax, float* delta_out) {
    if (c->nc == 6) {
        if (delta_out) { set_error("launch_sweep: source priming is not available with dual energy"); return DH_ERR_INVALID; }
        return launch_sweep_de(c, d, in, g, lam, kap, out, cmax);
    }
    const int N = c->N;
    Prof prof(c, PROF_SWEEP_X + d);
    SweepConst sc = make_sweep_const(c, lam, kap);
    Ptr5 pin; MPtr5 pout;
    const float* tmp[5];
    permute(d, in, tmp);
    for (int k = 0; k < 5; ++k) pin.p[k] = tmp[k];
    permute(d, out, tmp);
    for (int k = 0; k < 5; ++k) pout.p[k] = const_cast<float*>(tmp[k]);
    if (d == 0) {
        dim3 block; unsigned grid; long nrows = (long)N * N;
        x_geometry<KF>(N, block, grid, nrows);
        size_t sm = (size_t)FWD_SLOTS * block.x * block.y * sizeof(float);
        if (g) DH_LAUNCH((sweep_x_fwd_kernel<KF, true>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, nrows, delta_out);
        else DH_LAUNCH((sweep_x_fwd_kernel<KF, false>), grid, block, sm, c->stream, pin, g, pout, cmax, sc, nrows, delta_out);
    } else {
        DH_TRY(launch_sweep_march(c, d, pin, g, pout, cmax, sc, delta_out));
    }
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_sweep_vjp(dh_ctx* c, int d, float* const* in, const float* g, float lam, float kap,
                     float* const* cot_out, float* const* cot_in, float* g_bar, double* scal_bar) {
    if (c->nc == 6) return launch_sweep_de_vjp(c, d, in, g, lam, kap, cot_out, cot_in, g_bar, scal_bar);
    const int N = c->N;
    Prof prof(c, PROF_SWEEP_X_ADJ + d);
    SweepConst sc = make_sweep_const(c, lam, kap);
    Ptr5 pin, pco; MPtr5 pci;
    const float* tmp[5];
    permute(d, in, tmp);
    for (int k = 0; k < 5; ++k) pin.p[k] = tmp[k];
    permute(d, cot_out, tmp);
    for (int k = 0; k < 5; ++k) pco.p[k] = tmp[k];
    permute(d, cot_in, tmp);
    for (int k = 0; k < 5; ++k) pci.p[k] = const_cast<float*>(tmp[k]);
    if (d == 0) {
        dim3 block; unsigned grid; long nrows = (long)N * N;
        x_geometry<KA>(N, block, grid, nrows);
        size_t sm = (size_t)ADJ_SLOTS * block.x * block.y * sizeof(float);
        if (c->opt.want_dsched) {
            if (g) DH_LAUNCH((sweep_x_adj_kernel<KA, true, true>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc, nrows);
            else DH_LAUNCH((sweep_x_adj_kernel<KA, false, true>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc, nrows);
        } else {
            if (g) DH_LAUNCH((sweep_x_adj_kernel<KA, true, false>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc, nrows);
            else DH_LAUNCH((sweep_x_adj_kernel<KA, false, false>), grid, block, sm, c->stream, pin, g, pco, pci, g_bar, scal_bar, sc, nrows);
        }
    } else {
        DH_TRY(launch_sweep_march_vjp(c, d, pin, g, pco, pci, g_bar, scal_bar, sc));
    }
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

}  // namespace dh
