// sweep_common.cuh -- device functions shared by the sweep kernels (sweep.cu: x chain kernels; sweep_march.cu: y/z
// marching kernels): the flux split P(u), its transpose, the limiter, block reductions.  Product code: shares nothing
// with oracle/.
#pragma once
#include "dh_internal.cuh"

namespace dh {

struct SweepConst {
    float lam, kap;
    float gm1;       // gamma - 1
    float ggm1;      // gamma (gamma - 1)
    float gamma;
    float e_floor;
    float eps4;      // 4 * lim_eps
    float inv_lam;   // 1 / lam (0 when lam == 0): the marching adjoint forms lam_b from u* - u
    float src_flag, src_rho_bar;   // next step's Poisson source from this sweep's density: delta = src_flag rho' - src_rho_bar
    float de_eta;    // dual-energy variant (sweep_de.cu): thermal fraction below which q replaces eps - |m|^2/(2 rho)
    int N;
};

__device__ __forceinline__ float rcp_fast(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_fast(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// (G, H, c) = P(u)
__device__ __forceinline__ void prim_GH(const float (&u)[5], const SweepConst& sc, float (&G)[5], float (&H)[5], float& c) {
    const float rinv = rcp_fast(u[0]);
    const float v = u[1] * rinv;
    const float ke = 0.5f * (u[1] * u[1] + u[2] * u[2] + u[3] * u[3]) * rinv;
    const float e = (u[4] - ke) * rinv;
    const float ep = !(e <= sc.e_floor) ? e : sc.e_floor;   // NaN passes through to the CFL check
    const float p = sc.gm1 * u[0] * ep;
    const float cs = sqrt_fast(sc.ggm1 * ep);
    c = fabsf(v) + cs;
    float F[5];
    F[0] = u[1];
    F[1] = fmaf(u[1], v, p);
    F[2] = u[2] * v;
    F[3] = u[3] * v;
    F[4] = (u[4] + p) * v;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        G[k] = fmaf(c, u[k], F[k]);
        H[k] = fmaf(c, u[k], -F[k]);
    }
}

// Transpose of P at u: given cotangents Gb, Hb returns the cotangent of u and adds to gamma_b.
__device__ __forceinline__ void prim_GH_vjp(const float (&u)[5], const SweepConst& sc, const float (&Gb)[5],
                                            const float (&Hb)[5], float (&ub)[5], float& gamma_b) {
    const float rinv = rcp_fast(u[0]);
    const float v = u[1] * rinv;
    const float m2 = u[1] * u[1] + u[2] * u[2] + u[3] * u[3];
    const float ke = 0.5f * m2 * rinv;
    const float e = (u[4] - ke) * rinv;
    const bool active = !(e <= sc.e_floor);
    const float ep = active ? e : sc.e_floor;
    const float p = sc.gm1 * u[0] * ep;
    const float cs = sqrt_fast(sc.ggm1 * ep);
    const float c = fabsf(v) + cs;
    float cub[5], Fb[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) { cub[k] = Gb[k] + Hb[k]; Fb[k] = Gb[k] - Hb[k]; }
    float cb = 0.f;
#pragma unroll
    for (int k = 0; k < 5; ++k) { cb = fmaf(cub[k], u[k], cb); ub[k] = c * cub[k]; }
    // F = (m_n, m_n v + p, m_t1 v, m_t2 v, (eps + p) v)
    float mnb = fmaf(Fb[1], v, Fb[0]);
    float vb = Fb[1] * u[1] + Fb[2] * u[2] + Fb[3] * u[3] + Fb[4] * (u[4] + p);
    const float pb = fmaf(Fb[4], v, Fb[1]);
    float epsb = Fb[4] * v;
    // c = |v| + cs   (d|v|/dv = sign(v), sign(0) = 0: R26)
    const float sgn = (v > 0.f) ? 1.f : ((v < 0.f) ? -1.f : 0.f);
    vb = fmaf(sgn, cb, vb);
    // cs = sqrt(gamma (gamma-1) e+)
    const float half_cs_inv = 0.5f * rcp_fast(cs);
    float epb = cb * sc.ggm1 * half_cs_inv;
    gamma_b = fmaf(cb * (2.f * sc.gamma - 1.f) * ep, half_cs_inv, gamma_b);
    // p = (gamma - 1) rho e+
    gamma_b = fmaf(pb * u[0], ep, gamma_b);
    float rhob = pb * sc.gm1 * ep;
    epb = fmaf(pb * sc.gm1, u[0], epb);
    // e+ = max(e, floor);  e = (eps - ke)/rho, ke = m2/(2 rho)
    const float eb = active ? epb : 0.f;
    const float ebr = eb * rinv;
    epsb += ebr;
    rhob += ebr * (2.f * ke * rinv - u[4] * rinv);       // eb * (-eps/rho^2 + m2/rho^3)
    const float mcoef = -ebr * rinv;                       // -eb / rho^2
    mnb = fmaf(mcoef, u[1], mnb);
    // v = m_n / rho
    mnb = fmaf(vb, rinv, mnb);
    rhob -= vb * v * rinv;
    ub[0] += rhob;
    ub[1] += mnb;
    ub[2] += fmaf(mcoef, u[2], Fb[2] * v);
    ub[3] += fmaf(mcoef, u[3], Fb[3] * v);
    ub[4] += epsb;
}

// L(A,B) = AB / (A + B + sign(A) eps4) if AB > 0 else 0
__device__ __forceinline__ float limL(float A, float B, float eps4) {
    const float t = A * B;
    const float den = (A + B) + copysignf(eps4, A);
    const float r = t * rcp_fast(den);
    return t > 0.f ? r : 0.f;
}
// value and both partials:  L_A = B (B + s eps4)/den^2,  L_B = A (A + s eps4)/den^2
__device__ __forceinline__ float limL_grad(float A, float B, float eps4, float& LA, float& LB) {
    const float t = A * B;
    const float s = copysignf(eps4, A);
    const float den = (A + B) + s;
    const bool on = t > 0.f;
    // gate on the reciprocal and never square it: with AB > 0, |den| >= 4 eps and |B| / |den|, |B + s| / |den| <= 1,
    // whereas 1/den^2 overflows fp32 for |den| < 5.4e-20 (wave tails decaying into a uniform region, lim_eps = 1e-20)
    const float rd = on ? rcp_fast(den) : 0.f;
    LA = (B * rd) * ((B + s) * rd);
    LB = (A * rd) * ((A + s) * rd);
    return t * rd;
}

// Marching-kernel forms of the limiter.  EPS = false drops the sign(A) 4 eps term of the denominator: for
// 4 eps <= 4e-18 it changes L by at most 2 eps in absolute value (L = AB/(A+B) <= min(|A|,|B|)), far below one fp32
// rounding of any flux the scheme produces; the forward launcher picks EPS = true whenever lim_eps > 1e-18.
// The gate AB > 0 is applied to the reciprocal, so value and partials all vanish with one select.
// With AB > 0 the signs of A, B and A + B agree, so  A + B + sign(A) 4 eps = sign(A) (|A + B| + 4 eps):  the epsilon
// costs one FADD with free |.| modifiers instead of a sign transfer.
template <bool EPS>
__device__ __forceinline__ float limM(float A, float B, float eps4) {
    const float t = A * B;
    if (EPS) {
        const float r = t > 0.f ? rcp_fast(fabsf(A + B) + eps4) : 0.f;
        return A * (fabsf(B) * r);
    }
    const float r = t > 0.f ? rcp_fast(A + B) : 0.f;
    return t * r;
}
// value and partials: with w = 1/|den| (0 when gated off), L = A |B| w, L_A = |B| (|B| + 4 eps) w^2, L_B likewise.
// EPS = 2 ("denominator only", the adjoint's choice for 0 < lim_eps <= 1e-18): 4 eps stays in the denominator but not in
// the two numerators.  Dropping it everywhere (EPS = 0) is harmless for the VALUE (|dL| <= 2 eps) but not for the
// partials: where a wave tail decays into a background that is exactly zero (transverse momentum ahead of a shock)
// |A|, |B| fall below 4 eps over ~10 cells and B^2/(A+B)^2 stays O(1) while the true partial B (B+s)/(A+B+s)^2 -> 0.
// With 4 eps in the denominator only, the partials are wrong by at most 0.25 and only where |A| + |B| ~ 4 eps (a range of
// one decade, less than a cell of such a tail), for one instruction per limiter.
template <int EPS>
__device__ __forceinline__ float limM_grad(float A, float B, float eps4, float& LA, float& LB) {
    const float t = A * B;
    const float den = EPS ? fabsf(A + B) + eps4 : fabsf(A + B);
    const float r = t > 0.f ? rcp_fast(den) : 0.f;
    const float wA = fabsf(A) * r, wB = fabsf(B) * r;
    if (EPS == 1) {
        LA = wB * ((fabsf(B) + eps4) * r);
        LB = wA * ((fabsf(A) + eps4) * r);
    } else {
        LA = wB * wB;
        LB = wA * wA;
    }
    return A * wB;
}

// (Tried and dropped, r02: the marching forward pipeline on packed fp32 -- __ffma2_rn / __fadd2_rn / __fmul2_rn on the
// component pairs (0,1), (2,3) -- cuts the loop from 482 to 446 SASS instructions per two cells (the packed arithmetic
// saves 61 issue slots, register pairing costs 25 in MOV / LDC / CS2R at the 128-register cap) and measures 169.4 ->
// 171.2 us at 256^3: a packed instruction holds the FMA pipe for two cycles, and the pipe, not issue, is what the saved
// slots would have had to feed.)
// ---- dual-energy variant (sweep_de.cu states the scheme; readings R33-R36): P on six components and its transpose
// (G, H, c, v, p, q_s) = P(u, q);  u6 = (rho, m_n, m_t1, m_t2, eps, q)
__device__ __forceinline__ void prim_de(const float (&u)[6], const SweepConst& sc, float (&G)[6], float (&H)[6], float& c,
                                        float& v, float& p, float& qs) {
    const float rinv = rcp_fast(u[0]);
    v = u[1] * rinv;
    const float ke = 0.5f * (u[1] * u[1] + u[2] * u[2] + u[3] * u[3]) * rinv;
    const float eT = (u[4] - ke) * rinv;
    const bool useT = eT > sc.de_eta * (u[4] * rinv);
    const float e = useT ? eT : u[5] * rinv;
    qs = u[0] * e;
    const float ep = !(e <= sc.e_floor) ? e : sc.e_floor;
    p = sc.gm1 * u[0] * ep;
    const float cs = sqrt_fast(sc.ggm1 * ep);
    c = fabsf(v) + cs;
    const float U[6] = {u[0], u[1], u[2], u[3], u[4], qs};
    float F[6];
    F[0] = u[1];
    F[1] = fmaf(u[1], v, p);
    F[2] = u[2] * v;
    F[3] = u[3] * v;
    F[4] = (u[4] + p) * v;
    F[5] = qs * v;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        G[k] = fmaf(c, U[k], F[k]);
        H[k] = fmaf(c, U[k], -F[k]);
    }
}

// Transpose of P at (u, q): cotangents of G, H (six each) and the extra cotangents of v, p, q_s; returns ub (six: the last
// is the cotangent of q) and adds to gamma_b.
__device__ __forceinline__ void prim_de_vjp(const float (&u)[6], const SweepConst& sc, const float (&Gb)[6],
                                            const float (&Hb)[6], float vb0, float pb0, float qsb0, float (&ub)[6],
                                            float& gamma_b) {
    const float rinv = rcp_fast(u[0]);
    const float v = u[1] * rinv;
    const float m2 = u[1] * u[1] + u[2] * u[2] + u[3] * u[3];
    const float ke = 0.5f * m2 * rinv;
    const float eT = (u[4] - ke) * rinv;
    const bool useT = eT > sc.de_eta * (u[4] * rinv);
    const float e = useT ? eT : u[5] * rinv;
    const float qs = u[0] * e;
    const bool active = !(e <= sc.e_floor);
    const float ep = active ? e : sc.e_floor;
    const float p = sc.gm1 * u[0] * ep;
    const float cs = sqrt_fast(sc.ggm1 * ep);
    const float c = fabsf(v) + cs;
    const float U[6] = {u[0], u[1], u[2], u[3], u[4], qs};
    float cub[6], Fb[6], Ub[6];
    float cb = 0.f;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        cub[k] = Gb[k] + Hb[k];
        Fb[k] = Gb[k] - Hb[k];
        cb = fmaf(cub[k], U[k], cb);
        Ub[k] = c * cub[k];
    }
    float mnb = fmaf(Fb[1], v, Fb[0]);
    float vb = vb0 + Fb[1] * u[1] + Fb[2] * u[2] + Fb[3] * u[3] + Fb[4] * (u[4] + p) + Fb[5] * qs;
    const float pb = pb0 + fmaf(Fb[4], v, Fb[1]);
    float epsb = Fb[4] * v;
    const float qsb = qsb0 + Ub[5] + Fb[5] * v;
    const float sgn = (v > 0.f) ? 1.f : ((v < 0.f) ? -1.f : 0.f);
    vb = fmaf(sgn, cb, vb);
    const float half_cs_inv = 0.5f * rcp_fast(cs);
    float epb = cb * sc.ggm1 * half_cs_inv;
    gamma_b = fmaf(cb * (2.f * sc.gamma - 1.f) * ep, half_cs_inv, gamma_b);
    gamma_b = fmaf(pb * u[0], ep, gamma_b);
    float rhob = pb * sc.gm1 * ep;
    epb = fmaf(pb * sc.gm1, u[0], epb);
    float eb = active ? epb : 0.f;
    eb = fmaf(qsb, u[0], eb);                    // q_s = rho e
    rhob = fmaf(qsb, e, rhob);
    const float eTb = useT ? eb : 0.f;           // e = e_T or q / rho
    const float eIb = useT ? 0.f : eb;
    const float qb = eIb * rinv;
    rhob -= eIb * u[5] * rinv * rinv;
    const float ebr = eTb * rinv;
    epsb += ebr;
    rhob += ebr * (2.f * ke * rinv - u[4] * rinv);
    const float mcoef = -ebr * rinv;
    mnb = fmaf(mcoef, u[1], mnb);
    mnb = fmaf(vb, rinv, mnb);
    rhob -= vb * v * rinv;
    ub[0] = Ub[0] + rhob;
    ub[1] = Ub[1] + mnb;
    ub[2] = Ub[2] + fmaf(mcoef, u[2], Fb[2] * v);
    ub[3] = Ub[3] + fmaf(mcoef, u[3], Fb[3] * v);
    ub[4] = Ub[4] + epsb;
    ub[5] = qb;
}

struct Ptr5 { const float* p[5]; };
struct MPtr5 { float* p[5]; };

__device__ __forceinline__ void block_max_to_global(float v, float* out, int* smem_slot) {
    // all values are >= 0 or NaN: compare as ints (NaN = 0x7fc00000 wins, which is what the NONFINITE check wants)
    int iv = __float_as_int(v) & 0x7fffffff;
    iv = __reduce_max_sync(0xffffffffu, iv);
    if ((threadIdx.x + threadIdx.y * blockDim.x) % 32 == 0) atomicMax(smem_slot, iv);
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0) atomicMax(reinterpret_cast<int*>(out), *smem_slot);
}

__device__ __forceinline__ void block_sum3_to_global(float a, float b, float c, double* out, float* sm /*3*32*/) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
        c += __shfl_xor_sync(0xffffffffu, c, o);
    }
    const int t = threadIdx.x + threadIdx.y * blockDim.x;
    const int w = t >> 5, nw = (blockDim.x * blockDim.y + 31) >> 5;
    if ((t & 31) == 0) { sm[w] = a; sm[32 + w] = b; sm[64 + w] = c; }
    __syncthreads();
    if (t < 32) {
        double da = t < nw ? (double)sm[t] : 0.0, db = t < nw ? (double)sm[32 + t] : 0.0, dc = t < nw ? (double)sm[64 + t] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            da += __shfl_xor_sync(0xffffffffu, da, o);
            db += __shfl_xor_sync(0xffffffffu, db, o);
            dc += __shfl_xor_sync(0xffffffffu, dc, o);
        }
        if (t == 0) { atomicAdd(out + 0, da); atomicAdd(out + 1, db); atomicAdd(out + 2, dc); }
    }
}

SweepConst make_sweep_const(const dh_ctx* c, float lam, float kap);

// dual-energy variant (sweep_de.cu): six fields (rho, m_x, m_y, m_z, eps, q)
int launch_sweep_de(dh_ctx* c, int d, float* const in[6], const float* g, float lam, float kap, float* const out[6],
                    float* cmax);
int launch_sweep_de_vjp(dh_ctx* c, int d, float* const in[6], const float* g, float lam, float kap,
                        float* const cot_out[6], float* const cot_in[6], float* g_bar, double* scal_bar);

// marching forward y/z sweep of the dual-energy variant (sweep_march.cu); pointers permuted to (rho, m_n, m_t1, m_t2, eps, q)
int launch_sweep_march_de(dh_ctx* c, int d, const float* const in[6], const float* g, float* const out[6], float* cmax,
                          const SweepConst& sc);

int launch_sweep_march_de_vjp(dh_ctx* c, int d, const float* const in[6], const float* g, const float* const cot_out[6],
                              float* const cot_in[6], float* gbar, double* scal, const SweepConst& sc);

// marching y/z kernels (sweep_march.cu); the field pointers are already permuted to (rho, m_n, m_t1, m_t2, eps)
int launch_sweep_march(dh_ctx* c, int d, const Ptr5& pin, const float* g, const MPtr5& pout, float* cmax,
                       const SweepConst& sc, float* delta_out);
int launch_sweep_march_vjp(dh_ctx* c, int d, const Ptr5& pin, const float* g, const Ptr5& pco, const MPtr5& pci,
                           float* gbar, double* scal, const SweepConst& sc);

}  // namespace dh
