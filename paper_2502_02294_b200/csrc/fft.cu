// fft.cu -- the Poisson solve of the particle-mesh step as five own passes (forward) over the mesh, for sm_100a.
//
// What is computed (PAPER.md:71 "potential formalism ... Fourier operators", :83 g = -grad phi; reading R12 of DESIGN.md):
//   forward:  g'_d = IFFT3( i k~_d A delta^(k) / k^2 ) / N^3,  d = x, y, z         (0 at k = 0; k~_d = 0 on the axis-d Nyquist plane)
//   adjoint:  delta_bar = IFFT3( sum_d conj(i k~_d A / k^2) FFT3(g_bar_d) ) / N^3
// The 3-D transforms are factored into 1-D passes so that the Green multiply and the spectral gradient ride on the z
// pass instead of being a pass of their own, and no pass is repeated:
//   forward:  x R2C (rows)  ->  y C2C  ->  [ z C2C -> symbol x3 -> z C2C^-1 x3 ]  ->  y C2C^-1 x3  ->  x C2R x3
//   adjoint:  x R2C x3      ->  y C2C x3 -> [ z C2C x3 -> symbol^T, sum -> z C2C^-1 ] ->  y C2C^-1    ->  x C2R
// Algorithmic traffic 8 + 8 + 16 + 24 + 24 = 80 B/cell against 208 B/cell for 1 R2C + multiply + 3 C2R as 3-pass library
// transforms.  Grids whose side is not a power of two in [32, 1024] keep the cuFFT path of pm.cu.
//
// Spectrum layout (internal): a real row of N values becomes M = N/2 complex values kx = 0 .. M-1 stored [z][y][kx] (rows
// stay 128-byte aligned) plus its Nyquist value kx = M stored in a separate plane [z][y] behind the main block:
// N^2 (M + 1) complex in all, the size of the library's half spectrum.
//
// 1-D transform of length L = R1 * R2 by T = L / E threads holding E values each (two register-radix stages and one
// shared-memory exchange):
//   forward, n = R2 n1 + n2, k = k1 + R1 k2:
//     stage 1 (owner of n2):  Y[n2][k1] = w_L^(n2 k1) sum_n1 x[R2 n1 + n2] w_R1^(n1 k1)
//     stage 2 (owner of k1):  X[k1 + R1 k2] = sum_n2 Y[n2][k1] w_R2^(n2 k2)
//   inverse, the mirror image (owner of k1 first, then owner of m2; n = m2 + R2 m1), conjugate roots, unnormalised.
// The register FFTs are decimation-in-frequency: natural order in, bit-reversed order out; the permutation is applied
// as compile-time register renaming where the next step reads the values.
#include <cmath>

#include "dh_internal.cuh"

namespace dh {
namespace {

// ------------------------------------------------------------------------------------------ register FFTs ----
// cos(2 pi j / 32), j = 0 .. 8
__host__ __device__ constexpr float c32_table(int j) {
    constexpr float t[9] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                            0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                            0.19509032201612826785f, 0.0f};
    return t[j];
}
__host__ __device__ constexpr float cos32(int j) { return j <= 8 ? c32_table(j) : -c32_table(16 - j); }   // j in [0, 16]
__host__ __device__ constexpr float sin32(int j) { return j <= 8 ? c32_table(8 - j) : c32_table(j - 8); }  // j in [0, 16]

template <int R>
__host__ __device__ constexpr int brev(int j) {
    // bit reversal of the log2(R) low bits, R <= 32
    int r = ((j & 1) << 4) | ((j & 2) << 2) | (j & 4) | ((j & 8) >> 2) | ((j & 16) >> 4);
    return R == 32 ? r : (R == 16 ? r >> 1 : (R == 8 ? r >> 2 : (R == 4 ? r >> 3 : (R == 2 ? r >> 4 : 0))));
}

// butterflies i = I .. R/2 - 1 of one decimation-in-frequency level on a[OFF .. OFF + R)
template <int R, int OFF, int I, bool INV, int NT>
struct Bfly {
    static __device__ __forceinline__ void run(float2 (&a)[NT]) {
        constexpr int H = R / 2;
        if constexpr (I < H) {
            const float2 u = a[OFF + I], v = a[OFF + I + H];
            a[OFF + I] = make_float2(u.x + v.x, u.y + v.y);
            const float2 d = make_float2(u.x - v.x, u.y - v.y);
            if constexpr (I == 0) {
                a[OFF + I + H] = d;
            } else if constexpr (2 * I == H) {                       // times -i (forward) or +i (inverse)
                a[OFF + I + H] = INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);
            } else {
                constexpr float c = cos32(I * (32 / R)), s = sin32(I * (32 / R));
                a[OFF + I + H] = INV ? make_float2(fmaf(d.x, c, -d.y * s), fmaf(d.y, c, d.x * s))
                                     : make_float2(fmaf(d.x, c, d.y * s), fmaf(d.y, c, -d.x * s));
            }
            Bfly<R, OFF, I + 1, INV, NT>::run(a);
        }
    }
};

// R-point DFT of a[OFF .. OFF + R) in place: a[OFF + j] <- X[brev<R>(j)]
template <int R, int OFF, bool INV, int NT>
__device__ __forceinline__ void dif(float2 (&a)[NT]) {
    if constexpr (R > 1) {
        Bfly<R, OFF, 0, INV, NT>::run(a);
        dif<R / 2, OFF, INV, NT>(a);
        dif<R / 2, OFF + R / 2, INV, NT>(a);
    }
}

// ------------------------------------------------------------------------------------------------ plans ----
template <int L> struct Plan;
#define DH_PLAN(L_, R1_, R2_, E_)                                                                   \
    template <> struct Plan<L_> {                                                                   \
        static constexpr int R1 = R1_, R2 = R2_, E = E_, T = L_ / E_, S1 = E_ / R1_, S2 = E_ / R2_; \
    };
DH_PLAN(16, 4, 4, 16)
DH_PLAN(32, 8, 4, 16)
DH_PLAN(64, 8, 8, 16)
DH_PLAN(128, 16, 8, 16)
DH_PLAN(256, 16, 16, 16)
DH_PLAN(512, 32, 16, 32)
DH_PLAN(1024, 32, 32, 32)
#undef DH_PLAN

__device__ __forceinline__ float2 cmul(float2 a, float2 w) {          // a * w
    return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 w) {         // a * conj(w)
    return make_float2(fmaf(a.x, w.x, a.y * w.y), fmaf(a.y, w.x, -a.x * w.y));
}

// One pencil of length L handled by T threads (thread t), exchange buffer ex_re / ex_im already offset to this pencil;
// element (k1, n2) of the exchange lives at ((k1 (R2 + 1) + n2) * PP).  tw[j * TWS] = (cos, sin)(2 pi j / L).
template <int L>
struct Pencil {
    using P = Plan<L>;
    static constexpr int R1 = P::R1, R2 = P::R2, E = P::E, T = P::T, S1 = P::S1, S2 = P::S2;
    static constexpr int EX = R1 * (R2 + 1);      // exchange elements per pencil (padded)

    // forward stage 1: a[s R1 + n1] = x[R2 n1 + n2], n2 = t + T s.  ROWTAB: tw is laid out [k1][n2] (the row kernels,
    // whose lanes run over n2: consecutive entries, no bank conflicts) instead of tw[j TWS] = root j.
    template <bool ROWTAB = false>
    static __device__ __forceinline__ void fwd1(float2 (&a)[E], int t, float* ex_re, float* ex_im, int PP,
                                                const float2* tw, int TWS) {
#pragma unroll
        for (int s = 0; s < S1; ++s) {
            if (s == 0) dif<R1, 0, false, E>(a);
            if (s == 1) dif<R1, (S1 > 1 ? 1 : 0) * R1, false, E>(a);
            if (s == 2) dif<R1, (S1 > 2 ? 2 : 0) * R1, false, E>(a);
            if (s == 3) dif<R1, (S1 > 3 ? 3 : 0) * R1, false, E>(a);
        }
#pragma unroll
        for (int s = 0; s < S1; ++s) {
            const int n2 = t + T * s;
#pragma unroll
            for (int j = 0; j < R1; ++j) {
                const int k1 = brev<R1>(j);
                float2 v = a[s * R1 + j];
                if (k1 != 0) v = cmulc(v, ROWTAB ? tw[k1 * R2 + n2] : tw[n2 * k1 * TWS]);
                ex_re[(k1 * (R2 + 1) + n2) * PP] = v.x;
                ex_im[(k1 * (R2 + 1) + n2) * PP] = v.y;
            }
        }
    }
    // forward stage 2: b[s R2 + j] <- X[k1 + R1 brev<R2>(j)], k1 = t + T s
    static __device__ __forceinline__ void fwd2(float2 (&b)[E], int t, const float* ex_re, const float* ex_im, int PP) {
#pragma unroll
        for (int s = 0; s < S2; ++s) {
            const int k1 = t + T * s;
#pragma unroll
            for (int n2 = 0; n2 < R2; ++n2)
                b[s * R2 + n2] = make_float2(ex_re[(k1 * (R2 + 1) + n2) * PP], ex_im[(k1 * (R2 + 1) + n2) * PP]);
        }
#pragma unroll
        for (int s = 0; s < S2; ++s) {
            if (s == 0) dif<R2, 0, false, E>(b);
            if (s == 1) dif<R2, (S2 > 1 ? 1 : 0) * R2, false, E>(b);
            if (s == 2) dif<R2, (S2 > 2 ? 2 : 0) * R2, false, E>(b);
            if (s == 3) dif<R2, (S2 > 3 ? 3 : 0) * R2, false, E>(b);
        }
    }
    // inverse stage 1: c[s R2 + k2] = X[k1 + R1 k2], k1 = t + T s.  ROWTAB: tw is laid out [m2][k1].
    template <bool ROWTAB = false>
    static __device__ __forceinline__ void inv1(float2 (&c)[E], int t, float* ex_re, float* ex_im, int PP,
                                                const float2* tw, int TWS) {
#pragma unroll
        for (int s = 0; s < S2; ++s) {
            if (s == 0) dif<R2, 0, true, E>(c);
            if (s == 1) dif<R2, (S2 > 1 ? 1 : 0) * R2, true, E>(c);
            if (s == 2) dif<R2, (S2 > 2 ? 2 : 0) * R2, true, E>(c);
            if (s == 3) dif<R2, (S2 > 3 ? 3 : 0) * R2, true, E>(c);
        }
#pragma unroll
        for (int s = 0; s < S2; ++s) {
            const int k1 = t + T * s;
#pragma unroll
            for (int j = 0; j < R2; ++j) {
                const int m2 = brev<R2>(j);
                float2 v = c[s * R2 + j];
                if (m2 != 0) v = cmul(v, ROWTAB ? tw[m2 * R1 + k1] : tw[m2 * k1 * TWS]);
                ex_re[(k1 * (R2 + 1) + m2) * PP] = v.x;
                ex_im[(k1 * (R2 + 1) + m2) * PP] = v.y;
            }
        }
    }
    // inverse stage 2: d[s R1 + j] <- x[m2 + R2 brev<R1>(j)], m2 = t + T s
    static __device__ __forceinline__ void inv2(float2 (&d)[E], int t, const float* ex_re, const float* ex_im, int PP) {
#pragma unroll
        for (int s = 0; s < S1; ++s) {
            const int m2 = t + T * s;
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1)
                d[s * R1 + k1] = make_float2(ex_re[(k1 * (R2 + 1) + m2) * PP], ex_im[(k1 * (R2 + 1) + m2) * PP]);
        }
#pragma unroll
        for (int s = 0; s < S1; ++s) {
            if (s == 0) dif<R1, 0, true, E>(d);
            if (s == 1) dif<R1, (S1 > 1 ? 1 : 0) * R1, true, E>(d);
            if (s == 2) dif<R1, (S1 > 2 ? 2 : 0) * R1, true, E>(d);
            if (s == 3) dif<R1, (S1 > 3 ? 3 : 0) * R1, true, E>(d);
        }
    }
};

// ------------------------------------------------------------------------------------------- strided tiles ----
// A tile is PP = 16 pencils that are adjacent in memory (stride ps) and run along a strided axis (element stride es).
constexpr int PP = 16;

struct Tile { long base; int ps, es; bool nyq; int i0, i1; };   // i0, i1: the two fixed mesh indices (meaning per kernel)

// y pass: pencils along y.  Main block: one tile per (z, 16 kx); Nyquist plane [z][y]: one tile per 16 z.
__device__ __forceinline__ Tile y_tile(int b, int N) {
    const int M = N / 2, per_z = M / PP, n_main = N * per_z;
    Tile tl;
    if (b < n_main) {
        const int z = b / per_z, c = b - z * per_z;
        tl.base = (long)z * N * M + c * PP; tl.ps = 1; tl.es = M; tl.nyq = false; tl.i0 = z; tl.i1 = c * PP;
    } else {
        const int z0 = (b - n_main) * PP;
        tl.base = (long)N * N * M + (long)z0 * N; tl.ps = N; tl.es = 1; tl.nyq = true; tl.i0 = z0; tl.i1 = 0;
    }
    return tl;
}
// z pass: pencils along z.  Main block: one tile per (ky, 16 kx); Nyquist plane: one tile per 16 ky.
__device__ __forceinline__ Tile z_tile(int b, int N) {
    const int M = N / 2, per_y = M / PP, n_main = N * per_y;
    Tile tl;
    if (b < n_main) {
        const int y = b / per_y, c = b - y * per_y;
        tl.base = (long)y * M + c * PP; tl.ps = 1; tl.es = N * M; tl.nyq = false; tl.i0 = y; tl.i1 = c * PP;
    } else {
        const int y0 = (b - n_main) * PP;
        tl.base = (long)N * N * M + y0; tl.ps = 1; tl.es = N; tl.nyq = true; tl.i0 = y0; tl.i1 = 0;
    }
    return tl;
}
__host__ __device__ constexpr int tiles_per_pass(int N) { return N * (N / 2 / PP) + N / PP; }

template <int L> __device__ __forceinline__ void load_tw(float2* tw_s, const float2* __restrict__ tw_g, int nthr) {
    for (int j = threadIdx.x; j < L; j += nthr) tw_s[j] = tw_g[j];
}
// row kernels (N real -> M = N/2 complex): tw_s[0 .. M) = roots of order N (post-processing), tw_s[M .. 2M) = the stage
// table of the M-point transform, [k1][n2] (FWD) or [m2][k1] (inverse): entry (a, b) = root a b of order M
template <int N, bool FWD> __device__ __forceinline__ void load_tw_rows(float2* tw_s, const float2* __restrict__ tw_g, int nthr) {
    constexpr int M = N / 2;
    using P = Plan<M>;
    for (int j = threadIdx.x; j < M; j += nthr) {
        tw_s[j] = tw_g[j];
        const int a = FWD ? j / P::R2 : j / P::R1, b = FWD ? j % P::R2 : j % P::R1;
        tw_s[M + j] = tw_g[2 * a * b];
    }
}

// global <-> registers in the two ownership patterns of Pencil<L>
template <int L>
__device__ __forceinline__ void load_A(float2 (&a)[Plan<L>::E], const float2* __restrict__ src, long es, int t) {
    using P = Plan<L>;
#pragma unroll
    for (int s = 0; s < P::S1; ++s)
#pragma unroll
        for (int n1 = 0; n1 < P::R1; ++n1) a[s * P::R1 + n1] = src[(long)(P::R2 * n1 + t + P::T * s) * es];
}
template <int L>
__device__ __forceinline__ void store_A(const float2 (&d)[Plan<L>::E], float2* __restrict__ dst, long es, int t) {
    using P = Plan<L>;
#pragma unroll
    for (int s = 0; s < P::S1; ++s)
#pragma unroll
        for (int j = 0; j < P::R1; ++j) dst[(long)(t + P::T * s + P::R2 * brev<P::R1>(j)) * es] = d[s * P::R1 + j];
}
template <int L>
__device__ __forceinline__ void load_B(float2 (&c)[Plan<L>::E], const float2* __restrict__ src, long es, int t) {
    using P = Plan<L>;
#pragma unroll
    for (int s = 0; s < P::S2; ++s)
#pragma unroll
        for (int k2 = 0; k2 < P::R2; ++k2) c[s * P::R2 + k2] = src[(long)(t + P::T * s + P::R1 * k2) * es];
}
template <int L>
__device__ __forceinline__ void store_B(const float2 (&b)[Plan<L>::E], float2* __restrict__ dst, long es, int t) {
    using P = Plan<L>;
#pragma unroll
    for (int s = 0; s < P::S2; ++s)
#pragma unroll
        for (int j = 0; j < P::R2; ++j) dst[(long)(t + P::T * s + P::R1 * brev<P::R2>(j)) * es] = b[s * P::R2 + j];
}

struct Spec3 {
    float2* p[3];
    // component selected without indexing the parameter struct dynamically (that would spill it to local memory and
    // turn every access through it into a generic load)
    __device__ __forceinline__ float2* sel(int d) const { return d == 0 ? p[0] : (d == 1 ? p[1] : p[2]); }
};
template <int N> constexpr size_t tile_smem() { return (size_t)N * sizeof(float2) + (size_t)2 * Pencil<N>::EX * PP * sizeof(float); }

// y pass, in place, blockIdx.y = component
template <int N, bool INV>
__global__ void __launch_bounds__(PP * Plan<N>::T) fft_y_kernel(Spec3 sp, const float2* __restrict__ tw_g) {
    using PN = Pencil<N>;
    constexpr int E = PN::E, NTHR = PP * PN::T;
    extern __shared__ float smem_f[];
    float2* tw = reinterpret_cast<float2*>(smem_f);
    float* ex_re = smem_f + 2 * N;
    float* ex_im = ex_re + PN::EX * PP;
    load_tw<N>(tw, tw_g, NTHR);
    const int p = threadIdx.x % PP, t = threadIdx.x / PP;
    const Tile tl = y_tile(blockIdx.x, N);
    float2* const ptr = sp.sel(blockIdx.y) + tl.base + (long)p * tl.ps;
    float2 a[E];
    if (!INV) load_A<N>(a, ptr, tl.es, t); else load_B<N>(a, ptr, tl.es, t);
    __syncthreads();
    if (!INV) PN::fwd1(a, t, ex_re + p, ex_im + p, PP, tw, 1); else PN::inv1(a, t, ex_re + p, ex_im + p, PP, tw, 1);
    __syncthreads();
    if (!INV) { PN::fwd2(a, t, ex_re + p, ex_im + p, PP); store_B<N>(a, ptr, tl.es, t); }
    else { PN::inv2(a, t, ex_re + p, ex_im + p, PP); store_A<N>(a, ptr, tl.es, t); }
}

// i k~_d A / (k^2 N^3) = i n~_d coef / n^2 with coef = A L / (2 pi N^3); 0 at n = 0; n~_d = 0 on the axis-d Nyquist plane
__device__ __forceinline__ int kint(int j, int N) { return j <= N / 2 ? j : j - N; }
__device__ __forceinline__ void symbol(int ix, int iy, int iz, int N, float coef, float (&s)[3]) {
    const int nx = ix, ny = kint(iy, N), nz = kint(iz, N);
    const int n2 = nx * nx + ny * ny + nz * nz;
    const float q = n2 > 0 ? coef / (float)n2 : 0.f;
    s[0] = (nx == N / 2) ? 0.f : q * nx;
    s[1] = (ny == N / 2) ? 0.f : q * ny;
    s[2] = (nz == N / 2) ? 0.f : q * nz;
}

// fused z pass of the forward solve: delta^ (x, y transformed) -> z C2C -> g^_d = i s_d delta^ -> z C2C^-1 -> g_d (x, y spectral)
template <int N>
__global__ void __launch_bounds__(PP * Plan<N>::T, (N <= 256 ? 2 : 1)) fft_z_green_kernel(const float2* __restrict__ dhat, Spec3 g,
                                                                      const float2* __restrict__ tw_g, float coef) {
    using PN = Pencil<N>;
    using P = Plan<N>;
    constexpr int E = PN::E, NTHR = PP * PN::T;
    extern __shared__ float smem_f[];
    float2* tw = reinterpret_cast<float2*>(smem_f);
    float* ex_re = smem_f + 2 * N;
    float* ex_im = ex_re + PN::EX * PP;
    load_tw<N>(tw, tw_g, NTHR);
    const int p = threadIdx.x % PP, t = threadIdx.x / PP;
    const Tile tl = z_tile(blockIdx.x, N);
    const long off = tl.base + (long)p * tl.ps;
    const int ix = tl.nyq ? N / 2 : tl.i1 + p, iy = tl.nyq ? tl.i0 + p : tl.i0;
    float2 b[E];
    load_A<N>(b, dhat + off, tl.es, t);
    __syncthreads();
    PN::fwd1(b, t, ex_re + p, ex_im + p, PP, tw, 1);
    __syncthreads();
    PN::fwd2(b, t, ex_re + p, ex_im + p, PP);          // b[s R2 + j] = delta^(kz = k1 + R1 brev(j))
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        float2 c[E];
#pragma unroll
        for (int s = 0; s < P::S2; ++s)
#pragma unroll
            for (int k2 = 0; k2 < P::R2; ++k2) {
                float sy[3];
                symbol(ix, iy, t + P::T * s + P::R1 * k2, N, coef, sy);
                const float2 v = b[s * P::R2 + brev<P::R2>(k2)];
                c[s * P::R2 + k2] = make_float2(-sy[d] * v.y, sy[d] * v.x);
            }
        __syncthreads();                                 // everybody is done reading the previous exchange
        PN::inv1(c, t, ex_re + p, ex_im + p, PP, tw, 1);
        __syncthreads();
        PN::inv2(c, t, ex_re + p, ex_im + p, PP);
        store_A<N>(c, g.p[d] + off, tl.es, t);
    }
}

// fused z pass of the adjoint solve: g_bar^_d (x, y transformed) -> z C2C -> delta_bar^ = sum_d conj(i s_d) g_bar^_d -> z C2C^-1
template <int N>
__global__ void __launch_bounds__(PP * Plan<N>::T, (N <= 256 ? 2 : 1)) fft_z_green_adj_kernel(Spec3 gb, float2* __restrict__ dbhat,
                                                                          const float2* __restrict__ tw_g, float coef) {
    using PN = Pencil<N>;
    using P = Plan<N>;
    constexpr int E = PN::E, NTHR = PP * PN::T;
    extern __shared__ float smem_f[];
    float2* tw = reinterpret_cast<float2*>(smem_f);
    float* ex_re = smem_f + 2 * N;
    float* ex_im = ex_re + PN::EX * PP;
    load_tw<N>(tw, tw_g, NTHR);
    const int p = threadIdx.x % PP, t = threadIdx.x / PP;
    const Tile tl = z_tile(blockIdx.x, N);
    const long off = tl.base + (long)p * tl.ps;
    const int ix = tl.nyq ? N / 2 : tl.i1 + p, iy = tl.nyq ? tl.i0 + p : tl.i0;
    float2 acc[E];                                       // natural order: acc[s R2 + k2] at kz = k1 + R1 k2
#pragma unroll
    for (int i = 0; i < E; ++i) acc[i] = make_float2(0.f, 0.f);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        float2 b[E];
        load_A<N>(b, gb.p[d] + off, tl.es, t);
        __syncthreads();
        PN::fwd1(b, t, ex_re + p, ex_im + p, PP, tw, 1);
        __syncthreads();
        PN::fwd2(b, t, ex_re + p, ex_im + p, PP);
#pragma unroll
        for (int s = 0; s < P::S2; ++s)
#pragma unroll
            for (int k2 = 0; k2 < P::R2; ++k2) {
                float sy[3];
                symbol(ix, iy, t + P::T * s + P::R1 * k2, N, coef, sy);
                const float2 v = b[s * P::R2 + brev<P::R2>(k2)];
                acc[s * P::R2 + k2].x = fmaf(sy[d], v.y, acc[s * P::R2 + k2].x);
                acc[s * P::R2 + k2].y = fmaf(-sy[d], v.x, acc[s * P::R2 + k2].y);
            }
    }
    __syncthreads();
    PN::inv1(acc, t, ex_re + p, ex_im + p, PP, tw, 1);
    __syncthreads();
    PN::inv2(acc, t, ex_re + p, ex_im + p, PP);
    store_A<N>(acc, dbhat + off, tl.es, t);
}

// ------------------------------------------------------------------------------------------ power spectrum ----
// Binned power spectrum of a real field ("power spectra of the baryon density using a differentiable
// routine") on the same passes: x R2C -> y C2C -> [ z C2C -> |F|^2 into bins ].
//   bin b = round(|n|), n = integer wave vector, 1 <= b <= N/2;  P_b = (L^3 / N^6) sum_{k in b} |F_k|^2 / count_b,
// the sums over the FULL spectrum: a half-spectrum element counts twice unless kx = 0 or kx = N/2.
// Transpose: field_bar = 2 IFFT3_unnormalised( g_b(k) F_k ), g_b = (L^3 / N^6) P_bar_b / count_b -- the fused z pass of the
// Poisson solve with a real, bin-indexed symbol and one component.
__device__ __forceinline__ int ps_bin(int ix, int iy, int iz, int N) {
    const int ny = kint(iy, N), nz = kint(iz, N);
    const int n2 = ix * ix + ny * ny + nz * nz;
    return (int)(sqrtf((float)n2) + 0.5f);         // exact: sqrt(n2) is never within 2.8e-4 of a half-integer for N <= 1024
}

template <int N>
__global__ void __launch_bounds__(PP * Plan<N>::T, (N <= 256 ? 2 : 1)) fft_z_power_kernel(const float2* __restrict__ fhat,
                                                                      const float2* __restrict__ tw_g,
                                                                      double* __restrict__ bins /* [2][N/2 + 1] */) {
    using PN = Pencil<N>;
    using P = Plan<N>;
    constexpr int E = PN::E, NTHR = PP * PN::T, NB = N / 2 + 1;
    extern __shared__ float smem_f[];
    __shared__ float hist[2 * NB];
    float2* tw = reinterpret_cast<float2*>(smem_f);
    float* ex_re = smem_f + 2 * N;
    float* ex_im = ex_re + PN::EX * PP;
    load_tw<N>(tw, tw_g, NTHR);
    for (int j = threadIdx.x; j < 2 * NB; j += NTHR) hist[j] = 0.f;
    const int p = threadIdx.x % PP, t = threadIdx.x / PP;
    const Tile tl = z_tile(blockIdx.x, N);
    const long off = tl.base + (long)p * tl.ps;
    const int ix = tl.nyq ? N / 2 : tl.i1 + p, iy = tl.nyq ? tl.i0 + p : tl.i0;
    const float w = (ix == 0 || ix == N / 2) ? 1.f : 2.f;
    float2 b[E];
    load_A<N>(b, fhat + off, tl.es, t);
    __syncthreads();
    PN::fwd1(b, t, ex_re + p, ex_im + p, PP, tw, 1);
    __syncthreads();
    PN::fwd2(b, t, ex_re + p, ex_im + p, PP);          // b[s R2 + j] = F(kz = k1 + R1 brev(j))
#pragma unroll
    for (int s = 0; s < P::S2; ++s)
#pragma unroll
        for (int k2 = 0; k2 < P::R2; ++k2) {
            const int bin = ps_bin(ix, iy, t + P::T * s + P::R1 * k2, N);
            const float2 v = b[s * P::R2 + brev<P::R2>(k2)];
            if (bin >= 1 && bin <= N / 2) {
                atomicAdd(&hist[bin], w * fmaf(v.x, v.x, v.y * v.y));
                atomicAdd(&hist[NB + bin], w);
            }
        }
    __syncthreads();
    for (int j = threadIdx.x; j < 2 * NB; j += NTHR)
        if (hist[j] != 0.f) atomicAdd(bins + j, (double)hist[j]);
}

// z pass of the transpose: F -> z C2C -> times gtab[bin] -> z C2C^-1, in place
template <int N>
__global__ void __launch_bounds__(PP * Plan<N>::T, (N <= 256 ? 2 : 1)) fft_z_power_adj_kernel(float2* __restrict__ fhat,
                                                                          const float2* __restrict__ tw_g,
                                                                          const float* __restrict__ gtab_g /* [N/2 + 1] */) {
    using PN = Pencil<N>;
    using P = Plan<N>;
    constexpr int E = PN::E, NTHR = PP * PN::T, NB = N / 2 + 1;
    extern __shared__ float smem_f[];
    __shared__ float gtab[NB];
    float2* tw = reinterpret_cast<float2*>(smem_f);
    float* ex_re = smem_f + 2 * N;
    float* ex_im = ex_re + PN::EX * PP;
    load_tw<N>(tw, tw_g, NTHR);
    for (int j = threadIdx.x; j < NB; j += NTHR) gtab[j] = gtab_g[j];
    const int p = threadIdx.x % PP, t = threadIdx.x / PP;
    const Tile tl = z_tile(blockIdx.x, N);
    const long off = tl.base + (long)p * tl.ps;
    const int ix = tl.nyq ? N / 2 : tl.i1 + p, iy = tl.nyq ? tl.i0 + p : tl.i0;
    float2 b[E];
    load_A<N>(b, fhat + off, tl.es, t);
    __syncthreads();
    PN::fwd1(b, t, ex_re + p, ex_im + p, PP, tw, 1);
    __syncthreads();
    PN::fwd2(b, t, ex_re + p, ex_im + p, PP);
    float2 c[E];
#pragma unroll
    for (int s = 0; s < P::S2; ++s)
#pragma unroll
        for (int k2 = 0; k2 < P::R2; ++k2) {
            const int bin = ps_bin(ix, iy, t + P::T * s + P::R1 * k2, N);
            const float g = (bin >= 1 && bin <= N / 2) ? gtab[bin] : 0.f;
            const float2 v = b[s * P::R2 + brev<P::R2>(k2)];
            c[s * P::R2 + k2] = make_float2(g * v.x, g * v.y);
        }
    __syncthreads();
    PN::inv1(c, t, ex_re + p, ex_im + p, PP, tw, 1);
    __syncthreads();
    PN::inv2(c, t, ex_re + p, ex_im + p, PP);
    store_A<N>(c, fhat + off, tl.es, t);
}

// ---------------------------------------------------------------------------------------------- x passes ----
// A real row r[0 .. N) is transformed through the M = N/2 point complex transform of z[n] = r[2n] + i r[2n+1]:
//   X[k] = (Z[k] + conj Z[M-k]) / 2 - (i/2) w_N^k (Z[k] - conj Z[M-k]),  k = 0 .. M  (Z[M] = Z[0]),  w_N = exp(-2 pi i / N)
// and back (unnormalised, result N r):  Z'[k] = (X[k] + conj X[M-k]) + i conj(w_N^k) (X[k] - conj X[M-k]).
// Block = RB rows x T threads per row (t fastest, so a row's loads and stores are contiguous).
template <int N> struct RowCfg {
    static constexpr int M = N / 2;
    using PM = Pencil<M>;
    static constexpr int T = PM::T, RB = (256 / T) < 1 ? 1 : 256 / T, NTHR = T * RB;
    // a warp is 32 / T rows x T threads: row strides congruent to T modulo 32 words (exchange, 4-byte accesses) and to
    // T modulo 16 float2 (natural-order array, 8-byte accesses) keep its rows in disjoint banks
    static constexpr int EXS = PM::EX + (((T - PM::EX) % 32) + 32) % 32;
    static constexpr int ZS = M + (T < 16 ? T : 16) + (T == 1 ? 1 : 0);     // float2 elements; index M is used by the C2R
    // the exchange arrays and the natural-order array are live in different phases and share one region
    static constexpr int REGION = RB * (2 * EXS > 2 * ZS ? 2 * EXS : 2 * ZS);       // floats
    static constexpr size_t SMEM = (size_t)REGION * sizeof(float) + (size_t)N * sizeof(float2);
};

template <int N>
__global__ void __launch_bounds__(RowCfg<N>::NTHR) fft_x_r2c_kernel(const float* __restrict__ in0, const float* __restrict__ in1,
                                                                    const float* __restrict__ in2, Spec3 out,
                                                                    const float2* __restrict__ tw_g) {
    using C = RowCfg<N>;
    using PM = typename C::PM;
    constexpr int M = C::M, E = PM::E, T = C::T;
    extern __shared__ float smem_f[];
    float2* tw = reinterpret_cast<float2*>(smem_f);                       // N entries: (cos, sin)(2 pi j / N)
    float2* zn = tw + N;                                                   // natural-order Z, RB rows of ZS ...
    float* ex_re = smem_f + 2 * N;                                         // ... aliased with the exchange arrays
    float* ex_im = ex_re + C::RB * C::EXS;
    load_tw_rows<N, true>(tw, tw_g, C::NTHR);
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    const long row = (long)blockIdx.x * C::RB + r;
    const float* in = blockIdx.y == 0 ? in0 : (blockIdx.y == 1 ? in1 : in2);
    const float2* src = reinterpret_cast<const float2*>(in) + row * M;
    float2 a[E];
    load_A<M>(a, src, 1, t);
    __syncthreads();
    PM::template fwd1<true>(a, t, ex_re + r * C::EXS, ex_im + r * C::EXS, 1, tw + M, 0);
    __syncthreads();
    PM::fwd2(a, t, ex_re + r * C::EXS, ex_im + r * C::EXS, 1);
    __syncthreads();                                                       // the exchange is consumed: reuse it for Z
    using P = Plan<M>;
#pragma unroll
    for (int s = 0; s < P::S2; ++s)
#pragma unroll
        for (int j = 0; j < P::R2; ++j) {
            const int k = t + P::T * s + P::R1 * brev<P::R2>(j);
            zn[r * C::ZS + k] = a[s * P::R2 + j];
        }
    __syncthreads();
    float2* const outp = out.sel(blockIdx.y);
    float2* dst = outp + row * M;
#pragma unroll
    for (int i = 0; i < E; ++i) {
        const int k = t + T * i;
        const int km = (M - k) & (M - 1);
        const float2 zk = zn[r * C::ZS + k];
        float2 zm = zn[r * C::ZS + km];                                                  // conj Z[M-k]
        zm.y = -zm.y;
        if (k == 0) {
            dst[0] = make_float2(zk.x + zk.y, 0.f);
            outp[(long)N * N * M + row] = make_float2(zk.x - zk.y, 0.f);                   // Nyquist plane [z][y]
        } else {
            const float2 sm = make_float2(zk.x + zm.x, zk.y + zm.y), df = make_float2(zk.x - zm.x, zk.y - zm.y);
            const float2 w = tw[k];                                                        // w_N^k = (w.x, -w.y)
            // -(i/2) (w.x - i w.y) (df.x + i df.y) = (1/2) [ (w.x df.y - w.y df.x) - i (w.x df.x + w.y df.y) ]
            const float2 q = make_float2(fmaf(w.x, df.y, -w.y * df.x), -fmaf(w.x, df.x, w.y * df.y));
            dst[k] = make_float2(0.5f * (sm.x + q.x), 0.5f * (sm.y + q.y));
        }
    }
}

template <int N>
__global__ void __launch_bounds__(RowCfg<N>::NTHR) fft_x_c2r_kernel(Spec3 in, float* __restrict__ out0, float* __restrict__ out1,
                                                                    float* __restrict__ out2,
                                                                    const float2* __restrict__ tw_g) {
    using C = RowCfg<N>;
    using PM = typename C::PM;
    using P = Plan<N / 2>;
    constexpr int M = C::M, E = PM::E, T = C::T;
    extern __shared__ float smem_f[];
    float2* tw = reinterpret_cast<float2*>(smem_f);
    float2* xn = tw + N;                                                   // natural-order X, RB rows of ZS ...
    float* ex_re = smem_f + 2 * N;                                         // ... aliased with the exchange arrays
    float* ex_im = ex_re + C::RB * C::EXS;
    load_tw_rows<N, false>(tw, tw_g, C::NTHR);
    const int t = threadIdx.x % T, r = threadIdx.x / T;
    const long row = (long)blockIdx.x * C::RB + r;
    const float2* __restrict__ inp = in.sel(blockIdx.y);
    const float2* __restrict__ src = inp + row * M;
    {
        float2 v[E], vn = make_float2(0.f, 0.f);       // all loads first: one memory round trip
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = __ldg(src + t + T * i);
        if (t == 0) vn = __ldg(inp + (long)N * N * M + row);
#pragma unroll
        for (int i = 0; i < E; ++i) xn[r * C::ZS + t + T * i] = v[i];
        if (t == 0) xn[r * C::ZS + M] = vn;
    }
    __syncthreads();
    float2 c[E];
#pragma unroll
    for (int s = 0; s < P::S2; ++s)
#pragma unroll
        for (int k2 = 0; k2 < P::R2; ++k2) {
            const int k = t + P::T * s + P::R1 * k2;
            const float2 xk = xn[r * C::ZS + k];
            float2 xm = xn[r * C::ZS + M - k];                                                    // conj X[M-k]
            xm.y = -xm.y;
            if (k == 0) {
                c[s * P::R2 + k2] = make_float2(xk.x + xm.x, xk.x - xm.x);     // imaginary parts of X[0], X[M] are ignored
            } else {
                const float2 sm = make_float2(xk.x + xm.x, xk.y + xm.y), df = make_float2(xk.x - xm.x, xk.y - xm.y);
                const float2 w = tw[k];                                         // conj(w_N^k) = (w.x, +w.y)
                // i (w.x + i w.y)(df.x + i df.y) = -(w.x df.y + w.y df.x) + i (w.x df.x - w.y df.y)
                c[s * P::R2 + k2] = make_float2(sm.x - fmaf(w.x, df.y, w.y * df.x), sm.y + fmaf(w.x, df.x, -w.y * df.y));
            }
        }
    __syncthreads();                                                       // X is consumed: reuse it for the exchange
    PM::template inv1<true>(c, t, ex_re + r * C::EXS, ex_im + r * C::EXS, 1, tw + M, 0);
    __syncthreads();
    PM::inv2(c, t, ex_re + r * C::EXS, ex_im + r * C::EXS, 1);
    float* outp = blockIdx.y == 0 ? out0 : (blockIdx.y == 1 ? out1 : out2);
    store_A<M>(c, reinterpret_cast<float2*>(outp) + row * M, 1, t);
}

}  // namespace

// ----------------------------------------------------------------------------------------------- launchers ----
bool own_fft_supported(int N) { return N == 32 || N == 64 || N == 128 || N == 256 || N == 512 || N == 1024; }

static float green_coef_own(const dh_ctx* c, float A) {
    return (float)((double)A * c->box / (2.0 * M_PI) / (double)c->n3);
}

template <int N>
static int own_forward(dh_ctx* c, const float* delta, float A, float* const g_out[3]) {
    using C = RowCfg<N>;
    const float2* tw = c->fft_tw;
    Spec3 s0{{c->spec[0], c->spec[0], c->spec[0]}}, sg{{c->spec[1], c->spec[2], c->spec[3]}};
    const unsigned row_blocks = (unsigned)((long)N * N / C::RB), tiles = (unsigned)tiles_per_pass(N);
    DH_CUDA(cudaFuncSetAttribute(fft_x_r2c_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    DH_CUDA(cudaFuncSetAttribute(fft_x_c2r_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    DH_CUDA(cudaFuncSetAttribute(fft_y_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_y_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_z_green_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_z_green_adj_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    {
        Prof prof(c, PROF_FFT_X1);
        fft_x_r2c_kernel<N><<<dim3(row_blocks, 1), C::NTHR, C::SMEM, c->stream>>>(delta, delta, delta, s0, tw);
    }
    {
        Prof prof(c, PROF_FFT_Y1);
        fft_y_kernel<N, false><<<dim3(tiles, 1), PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(s0, tw);
    }
    {
        Prof prof(c, PROF_GREEN);
        fft_z_green_kernel<N><<<tiles, PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(c->spec[0], sg, tw, green_coef_own(c, A));
    }
    {
        Prof prof(c, PROF_FFT_Y3);
        fft_y_kernel<N, true><<<dim3(tiles, 3), PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(sg, tw);
    }
    {
        Prof prof(c, PROF_FFT_X3);
        fft_x_c2r_kernel<N><<<dim3(row_blocks, 3), C::NTHR, C::SMEM, c->stream>>>(sg, g_out[0], g_out[1], g_out[2], tw);
    }
    c->launches += 5;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

template <int N>
static int own_adjoint(dh_ctx* c, float* const g_bar[3], float A, float* delta_bar) {
    using C = RowCfg<N>;
    const float2* tw = c->fft_tw;
    Spec3 s0{{c->spec[0], c->spec[0], c->spec[0]}}, sg{{c->spec[1], c->spec[2], c->spec[3]}};
    const unsigned row_blocks = (unsigned)((long)N * N / C::RB), tiles = (unsigned)tiles_per_pass(N);
    DH_CUDA(cudaFuncSetAttribute(fft_x_r2c_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    DH_CUDA(cudaFuncSetAttribute(fft_x_c2r_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    DH_CUDA(cudaFuncSetAttribute(fft_y_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_y_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_z_green_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_z_green_adj_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    {
        Prof prof(c, PROF_FFT_X3);
        fft_x_r2c_kernel<N><<<dim3(row_blocks, 3), C::NTHR, C::SMEM, c->stream>>>(g_bar[0], g_bar[1], g_bar[2], sg, tw);
    }
    {
        Prof prof(c, PROF_FFT_Y3);
        fft_y_kernel<N, false><<<dim3(tiles, 3), PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(sg, tw);
    }
    {
        Prof prof(c, PROF_GREEN_ADJ);
        fft_z_green_adj_kernel<N><<<tiles, PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(sg, c->spec[0], tw, green_coef_own(c, A));
    }
    {
        Prof prof(c, PROF_FFT_Y1);
        fft_y_kernel<N, true><<<dim3(tiles, 1), PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(s0, tw);
    }
    {
        Prof prof(c, PROF_FFT_X1);
        fft_x_c2r_kernel<N><<<dim3(row_blocks, 1), C::NTHR, C::SMEM, c->stream>>>(s0, delta_bar, delta_bar, delta_bar, tw);
    }
    c->launches += 5;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

// x and y forward passes of `field` into spec[0]
template <int N>
static int own_xy_forward(dh_ctx* c, const float* field) {
    using C = RowCfg<N>;
    Spec3 s0{{c->spec[0], c->spec[0], c->spec[0]}};
    const unsigned row_blocks = (unsigned)((long)N * N / C::RB), tiles = (unsigned)tiles_per_pass(N);
    DH_CUDA(cudaFuncSetAttribute(fft_x_r2c_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    DH_CUDA(cudaFuncSetAttribute(fft_y_kernel<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    fft_x_r2c_kernel<N><<<dim3(row_blocks, 1), C::NTHR, C::SMEM, c->stream>>>(field, field, field, s0, c->fft_tw);
    fft_y_kernel<N, false><<<dim3(tiles, 1), PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(s0, c->fft_tw);
    c->launches += 2;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

template <int N>
static int own_power(dh_ctx* c, const float* field, double* bins_dev) {
    DH_TRY(own_xy_forward<N>(c, field));
    DH_CUDA(cudaFuncSetAttribute(fft_z_power_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    fft_z_power_kernel<N><<<(unsigned)tiles_per_pass(N), PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(c->spec[0], c->fft_tw,
                                                                                                      bins_dev);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

template <int N>
static int own_power_adj(dh_ctx* c, const float* field, const float* gtab_dev, float* field_bar) {
    using C = RowCfg<N>;
    DH_TRY(own_xy_forward<N>(c, field));
    Spec3 s0{{c->spec[0], c->spec[0], c->spec[0]}};
    const unsigned row_blocks = (unsigned)((long)N * N / C::RB), tiles = (unsigned)tiles_per_pass(N);
    DH_CUDA(cudaFuncSetAttribute(fft_z_power_adj_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_y_kernel<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tile_smem<N>()));
    DH_CUDA(cudaFuncSetAttribute(fft_x_c2r_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    fft_z_power_adj_kernel<N><<<tiles, PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(c->spec[0], c->fft_tw, gtab_dev);
    fft_y_kernel<N, true><<<dim3(tiles, 1), PP * Plan<N>::T, tile_smem<N>(), c->stream>>>(s0, c->fft_tw);
    fft_x_c2r_kernel<N><<<dim3(row_blocks, 1), C::NTHR, C::SMEM, c->stream>>>(s0, field_bar, field_bar, field_bar, c->fft_tw);
    c->launches += 3;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

#define DH_FFT_DISPATCH(FN, ...)                           \
    switch (c->N) {                                        \
        case 32: return FN<32>(__VA_ARGS__);               \
        case 64: return FN<64>(__VA_ARGS__);               \
        case 128: return FN<128>(__VA_ARGS__);             \
        case 256: return FN<256>(__VA_ARGS__);             \
        case 512: return FN<512>(__VA_ARGS__);             \
        case 1024: return FN<1024>(__VA_ARGS__);           \
        default: set_error("own FFT: unsupported grid %d", c->N); return DH_ERR_INVALID; \
    }

int own_poisson_forward(dh_ctx* c, const float* delta, float A, float* const g_out[3]) {
    DH_FFT_DISPATCH(own_forward, c, delta, A, g_out)
}
int own_poisson_adjoint(dh_ctx* c, float* const g_bar[3], float A, float* delta_bar) {
    DH_FFT_DISPATCH(own_adjoint, c, g_bar, A, delta_bar)
}
int own_power_spectrum(dh_ctx* c, const float* field, double* bins_dev) {
    DH_FFT_DISPATCH(own_power, c, field, bins_dev)
}
int own_power_spectrum_adjoint(dh_ctx* c, const float* field, const float* gtab_dev, float* field_bar) {
    DH_FFT_DISPATCH(own_power_adj, c, field, gtab_dev, field_bar)
}

// (cos, sin)(2 pi j / N), j = 0 .. N-1, computed in double on the host
int own_fft_init(dh_ctx* c) {
    const int N = c->N;
    std::vector<float2> h(N);
    for (int j = 0; j < N; ++j) {
        const double th = 2.0 * M_PI * j / N;
        h[j] = make_float2((float)cos(th), (float)sin(th));
    }
    DH_TRY(dev_alloc(c, (void**)&c->fft_tw, N * sizeof(float2)));
    DH_CUDA(cudaMemcpy(c->fft_tw, h.data(), N * sizeof(float2), cudaMemcpyHostToDevice));
    return DH_OK;
}

}  // namespace dh
