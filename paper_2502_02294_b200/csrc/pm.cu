// pm.cu -- particle-mesh kernels (forward and adjoint) for sm_100a.
//
//   deposit      : delta_tot = [gas] rho_gas - rho_bar + m_p sum_p W(x_p - cell)      cloud in cell
//   green        : g^_d(k) = i k~_d A delta^(k) / (k^2 N^3)                            PAPER.md:71, :83, reading R12
//   kick_drift   : w += K g'(x);  x += w Dtau/dx, wrapped to [0, N)                    Eq. 2-3
// and their transposes.  CIC convention (reading R13): mesh values live at cell centres (i + 1/2), so s = x - 1/2,
// i0 = floor(s), f = s - i0, i1 = i0 + 1, both wrapped mod N, weights (1-f | f) per axis; the same (i0, f) serve
// deposit and gather, so there is no self-force.  cuFFT does the 3-D R2C / C2R transforms only.
#include "dh_internal.cuh"

namespace dh {

// ------------------------------------------------------------------------------------------------- CIC index ----
struct Cic {
    int i0[3], i1[3];
    float f[3];
};

// i0 = floor(x - 0.5) mod N.  x - 0.5f is exact in fp32 for x >= 0.25 and cannot round across an integer below that,
// so this integer is bit-identical to the fp64 evaluation on the same fp32 input (reading R22).
__device__ __forceinline__ void cic_axis(float x, int N, int& i0, int& i1, float& f) {
    const float s = x - 0.5f;
    const float fl = floorf(s);
    f = s - fl;
    int i = (int)fl;
    i = i < 0 ? i + N : i;
    i = i >= N ? i - N : i;
    i0 = i;
    i1 = (i + 1 == N) ? 0 : i + 1;
}

__device__ __forceinline__ Cic cic_of(float x, float y, float z, int N) {
    Cic c;
    cic_axis(x, N, c.i0[0], c.i1[0], c.f[0]);
    cic_axis(y, N, c.i0[1], c.i1[1], c.f[1]);
    cic_axis(z, N, c.i0[2], c.i1[2], c.f[2]);
    return c;
}

// The 8 cells of a particle's cloud as 32-bit linear indices (N^3 <= 2^30): lo[j] / hi[j] = lower- / upper-x cell of
// row j = 2 cz + cy, and the row weights wzy[j] = wz[cz] wy[cy].  All index arithmetic of the particle kernels is
// 32-bit: these kernels are bound by instruction issue, not by bytes, and 64-bit address chains were half of it.
struct Cic8 {
    int lo[4], hi[4];
    float wzy[4], wx0, wx1;
    int i0x, i1x, row;     // row = i0z N + i0y identifies the 2x2 group of rows
    float fy, fz;
};

__device__ __forceinline__ Cic8 cic8_of(float x, float y, float z, int N) {
    Cic8 q;
    int i0y, i1y, i0z, i1z;
    float fx;
    cic_axis(x, N, q.i0x, q.i1x, fx);
    cic_axis(y, N, i0y, i1y, q.fy);
    cic_axis(z, N, i0z, i1z, q.fz);
    const int z0 = i0z * N, z1 = i1z * N;
    q.row = z0 + i0y;
    const int r[4] = {(z0 + i0y) * N, (z0 + i1y) * N, (z1 + i0y) * N, (z1 + i1y) * N};
#pragma unroll
    for (int j = 0; j < 4; ++j) { q.lo[j] = r[j] + q.i0x; q.hi[j] = r[j] + q.i1x; }
    q.wx0 = 1.f - fx; q.wx1 = fx;
    const float wy0 = 1.f - q.fy, wz0 = 1.f - q.fz;
    q.wzy[0] = wz0 * wy0; q.wzy[1] = wz0 * q.fy; q.wzy[2] = q.fz * wy0; q.wzy[3] = q.fz * q.fy;
    return q;
}

__global__ void cell_index_kernel(const float* __restrict__ x, int64_t n, int N, int32_t* i0, int32_t* i1) {
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    int a, b; float f;
    cic_axis(x[p], N, a, b, f);
    i0[p] = a; i1[p] = b;
}

__global__ void fill_kernel(float* p, int64_t n, float v) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; i < n; i += stride) p[i] = v;
}

// --------------------------------------------------------------------------------------------------- deposit ----
// delta = flag * rho_gas - rho_bar  (replaces the memset of the mesh)
__global__ void source_init_kernel(const float4* __restrict__ rho, float4* __restrict__ delta, int64_t n4, float flag,
                                   float rho_bar) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; i < n4; i += stride) {
        float4 r = rho ? __ldg(rho + i) : make_float4(0.f, 0.f, 0.f, 0.f);
        delta[i] = make_float4(fmaf(flag, r.x, -rho_bar), fmaf(flag, r.y, -rho_bar), fmaf(flag, r.z, -rho_bar),
                               fmaf(flag, r.w, -rho_bar));
    }
}

// Particles are stored in lattice order (particle p started at lattice site p) and neighbouring particles move
// together, so the 32 lanes of a warp (32 consecutive lattice sites along x) deposit into a compact, mostly
// consecutive run of cells: lane l's upper-x cell is usually lane l+1's lower-x cell.  The kernel uses that in
// registers: every lane hands the four upper-x contributions to the next lane when the cells match (one shuffle
// each), so a warp issues 4 coalesced RED.ADD.F32 on consecutive addresses instead of 8, and only the lanes whose
// neighbour does not match (warp end, a particle that crossed its neighbour, a row change) issue the other 4.  The
// reductions go straight to the mesh in L2: on B200 coalesced fp32 RED runs at > 1.4e12 adds/s, faster than any
// shared-memory tile (fp32 shared atomics are compare-and-swap loops on sm_100), and no assumption is made about how
// far particles have moved.
__global__ void __launch_bounds__(256) deposit_kernel(const float* __restrict__ x, const float* __restrict__ y,
                                                      const float* __restrict__ z, int np, int N, float mp,
                                                      float* __restrict__ delta) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = p < np;
    const int lane = threadIdx.x & 31;
    Cic8 q = cic8_of(live ? __ldg(x + p) : 1.f, live ? __ldg(y + p) : 1.f, live ? __ldg(z + p) : 1.f, N);
    const int row = live ? q.row : -7;
    const int row_next = __shfl_down_sync(0xffffffffu, row, 1);
    const int i0x_next = __shfl_down_sync(0xffffffffu, q.i0x, 1);
    const bool pass = live && lane < 31 && row_next == row && i0x_next == q.i1x;
    const float wlo = mp * q.wx0, whi = mp * q.wx1;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float up = q.wzy[j] * whi;
        const float recv = __shfl_up_sync(0xffffffffu, pass ? up : 0.f, 1);
        const float lo = fmaf(q.wzy[j], wlo, lane > 0 ? recv : 0.f);
        if (live) {
            atomicAdd(delta + q.lo[j], lo);
            if (!pass) atomicAdd(delta + q.hi[j], up);
        }
    }
}

// north_star (a)'s design, kept for the A/B in profiles/ (dh_tune "deposit_tile"): a block owns a brick of TBX x TBY x TBZ
// lattice sites, accumulates their clouds into a shared-memory tile that covers the brick plus a margin of TR cells, and
// flushes the tile to the mesh with coalesced RED; contributions that leave the tile (a particle displaced by more than
// TR cells) go straight to the mesh.  fp32 atomicAdd on shared memory compiles to an ATOMS.CAST.SPIN loop on sm_100
// (compare-and-swap; SASS excerpt in profiles/), so every one of the 8 tile updates per particle is a retry loop under
// contention, and the flush still issues (TBX+2TR)(TBY+2TR)(TBZ+2TR) / (TBX TBY TBZ) = 3.6 RED lanes per particle where the
// run-aggregated kernel above issues 4 to 5 -- measured slower at 256^3 both early and late (profiles/r02.md).
constexpr int TBX = 32, TBY = 8, TBZ = 8, TR = 3;
constexpr int TLX = TBX + 2 * TR, TLY = TBY + 2 * TR, TLZ = TBZ + 2 * TR;
// FIXED = true: the tile holds 32-bit fixed-point sums (weights in units of m_p 2^-22; native ATOMS.ADD on integers)
// instead of fp32 (ATOMS.CAST.SPIN): the experiment that separates the cost of the CAS loop from the cost of the design.
template <bool FIXED>
__global__ void __launch_bounds__(1024) deposit_tile_kernel(const float* __restrict__ x, const float* __restrict__ y,
                                                            const float* __restrict__ z, int nps, int N, float mp,
                                                            float* __restrict__ delta) {
    __shared__ float tile[TLZ * TLY * TLX];
    int* const itile = reinterpret_cast<int*>(tile);
    constexpr float FX = 4194304.f;            // 2^22: a cell holds up to 2^9 particle masses
    const int tid = threadIdx.x;
    for (int i = tid; i < TLZ * TLY * TLX; i += blockDim.x) tile[i] = 0.f;
    __syncthreads();
    const int bx = blockIdx.x * TBX, by = blockIdx.y * TBY, bz = blockIdx.z * TBZ;      // brick origin (lattice sites)
    const float scale = (float)N / (float)nps;                                          // cells per lattice spacing
    // tile origin in cells: the cell of the brick's first lattice site minus the margin
    const int ox = (int)floorf((bx + 0.5f) * scale - 0.5f) - TR, oy = (int)floorf((by + 0.5f) * scale - 0.5f) - TR,
              oz = (int)floorf((bz + 0.5f) * scale - 0.5f) - TR;
    for (int s = tid; s < TBX * TBY * TBZ; s += blockDim.x) {
        const int lx = bx + s % TBX, ly = by + (s / TBX) % TBY, lz = bz + s / (TBX * TBY);
        if (lx >= nps || ly >= nps || lz >= nps) continue;
        const int p = (lz * nps + ly) * nps + lx;
        const Cic c = cic_of(__ldg(x + p), __ldg(y + p), __ldg(z + p), N);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int dx = k & 1, dy = (k >> 1) & 1, dz = k >> 2;
            const int ix = dx ? c.i1[0] : c.i0[0], iy = dy ? c.i1[1] : c.i0[1], iz = dz ? c.i1[2] : c.i0[2];
            const float w = mp * (dx ? c.f[0] : 1.f - c.f[0]) * (dy ? c.f[1] : 1.f - c.f[1]) * (dz ? c.f[2] : 1.f - c.f[2]);
            // tile coordinates, periodic distance from the tile origin
            int tx = ix - ox, ty = iy - oy, tz = iz - oz;
            tx = tx < 0 ? tx + N : (tx >= N ? tx - N : tx);
            ty = ty < 0 ? ty + N : (ty >= N ? ty - N : ty);
            tz = tz < 0 ? tz + N : (tz >= N ? tz - N : tz);
            if (tx < TLX && ty < TLY && tz < TLZ) {
                if (FIXED) atomicAdd(&itile[(tz * TLY + ty) * TLX + tx], __float2int_rn(w * (FX / mp)));
                else atomicAdd(&tile[(tz * TLY + ty) * TLX + tx], w);
            } else {
                atomicAdd(delta + ((size_t)iz * N + iy) * N + ix, w);
            }
        }
    }
    __syncthreads();
    for (int i = tid; i < TLZ * TLY * TLX; i += blockDim.x) {
        const float v = FIXED ? (float)itile[i] * (mp / FX) : tile[i];
        if (v == 0.f) continue;
        int ix = ox + i % TLX, iy = oy + (i / TLX) % TLY, iz = oz + i / (TLX * TLY);
        ix = ((ix % N) + N) % N; iy = ((iy % N) + N) % N; iz = ((iz % N) + N) % N;
        atomicAdd(delta + ((size_t)iz * N + iy) * N + ix, v);
    }
}

// ----------------------------------------------------------------------------------------- Green's function ----
__device__ __forceinline__ int kint(int j, int N) { return j <= N / 2 ? j : j - N; }

// one thread per complex element of the half spectrum [z][y][x <= N/2]
__device__ __forceinline__ void green_symbol(int64_t c, int N, int nxh, float coef, float& sx, float& sy, float& sz) {
    const int ix = (int)(c % nxh);
    const int64_t r = c / nxh;
    const int iy = (int)(r % N), iz = (int)(r / N);
    const int nx = ix, ny = kint(iy, N), nz = kint(iz, N);
    const int n2 = nx * nx + ny * ny + nz * nz;
    // i k~_d A / k^2 = i n~_d (A L / 2 pi) / n^2 ;  0 at k = 0 ;  n~_d = 0 on the axis-d Nyquist plane
    const float s = n2 > 0 ? coef / (float)n2 : 0.f;
    sx = (nx == N / 2) ? 0.f : s * nx;
    sy = (ny == N / 2) ? 0.f : s * ny;
    sz = (nz == N / 2) ? 0.f : s * nz;
}

__global__ void __launch_bounds__(256) green_kernel(const float2* __restrict__ dh, float2* __restrict__ gx,
                                                    float2* __restrict__ gy, float2* __restrict__ gz, int N,
                                                    int64_t nspec, float coef /* A L / (2 pi N^3) */) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nspec) return;
    float sx, sy, sz;
    green_symbol(c, N, N / 2 + 1, coef, sx, sy, sz);
    const float2 d = __ldg(dh + c);
    gx[c] = make_float2(-sx * d.y, sx * d.x);
    gy[c] = make_float2(-sy * d.y, sy * d.x);
    gz[c] = make_float2(-sz * d.y, sz * d.x);
}

// delta_bar^ = sum_d conj(i s_d) g_bar^_d = sum_d s_d (im, -re)
__global__ void __launch_bounds__(256) green_adj_kernel(const float2* __restrict__ gx, const float2* __restrict__ gy,
                                                        const float2* __restrict__ gz, float2* __restrict__ db, int N,
                                                        int64_t nspec, float coef) {
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nspec) return;
    float sx, sy, sz;
    green_symbol(c, N, N / 2 + 1, coef, sx, sy, sz);
    const float2 a = __ldg(gx + c), b = __ldg(gy + c), e = __ldg(gz + c);
    db[c] = make_float2(sx * a.y + sy * b.y + sz * e.y, -(sx * a.x + sy * b.x + sz * e.x));
}

// ------------------------------------------------------------------------------------------- gather helpers ----
// The 8 cloud values of every mesh a kernel gathers from are loaded in one batch (all loads issued before the first
// use) and reduced afterwards: one memory round trip per kernel phase instead of one per cloud row.  ptxas only keeps
// the batch together when the kernel's launch bounds allow it more than 32 registers (minimum blocks per SM given).
// (Tried and dropped, r02: taking the upper-x value from the next lane's register by shuffle when the two particles
// continue the run of cells, so that only the lower-x loads are full-width requests -- 244 -> 254 us kick_drift, 136 ->
// 157 us deposit_adj, 467 -> 486 us kick_drift_adj at 256^3: the 12 extra SHFL wait on the loads they forward.)
struct Gath8 { float lo[4], hi[4]; };
__device__ __forceinline__ void gather_issue(const float* __restrict__ m, const Cic8& q, Gath8& v) {
#pragma unroll
    for (int j = 0; j < 4; ++j) { v.lo[j] = __ldg(m + q.lo[j]); v.hi[j] = __ldg(m + q.hi[j]); }
}
__device__ __forceinline__ float gather_reduce(const Gath8& v, const Cic8& q) {
    float acc = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) acc = fmaf(q.wzy[j], fmaf(q.wx0, v.lo[j], q.wx1 * v.hi[j]), acc);
    return acc;
}

// ---------------------------------------------------------------------------------------------- kick + drift ----
// x mod N into [0, N) without a division: the reciprocal form can be one period off next to a multiple of N, which the
// two corrections absorb (any finite x).
__device__ __forceinline__ float wrap_pos(float x, float fN, float invN) {
    x = fmaf(-fN, floorf(x * invN), x);
    x = x < 0.f ? x + fN : x;
    return x >= fN ? x - fN : x;
}

// in -> out (the same arrays when the update is in place; one thread reads and writes only its own particle)
// Block size and register cap measured at 256^3: 64-128 threads 230 us, 256 threads 237 us, 512 threads 278 us; flat in
// the register cap between 32 and 85; two particles per thread 264-314 us (this kernel wants warps, not ILP).
// (Tried and dropped, r02: depositing the NEW positions from this kernel inside dh_run, so that the next step starts with
// its Poisson solve -- the REDs cost what they cost in a kernel of their own: kick_drift 231 -> 286 us, + 15 us to zero the
// mesh, + the last sweep adding rho' - rho_bar by RED instead of storing it; forward 1.155 -> 1.154 ms/step early, 1.229 ->
// 1.196 late, forward + VJP unchanged.  Persistent blocks with the next chunk's six fields prefetched into registers, the
// adjoint's schedule: 246 - 300 us against 231 for 128 x 4 ... 256 x 4 threads x blocks per SM -- with 60 B per particle the
// one-shot grid's 24 warps per SM already cover the two round trips, and the persistent loop only lowers occupancy.)
constexpr int KD_T = 128;
__global__ void __launch_bounds__(KD_T, 6) kick_drift_kernel(const float* __restrict__ gx, const float* __restrict__ gy,
                                                         const float* __restrict__ gz, const float* px, const float* py,
                                                         const float* pz, const float* wx_, const float* wy_,
                                                         const float* wz_, float* ox, float* oy, float* oz, float* owx,
                                                         float* owy, float* owz, int np, int N, float K,
                                                         float dtau_dx, float fN, float invN, int gravity) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const float x = px[p], y = py[p], z = pz[p];
    float ux = wx_[p], uy = wy_[p], uz = wz_[p];
    if (gravity) {
        const Cic8 q = cic8_of(x, y, z, N);
        Gath8 a, b, c;
        gather_issue(gx, q, a); gather_issue(gy, q, b); gather_issue(gz, q, c);
        ux = fmaf(K, gather_reduce(a, q), ux);
        uy = fmaf(K, gather_reduce(b, q), uy);
        uz = fmaf(K, gather_reduce(c, q), uz);
    }
    ox[p] = wrap_pos(fmaf(ux, dtau_dx, x), fN, invN);
    oy[p] = wrap_pos(fmaf(uy, dtau_dx, y), fN, invN);
    oz[p] = wrap_pos(fmaf(uz, dtau_dx, z), fN, invN);
    owx[p] = ux; owy[p] = uy; owz[p] = uz;
}

__device__ __forceinline__ void block_sum2_to_global(float a, float b, double* outa, double* outb, float* sm /*64*/) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    const int t = threadIdx.x, w = t >> 5, nw = (blockDim.x + 31) >> 5;
    if ((t & 31) == 0) { sm[w] = a; sm[32 + w] = b; }
    __syncthreads();
    if (t < 32) {
        double da = t < nw ? (double)sm[t] : 0.0, db = t < nw ? (double)sm[32 + t] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            da += __shfl_xor_sync(0xffffffffu, da, o);
            db += __shfl_xor_sync(0xffffffffu, db, o);
        }
        if (t == 0) { atomicAdd(outa, da); if (outb) atomicAdd(outb, db); }
    }
}

// ------------------------------------------------------------------------ adjoint of kick + drift + gather ----
// Forward: w' = w + K g_p(x); x' = wrap(x + w' dtau/dx).
//   wt_b = w'_b + (dtau/dx) x'_b;  w_b = wt_b;  x_b = x'_b + K sum_d wt_b,d d g_p,d / dx;
//   g'_b(cell) += W K wt_b (vector deposit);  K_b += wt_b . g_p;  (dtau/dx)_b += x'_b . w'
// The vector deposit aggregates along x inside the warp exactly like deposit_kernel: 12 coalesced RED per warp
// instead of 24, the rest only from lanes whose neighbour does not continue the run of cells.
// Persistent blocks of RT threads walk chunks of RT consecutive particles; the 12 per-particle fields of the NEXT chunk
// are loaded into registers before the current chunk's 24 gathers are issued, so one memory round trip per chunk is
// exposed instead of two, and the two scalar sums leave the block once per kernel instead of once per 256 particles.
// The register budget matters more than occupancy here (measured at 256^3: 80 registers / 3 blocks per SM 465 us,
// 64 / 4 635 us, 48 / 5 813 us; one particle per thread, a block per 256 particles 765 us): with fewer registers
// ptxas splits the gather batch and every split is another exposed round trip.
constexpr int RT = 256;
struct CPtr3 { const float* p[3]; };
struct MPtr3 { float* p[3]; };
struct CPtr12 { const float* p[12]; };
struct MPtr6 { float* p[6]; };

template <int NF, class Src>
__device__ __forceinline__ void reg_load(const Src& src, int p, int np, float (&v)[NF]) {
    if (p < np) {
#pragma unroll
        for (int f = 0; f < NF; ++f) v[f] = src.p[f][p];
    } else {
#pragma unroll
        for (int f = 0; f < NF; ++f) v[f] = f < 3 ? 1.f : 0.f;
    }
}

template <bool GRAV>
__global__ void __launch_bounds__(RT, 3) kick_drift_adj_kernel(CPtr3 g, CPtr12 pin, MPtr6 cot_in, MPtr3 gbar, int np,
                                                                   int nchunks, int N, float K, float dtau_dx, double* K_b,
                                                                   double* dtdx_b) {
    __shared__ float sm_red[64];
    const int lane = threadIdx.x & 31;
    float kacc = 0.f, dacc = 0.f;
    int c = blockIdx.x;
    float cur[12], nxt[12];
    reg_load<12>(pin, c * RT + threadIdx.x, np, cur);
    for (; c < nchunks; c += gridDim.x) {
        const int p = c * RT + threadIdx.x;
        const bool live = p < np;
        const int cn = c + gridDim.x;
        reg_load<12>(pin, cn < nchunks ? cn * RT + threadIdx.x : np, np, nxt);
        const float x = cur[0], y = cur[1], z = cur[2];
        const float w0[3] = {cur[3], cur[4], cur[5]}, xb[3] = {cur[6], cur[7], cur[8]}, wb[3] = {cur[9], cur[10], cur[11]};
        const float wt[3] = {fmaf(dtau_dx, xb[0], wb[0]), fmaf(dtau_dx, xb[1], wb[1]), fmaf(dtau_dx, xb[2], wb[2])};
        float gp[3] = {0.f, 0.f, 0.f};
        float xo[3] = {xb[0], xb[1], xb[2]};
        if (GRAV) {
            const Cic8 q = cic8_of(x, y, z, N);
            const int row = live ? q.row : -7;
            const int row_next = __shfl_down_sync(0xffffffffu, row, 1);
            const int i0x_next = __shfl_down_sync(0xffffffffu, q.i0x, 1);
            const bool pass = live && lane < 31 && row_next == row && i0x_next == q.i1x;
            const float kw[3] = {K * wt[0], K * wt[1], K * wt[2]};
            const float wy[2] = {1.f - q.fy, q.fy}, wz[2] = {1.f - q.fz, q.fz};
            Gath8 vx, vy, vz;
            if (live) { gather_issue(g.p[0], q, vx); gather_issue(g.p[1], q, vy); gather_issue(g.p[2], q, vz); }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int cz = j >> 1, cy = j & 1;
                const float wzy = q.wzy[j];
                const float dzy = (cz ? 1.f : -1.f) * wy[cy], dyz = (cy ? 1.f : -1.f) * wz[cz];
                float s_lo = 0.f, s_hi = 0.f;
                if (live) {
                    const float a0 = vx.lo[j], a1 = vy.lo[j], a2 = vz.lo[j];
                    const float b0 = vx.hi[j], b1 = vy.hi[j], b2 = vz.hi[j];
                    const float wl = wzy * q.wx0, wh = wzy * q.wx1;
                    gp[0] = fmaf(wl, a0, fmaf(wh, b0, gp[0]));
                    gp[1] = fmaf(wl, a1, fmaf(wh, b1, gp[1]));
                    gp[2] = fmaf(wl, a2, fmaf(wh, b2, gp[2]));
                    s_lo = kw[0] * a0 + kw[1] * a1 + kw[2] * a2;
                    s_hi = kw[0] * b0 + kw[1] * b1 + kw[2] * b2;
                }
                const float s_x = fmaf(q.wx0, s_lo, q.wx1 * s_hi);
                xo[0] = fmaf(wzy, s_hi - s_lo, xo[0]);
                xo[1] = fmaf(dyz, s_x, xo[1]);
                xo[2] = fmaf(dzy, s_x, xo[2]);
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const float up = wzy * q.wx1 * kw[d];
                    const float recv = __shfl_up_sync(0xffffffffu, pass ? up : 0.f, 1);
                    const float lo = fmaf(wzy * q.wx0, kw[d], lane > 0 ? recv : 0.f);
                    if (live) {
                        atomicAdd(gbar.p[d] + q.lo[j], lo);
                        if (!pass) atomicAdd(gbar.p[d] + q.hi[j], up);
                    }
                }
            }
        }
        if (live) {
            const float wn[3] = {fmaf(K, gp[0], w0[0]), fmaf(K, gp[1], w0[1]), fmaf(K, gp[2], w0[2])};
            kacc += wt[0] * gp[0] + wt[1] * gp[1] + wt[2] * gp[2];
            dacc += xb[0] * wn[0] + xb[1] * wn[1] + xb[2] * wn[2];
#pragma unroll
            for (int d = 0; d < 3; ++d) { cot_in.p[d][p] = xo[d]; cot_in.p[3 + d][p] = wt[d]; }
        }
#pragma unroll
        for (int f = 0; f < 12; ++f) cur[f] = nxt[f];
    }
    block_sum2_to_global(kacc, dacc, K_b, dtdx_b, sm_red);
}

// Adjoint of the deposit: x_b += m_p sum_cells delta_b(cell) dW/dx_p
__global__ void __launch_bounds__(256) deposit_adj_kernel(const float* __restrict__ db, const float* __restrict__ px,
                                                          const float* __restrict__ py, const float* __restrict__ pz,
                                                          float* __restrict__ xb, float* __restrict__ yb,
                                                          float* __restrict__ zb, int np, int N, float mp) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const Cic8 q = cic8_of(px[p], py[p], pz[p], N);
    const float wy[2] = {1.f - q.fy, q.fy}, wz[2] = {1.f - q.fz, q.fz};
    float a0 = 0.f, a1 = 0.f, a2 = 0.f;
    Gath8 v;
    gather_issue(db, q, v);
    const float xb0 = xb[p], yb0 = yb[p], zb0 = zb[p];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int cz = j >> 1, cy = j & 1;
        const float vlo = v.lo[j], vhi = v.hi[j];
        const float vx = fmaf(q.wx0, vlo, q.wx1 * vhi);
        a0 = fmaf(q.wzy[j], vhi - vlo, a0);
        a1 = fmaf((cy ? 1.f : -1.f) * wz[cz], vx, a1);
        a2 = fmaf((cz ? 1.f : -1.f) * wy[cy], vx, a2);
    }
    xb[p] = fmaf(mp, a0, xb0);
    yb[p] = fmaf(mp, a1, yb0);
    zb[p] = fmaf(mp, a2, zb0);
}

// y += a * x  (float4)
__global__ void axpy_kernel(const float4* __restrict__ x, float4* __restrict__ y, int64_t n4, float a) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; i < n4; i += stride) {
        const float4 u = __ldg(x + i);
        float4 v = y[i];
        v.x = fmaf(a, u.x, v.x); v.y = fmaf(a, u.y, v.y); v.z = fmaf(a, u.z, v.z); v.w = fmaf(a, u.w, v.w);
        y[i] = v;
    }
}

// out += scale * sum_d <a_d, b_d>   (fp64 accumulation across blocks)
__global__ void __launch_bounds__(256) dot3_kernel(const float4* __restrict__ a0, const float4* __restrict__ a1,
                                                   const float4* __restrict__ a2, const float4* __restrict__ b0,
                                                   const float4* __restrict__ b1, const float4* __restrict__ b2,
                                                   int64_t n4, double scale, double* out) {
    __shared__ double smd[32];
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double acc = 0.0;
    for (; i < n4; i += stride) {
        float s = 0.f;
        float4 u = __ldg(a0 + i), v = __ldg(b0 + i);
        s = fmaf(u.x, v.x, s); s = fmaf(u.y, v.y, s); s = fmaf(u.z, v.z, s); s = fmaf(u.w, v.w, s);
        u = __ldg(a1 + i); v = __ldg(b1 + i);
        s = fmaf(u.x, v.x, s); s = fmaf(u.y, v.y, s); s = fmaf(u.z, v.z, s); s = fmaf(u.w, v.w, s);
        u = __ldg(a2 + i); v = __ldg(b2 + i);
        s = fmaf(u.x, v.x, s); s = fmaf(u.y, v.y, s); s = fmaf(u.z, v.z, s); s = fmaf(u.w, v.w, s);
        acc += (double)s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    const int t = threadIdx.x;
    if ((t & 31) == 0) smd[t >> 5] = acc;
    __syncthreads();
    if (t < 32) {
        double v = t < (int)(blockDim.x >> 5) ? smd[t] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (t == 0) atomicAdd(out, scale * v);
    }
}

// ------------------------------------------------------------------------------------------------ launchers ----
static inline unsigned grid_for(int64_t n, int block, int sm_count, int per_sm) {
    int64_t g = (n + block - 1) / block;
    int64_t cap = (int64_t)sm_count * per_sm;
    return (unsigned)(g < cap ? (g > 0 ? g : 1) : cap);
}

// grid of a persistent kernel: as many blocks as are resident on the device at once, never more than there are chunks
template <class Kern>
static int persistent_grid(dh_ctx* c, Kern kern, int threads, int nchunks, unsigned& grid) {
    static int per_sm = 0;      // one per kernel instantiation
    if (per_sm == 0) {
        int n = 0;
        DH_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kern, threads, 0));
        per_sm = n < 1 ? 1 : n;
    }
    const int64_t g = (int64_t)c->sm_count * per_sm;
    grid = (unsigned)(g < nchunks ? g : nchunks);
    return DH_OK;
}

int launch_fill(dh_ctx* c, float* p, int64_t n, float v) {
    Prof prof(c, PROF_FILL);
    fill_kernel<<<grid_for(n, 256, c->sm_count, 8), 256, 0, c->stream>>>(p, n, v);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_cell_index(dh_ctx* c, const float* x, int64_t n, int32_t* i0, int32_t* i1) {
    if (n <= 0) return DH_OK;
    cell_index_kernel<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(x, n, c->N, i0, i1);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_deposit(dh_ctx* c, const float* rho_gas, const float* x, const float* y, const float* z, float* delta,
                   bool primed) {
    const float flag = (c->opt.gas_sources_gravity && rho_gas) ? 1.f : 0.f;
    const int64_t n4 = c->n3 / 4;
    if (!primed) {
        Prof prof(c, PROF_SOURCE_INIT);
        source_init_kernel<<<grid_for(n4, 256, c->sm_count, 8), 256, 0, c->stream>>>(
            reinterpret_cast<const float4*>(flag != 0.f ? rho_gas : nullptr), reinterpret_cast<float4*>(delta), n4, flag,
            (float)c->rho_bar);
        c->launches++;
    }
    DH_CUDA(cudaGetLastError());
    if (c->np > 0) {
        Prof prof(c, PROF_DEPOSIT);
        if (c->tune_deposit_tile && c->nps % TBX == 0 && c->N >= TLX) {
            const dim3 grid(c->nps / TBX, (c->nps + TBY - 1) / TBY, (c->nps + TBZ - 1) / TBZ);
            if (c->tune_deposit_tile == 2)
                deposit_tile_kernel<true><<<grid, 1024, 0, c->stream>>>(x, y, z, c->nps, c->N, (float)c->m_p, delta);
            else
                deposit_tile_kernel<false><<<grid, 1024, 0, c->stream>>>(x, y, z, c->nps, c->N, (float)c->m_p, delta);
        } else {
            deposit_kernel<<<(unsigned)((c->np + 255) / 256), 256, 0, c->stream>>>(x, y, z, (int)c->np, c->N, (float)c->m_p, delta);
        }
        c->launches++;
        DH_CUDA(cudaGetLastError());
    }
    return DH_OK;
}

static float green_coef(const dh_ctx* c, float A) {
    // i k_d A / k^2 with k = (2 pi / L) n  ->  i n_d (A L / 2 pi) / n^2 ; the 1/N^3 normalises the unnormalised cuFFT pair
    return (float)((double)A * c->box / (2.0 * M_PI) / (double)c->n3);
}

int launch_green(dh_ctx* c, const float2* dhat, float A, float2* const ghat[3]) {
    const int64_t nspec = (int64_t)c->N * c->N * (c->N / 2 + 1);
    Prof prof(c, PROF_GREEN);
    green_kernel<<<(unsigned)((nspec + 255) / 256), 256, 0, c->stream>>>(dhat, ghat[0], ghat[1], ghat[2], c->N, nspec,
                                                                          green_coef(c, A));
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_green_adj(dh_ctx* c, float2* const gbhat[3], float A, float2* dbhat) {
    const int64_t nspec = (int64_t)c->N * c->N * (c->N / 2 + 1);
    Prof prof(c, PROF_GREEN_ADJ);
    green_adj_kernel<<<(unsigned)((nspec + 255) / 256), 256, 0, c->stream>>>(gbhat[0], gbhat[1], gbhat[2], dbhat, c->N,
                                                                              nspec, green_coef(c, A));
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int poisson_forward(dh_ctx* c, const float* delta, float A, float* const g_out[3]) {
    if (c->own_fft && c->tune_own_fft) return own_poisson_forward(c, delta, A, g_out);
    {
        Prof prof(c, PROF_FFT_R2C);
        DH_CUFFT(cufftExecR2C(c->plan_r2c, const_cast<float*>(delta), reinterpret_cast<cufftComplex*>(c->spec[0])));
    }
    float2* gh[3] = {c->spec[1], c->spec[2], c->spec[3]};
    DH_TRY(launch_green(c, c->spec[0], A, gh));
    for (int d = 0; d < 3; ++d) {
        Prof prof(c, PROF_FFT_C2R);
        DH_CUFFT(cufftExecC2R(c->plan_c2r, reinterpret_cast<cufftComplex*>(gh[d]), g_out[d]));
    }
    return DH_OK;
}

int poisson_adjoint(dh_ctx* c, float* const g_bar[3], float A, float* delta_bar) {
    if (c->own_fft && c->tune_own_fft) return own_poisson_adjoint(c, g_bar, A, delta_bar);
    float2* gh[3] = {c->spec[1], c->spec[2], c->spec[3]};
    for (int d = 0; d < 3; ++d) {
        Prof prof(c, PROF_FFT_R2C);
        DH_CUFFT(cufftExecR2C(c->plan_r2c, g_bar[d], reinterpret_cast<cufftComplex*>(gh[d])));
    }
    DH_TRY(launch_green_adj(c, gh, A, c->spec[0]));
    {
        Prof prof(c, PROF_FFT_C2R);
        DH_CUFFT(cufftExecC2R(c->plan_c2r, reinterpret_cast<cufftComplex*>(c->spec[0]), delta_bar));
    }
    return DH_OK;
}

int launch_kick_drift(dh_ctx* c, float* const g[3], float* const part[6], float* const part_out[6], float K,
                      float dtau_dx) {
    if (c->np <= 0) return DH_OK;
    const int grav = c->opt.gravity_on && g && g[0];
    Prof prof(c, PROF_KICK_DRIFT);
    const unsigned grid = (unsigned)((c->np + KD_T - 1) / KD_T);
    kick_drift_kernel<<<grid, KD_T, 0, c->stream>>>(
        grav ? g[0] : nullptr, grav ? g[1] : nullptr, grav ? g[2] : nullptr, part[0], part[1], part[2], part[3], part[4],
        part[5], part_out[0], part_out[1], part_out[2], part_out[3], part_out[4], part_out[5], (int)c->np, c->N, K,
        dtau_dx, (float)c->N, 1.f / (float)c->N, grav);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_kick_drift_vjp(dh_ctx* c, float* const g[3], float* const part_in[6], float* const cot_out[6],
                          float* const cot_in[6], float* const gbar[3], float K, float dtau_dx, double* scal_bar) {
    if (c->np <= 0) return DH_OK;
    const int grav = c->opt.gravity_on && g && g[0];
    Prof prof(c, PROF_KICK_DRIFT_ADJ);
    const int nchunks = (int)((c->np + RT - 1) / RT);
    CPtr3 gm; CPtr12 pi; MPtr6 ci; MPtr3 gb;
    for (int d = 0; d < 3; ++d) { gm.p[d] = grav ? g[d] : nullptr; gb.p[d] = grav ? gbar[d] : nullptr; }
    for (int k = 0; k < 6; ++k) { pi.p[k] = part_in[k]; pi.p[6 + k] = cot_out[k]; ci.p[k] = cot_in[k]; }
    unsigned grid;
    if (grav) {
        DH_TRY(persistent_grid(c, kick_drift_adj_kernel<true>, RT, nchunks, grid));
        kick_drift_adj_kernel<true><<<grid, RT, 0, c->stream>>>(gm, pi, ci, gb, (int)c->np, nchunks, c->N, K, dtau_dx,
                                                                 scal_bar + 3, scal_bar + 4);
    } else {
        DH_TRY(persistent_grid(c, kick_drift_adj_kernel<false>, RT, nchunks, grid));
        kick_drift_adj_kernel<false><<<grid, RT, 0, c->stream>>>(gm, pi, ci, gb, (int)c->np, nchunks, c->N, K, dtau_dx,
                                                                  scal_bar + 3, scal_bar + 4);
    }
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

// y += a x over one mesh
int launch_axpy(dh_ctx* c, const float* x, float* y, float a) {
    const int64_t n4 = c->n3 / 4;
    Prof prof(c, PROF_AXPY);
    axpy_kernel<<<grid_for(n4, 256, c->sm_count, 8), 256, 0, c->stream>>>(reinterpret_cast<const float4*>(x),
                                                                         reinterpret_cast<float4*>(y), n4, a);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_deposit_vjp(dh_ctx* c, const float* delta_bar, float* const part_in[6], float* rho_bar_gas,
                       float* const xbar[3]) {
    if (c->opt.gas_sources_gravity && rho_bar_gas) DH_TRY(launch_axpy(c, delta_bar, rho_bar_gas, 1.f));
    if (c->np > 0) {
        Prof prof(c, PROF_DEPOSIT_ADJ);
        deposit_adj_kernel<<<(unsigned)((c->np + 255) / 256), 256, 0, c->stream>>>(
            delta_bar, part_in[0], part_in[1], part_in[2], xbar[0], xbar[1], xbar[2], (int)c->np, c->N, (float)c->m_p);
        c->launches++;
        DH_CUDA(cudaGetLastError());
    }
    return DH_OK;
}

int launch_dot3(dh_ctx* c, float* const a[3], float* const b[3], double scale, double* out) {
    const int64_t n4 = c->n3 / 4;
    Prof prof(c, PROF_DOT3);
    dot3_kernel<<<grid_for(n4, 256, c->sm_count, 4), 256, 0, c->stream>>>(
        reinterpret_cast<const float4*>(a[0]), reinterpret_cast<const float4*>(a[1]), reinterpret_cast<const float4*>(a[2]),
        reinterpret_cast<const float4*>(b[0]), reinterpret_cast<const float4*>(b[1]), reinterpret_cast<const float4*>(b[2]),
        n4, scale, out);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

}  // namespace dh
