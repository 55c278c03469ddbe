// subgrid.cu -- the sub-grid star-formation / energy-injection step (section 2.4, :226-283; SURVEY.md 8(f)
// NEXT-2) and its transpose, for sm_100a.  Pointwise over the mesh, one pass each:
//   delta = rho / rho_mean - 1,  T = t_per_e (eps/rho - |m|^2 / (2 rho^2))
//   pi0 = Pi0 sigma((delta - delta_c)/a) sigma((T_c - T)/b)                                     Eq. 25 (:279)
//   z   = sigma(((log pi0 + g0) - (log(1 - pi0) + g1)) / tau)     relaxed Bernoulli of Eq. 24 (:265), g0, g1 ~ Gumbel(0,1)
//         are INPUTS (the reparametrisation of Eq. 22-23); evaluated through its log-odds so that tau = 0.1 cannot overflow
//   eps += e_inject rho z                                                    energy injection into the cell (:236)
// plus the cloud-in-cell readout of the star-forming field z at the particle positions into their auxiliary variable
// (:244, diagnostic only).  Forward: 20 + 8 B/cell in, 4 + 4 out; transpose: 20 + 8 + 20 (+ 4) in, 20 out + 4 scalars.
// Readings R29-R32 of DESIGN.md section 16.  Product code: shares nothing with oracle/.
#include "dh_internal.cuh"

namespace dh {

struct SgConst {
    float inv_rho_mean, t_per_e, T_c, delta_c, log_Pi0, inv_Pi0, e_inject, inv_a, inv_b, inv_tau;
};
struct SgGas { float* p[5]; };
struct SgGasC { const float* p[5]; };

// log sigma(x) and sigma(-x), stable for any x
__device__ __forceinline__ void log_sigmoid(float x, float& ls, float& s_neg) {
    const float e = __expf(-fabsf(x));                // in (0, 1]
    const float l1p = log1pf(e);
    ls = -(fmaxf(-x, 0.f) + l1p);
    const float r = 1.f / (1.f + e);
    s_neg = x >= 0.f ? e * r : r;                     // sigma(-x)
}

struct SgPoint { float z, zc, pi0, sx, sy; };          // z, 1 - z, pi0, sigma(-x), sigma(-y)

__device__ __forceinline__ SgPoint sg_point(float rho, float m0, float m1, float m2, float eps, float g0, float g1,
                                            const SgConst& k) {
    const float rinv = 1.f / rho;
    const float ke = 0.5f * (m0 * m0 + m1 * m1 + m2 * m2) * rinv;
    const float T = k.t_per_e * ((eps - ke) * rinv);          // the order of prim_GH (sweep_common.cuh): one cancellation
    const float x = (rho * k.inv_rho_mean - 1.f - k.delta_c) * k.inv_a;
    const float y = (k.T_c - T) * k.inv_b;
    float lx, ly;
    SgPoint q;
    log_sigmoid(x, lx, q.sx);
    log_sigmoid(y, ly, q.sy);
    const float ell = k.log_Pi0 + lx + ly;
    q.pi0 = __expf(ell);
    const float u = (ell - log1pf(-q.pi0) + g0 - g1) * k.inv_tau;
    const float eu = __expf(-fabsf(u)), ru = 1.f / (1.f + eu);
    q.z = u >= 0.f ? ru : eu * ru;                    // sigma(u) and sigma(-u) without cancellation on either side
    q.zc = u >= 0.f ? eu * ru : ru;
    return q;
}

__global__ void __launch_bounds__(256) subgrid_fwd_kernel(SgGas gas, const float* __restrict__ g0,
                                                          const float* __restrict__ g1, float* __restrict__ zout,
                                                          int64_t n, SgConst k) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float rho = gas.p[0][i], eps = gas.p[4][i];
        const SgPoint q = sg_point(rho, gas.p[1][i], gas.p[2][i], gas.p[3][i], eps, __ldg(g0 + i), __ldg(g1 + i), k);
        gas.p[4][i] = fmaf(k.e_inject * rho, q.z, eps);
        if (zout) zout[i] = q.z;
    }
}

// cot (5 arrays): in = cotangent of the step's output, out = cotangent of its input (in place); scal += (dT_c, ddelta_c,
// dPi0, de_inject) in fp64
__global__ void __launch_bounds__(256) subgrid_adj_kernel(SgGasC gas, const float* __restrict__ g0,
                                                          const float* __restrict__ g1, SgGas cot,
                                                          const float* __restrict__ cot_z, int64_t n, SgConst k,
                                                          double* scal) {
    __shared__ double sm[4][8];
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float rho = __ldg(gas.p[0] + i), eps = __ldg(gas.p[4] + i);
        const float m[3] = {__ldg(gas.p[1] + i), __ldg(gas.p[2] + i), __ldg(gas.p[3] + i)};
        const SgPoint q = sg_point(rho, m[0], m[1], m[2], eps, __ldg(g0 + i), __ldg(g1 + i), k);
        const float eb_out = cot.p[4][i];
        const float z_b = fmaf(eb_out * k.e_inject, rho, cot_z ? __ldg(cot_z + i) : 0.f);
        const float ell_b = z_b * q.z * q.zc * k.inv_tau / (1.f - q.pi0);
        const float x_b = ell_b * q.sx, y_b = ell_b * q.sy;
        const float rinv = 1.f / rho;
        const float e_b = -y_b * k.inv_b * k.t_per_e;                       // cotangent of e~
        const float m2 = m[0] * m[0] + m[1] * m[1] + m[2] * m[2];
        float rho_b = eb_out * k.e_inject * q.z + x_b * k.inv_a * k.inv_rho_mean +
                      e_b * (m2 * rinv - eps) * rinv * rinv;
        cot.p[0][i] += rho_b;
        const float mc = -e_b * rinv * rinv;
        cot.p[1][i] += mc * m[0]; cot.p[2][i] += mc * m[1]; cot.p[3][i] += mc * m[2];
        cot.p[4][i] = eb_out + e_b * rinv;
        acc[0] += (double)(y_b * k.inv_b);
        acc[1] -= (double)(x_b * k.inv_a);
        acc[2] += (double)(ell_b * k.inv_Pi0);
        acc[3] += (double)(eb_out * rho * q.z);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[j] += __shfl_xor_sync(0xffffffffu, acc[j], o);
        if ((threadIdx.x & 31) == 0) sm[j][threadIdx.x >> 5] = acc[j];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double v = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += sm[threadIdx.x][w];
        atomicAdd(scal + threadIdx.x, v);
    }
}

// aux_p += sum_cells W(x_p - cell) z(cell): the CIC readout of :244 with the weights of pm.cu (s = x - 1/2)
__global__ void __launch_bounds__(256) cic_readout_kernel(const float* __restrict__ mesh, const float* __restrict__ px,
                                                          const float* __restrict__ py, const float* __restrict__ pz,
                                                          float* __restrict__ aux, int np, int N) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    int i0[3], i1[3];
    float f[3];
    const float pos[3] = {px[p], py[p], pz[p]};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const float s = pos[d] - 0.5f, fl = floorf(s);
        f[d] = s - fl;
        int i = (int)fl;
        i = i < 0 ? i + N : i;
        i = i >= N ? i - N : i;
        i0[d] = i; i1[d] = (i + 1 == N) ? 0 : i + 1;
    }
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const int ix = (c & 1) ? i1[0] : i0[0], iy = (c & 2) ? i1[1] : i0[1], iz = (c & 4) ? i1[2] : i0[2];
        const float w = ((c & 1) ? f[0] : 1.f - f[0]) * ((c & 2) ? f[1] : 1.f - f[1]) * ((c & 4) ? f[2] : 1.f - f[2]);
        acc = fmaf(w, __ldg(mesh + ((size_t)iz * N + iy) * N + ix), acc);
    }
    aux[p] += acc;
}

static SgConst sg_const(const dh_subgrid_params& q) {
    SgConst k;
    k.inv_rho_mean = (float)(1.0 / q.rho_mean); k.t_per_e = (float)q.t_per_e; k.T_c = (float)q.T_c;
    k.delta_c = (float)q.delta_c; k.log_Pi0 = (float)log(q.Pi0); k.inv_Pi0 = (float)(1.0 / q.Pi0);
    k.e_inject = (float)q.e_inject; k.inv_a = (float)(1.0 / q.a_width); k.inv_b = (float)(1.0 / q.b_width);
    k.inv_tau = (float)(1.0 / q.tau);
    return k;
}

static unsigned sg_grid(const dh_ctx* c) {
    const int64_t blocks = (c->n3 + 255) / 256, cap = (int64_t)c->sm_count * 8;
    return (unsigned)(blocks < cap ? blocks : cap);
}

int launch_subgrid(dh_ctx* c, float* const gas[5], const float* g0, const float* g1, const dh_subgrid_params& q,
                   float* zout) {
    SgGas g;
    for (int k = 0; k < 5; ++k) g.p[k] = gas[k];
    subgrid_fwd_kernel<<<sg_grid(c), 256, 0, c->stream>>>(g, g0, g1, zout, c->n3, sg_const(q));
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_subgrid_vjp(dh_ctx* c, float* const gas_in[5], const float* g0, const float* g1, const dh_subgrid_params& q,
                       float* const cot[5], const float* cot_z, double* scal4_dev) {
    SgGasC g; SgGas ct;
    for (int k = 0; k < 5; ++k) { g.p[k] = gas_in[k]; ct.p[k] = cot[k]; }
    subgrid_adj_kernel<<<sg_grid(c), 256, 0, c->stream>>>(g, g0, g1, ct, cot_z, c->n3, sg_const(q), scal4_dev);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_cic_readout(dh_ctx* c, const float* mesh, float* const pos[3], float* aux) {
    if (c->np <= 0) return DH_OK;
    cic_readout_kernel<<<(unsigned)((c->np + 255) / 256), 256, 0, c->stream>>>(mesh, pos[0], pos[1], pos[2], aux, (int)c->np,
                                                                              c->N);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

}  // namespace dh
