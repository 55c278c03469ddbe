// ic.cu -- the initial-condition map  delta_init -> (gas, particles)  and its transpose, for sm_100a (SURVEY.md 8(f)
// NEXT-1: the step on the input side of the path, so that "gradient w.r.t. the initial density field" is one
// device-resident call).
//
// What is computed (section 2.1: initial conditions by Lagrangian perturbation theory; reading R19 of
// DESIGN.md takes first order, the Zel'dovich map, of a given density contrast at the starting scale factor):
//   psi_d = IFFT3( i k~_d delta^(k) / k^2 )      -- the Poisson solve of fft.cu / pm.cu with A = 1 (div psi = -delta)
//   x_p = wrap(q_p + psi(q_p) / dx),  w_p = vf psi(q_p)          q_p = centre of cell p, one particle per cell
//   rho = f_b (1 + delta),  m = rho vf psi,  eps = rho (e0 + vf^2 |psi|^2 / 2)
// and the transpose of its Jacobian: rho_b, psi_b pointwise, then  delta_b = f_b rho_b + G^T psi_b  with the Poisson
// adjoint.  Both pointwise kernels are one pass over the mesh: 16 B/cell in + 44 out, and 60 in + 16 out.
// Product code: shares nothing with oracle/.
#include "dh_internal.cuh"

namespace dh {

__device__ __forceinline__ float wrap_unit(float x, float fN) {
    x = x < 0.f ? x + fN : x;
    return x >= fN ? x - fN : x;
}

struct IcOut { float* gas[5]; float* part[6]; };
struct IcCot { const float* gas[5]; const float* part[6]; };

// one thread per cell; |psi| / dx < N is assumed (a displacement of a whole box is not an initial condition)
__global__ void __launch_bounds__(256) ic_state_kernel(const float* __restrict__ delta, const float* __restrict__ px,
                                                       const float* __restrict__ py, const float* __restrict__ pz,
                                                       IcOut out, int N, float inv_dx, float vf, float f_b, float e0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int n3 = N * N * N;
    if (i >= n3) return;
    const int x = i % N, y = (i / N) % N, z = i / (N * N);
    const float d = __ldg(delta + i);
    const float p0 = __ldg(px + i), p1 = __ldg(py + i), p2 = __ldg(pz + i);
    const float fN = (float)N;
    out.part[0][i] = wrap_unit(fmaf(p0, inv_dx, (float)x + 0.5f), fN);
    out.part[1][i] = wrap_unit(fmaf(p1, inv_dx, (float)y + 0.5f), fN);
    out.part[2][i] = wrap_unit(fmaf(p2, inv_dx, (float)z + 0.5f), fN);
    const float v0 = vf * p0, v1 = vf * p1, v2 = vf * p2;
    out.part[3][i] = v0; out.part[4][i] = v1; out.part[5][i] = v2;
    const float rho = f_b * (1.f + d);
    out.gas[0][i] = rho;
    out.gas[1][i] = rho * v0; out.gas[2][i] = rho * v1; out.gas[3][i] = rho * v2;
    out.gas[4][i] = rho * fmaf(0.5f, v0 * v0 + v1 * v1 + v2 * v2, e0);
}

// transpose: grad[i] = f_b rho_b (the Poisson adjoint of psi_b is added afterwards), psib_d[i] = psi_b,d
__global__ void __launch_bounds__(256) ic_state_adj_kernel(const float* __restrict__ delta, const float* __restrict__ px,
                                                           const float* __restrict__ py, const float* __restrict__ pz,
                                                           IcCot cot, float* __restrict__ grad, float* __restrict__ bx,
                                                           float* __restrict__ by, float* __restrict__ bz, int n3,
                                                           float inv_dx, float vf, float f_b, float e0) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    const float d = __ldg(delta + i);
    const float v[3] = {vf * __ldg(px + i), vf * __ldg(py + i), vf * __ldg(pz + i)};
    const float rho = f_b * (1.f + d);
    const float c0 = __ldg(cot.gas[0] + i), c4 = __ldg(cot.gas[4] + i);
    const float cm[3] = {__ldg(cot.gas[1] + i), __ldg(cot.gas[2] + i), __ldg(cot.gas[3] + i)};
    const float rho_b = c0 + (cm[0] * v[0] + cm[1] * v[1] + cm[2] * v[2]) +
                        c4 * fmaf(0.5f, v[0] * v[0] + v[1] * v[1] + v[2] * v[2], e0);
    grad[i] = f_b * rho_b;
    float* const pb[3] = {bx, by, bz};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float v_b = rho * fmaf(c4, v[k], cm[k]);                       // from m = rho v and eps = rho (e0 + v^2 / 2)
        const float xb = cot.part[k] ? __ldg(cot.part[k] + i) : 0.f;        // x = q + psi / dx (wrap: derivative 1)
        const float wb = cot.part[3 + k] ? __ldg(cot.part[3 + k] + i) : 0.f;
        pb[k][i] = fmaf(vf, v_b + wb, xb * inv_dx);
    }
}

int launch_ic_state(dh_ctx* c, const float* delta, float* const psi[3], float* const gas[5], float* const part[6],
                    float vf, float e0) {
    IcOut o;
    for (int k = 0; k < 5; ++k) o.gas[k] = gas[k];
    for (int k = 0; k < 6; ++k) o.part[k] = part[k];
    ic_state_kernel<<<(unsigned)((c->n3 + 255) / 256), 256, 0, c->stream>>>(delta, psi[0], psi[1], psi[2], o, c->N,
                                                                            (float)(1.0 / c->dx), vf, (float)c->f_b, e0);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

int launch_ic_state_vjp(dh_ctx* c, const float* delta, float* const psi[3], const float* const cot_gas[5],
                        const float* const cot_part[6], float* grad, float* const psi_b[3], float vf, float e0) {
    IcCot q;
    for (int k = 0; k < 5; ++k) q.gas[k] = cot_gas[k];
    for (int k = 0; k < 6; ++k) q.part[k] = cot_part ? cot_part[k] : nullptr;
    ic_state_adj_kernel<<<(unsigned)((c->n3 + 255) / 256), 256, 0, c->stream>>>(
        delta, psi[0], psi[1], psi[2], q, grad, psi_b[0], psi_b[1], psi_b[2], (int)c->n3, (float)(1.0 / c->dx), vf,
        (float)c->f_b, e0);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

}  // namespace dh

// ------------------------------------------------------------------------------------------------ data term ----
// The output end of the path: the noise-weighted squared error of Eq. 27,
//   L = weight * sum_i (scale * O_i - d_i)^2 / N_i,    Eq. 27: weight = 1/2,
// and its cotangent w.r.t. the gas state, in one pass (20 + 4 [+ 4] B/cell in, 20 out).  Observable O:
//   0: gas density rho                                   (the loss of BASELINE.json's configs 0, 2-4, reading R21)
//   1: internal energy density eps - |m|^2 / (2 rho)     ("delta_b T ... corresponds roughly to the internal energy
//      density of the field"; = a^2 rho e in the tilde variables, the constant goes into `scale`)
// The prior term of Eq. 27 acts on the input phases and is not part of this kernel.
namespace dh {

struct Gas5c { const float* p[5]; };
struct Gas5m { float* p[5]; };

template <int OBS, bool COT>
__global__ void __launch_bounds__(256) data_term_kernel(Gas5c gas, const float* __restrict__ data,
                                                        const float* __restrict__ noise_var, Gas5m cot, int64_t n,
                                                        float scale, float weight, double* loss) {
    __shared__ double sm[8];
    double acc = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const float rho = __ldg(gas.p[0] + i);
        float obs, m[3] = {0.f, 0.f, 0.f}, rinv = 0.f;
        if (OBS == 0) {
            obs = rho;
        } else {
            rinv = 1.f / rho;
            m[0] = __ldg(gas.p[1] + i); m[1] = __ldg(gas.p[2] + i); m[2] = __ldg(gas.p[3] + i);
            obs = __ldg(gas.p[4] + i) - 0.5f * (m[0] * m[0] + m[1] * m[1] + m[2] * m[2]) * rinv;
        }
        const float r = fmaf(scale, obs, -__ldg(data + i));
        const float iv = noise_var ? 1.f / __ldg(noise_var + i) : 1.f;
        acc += (double)(r * r * iv);
        if (COT) {
            const float ob = 2.f * weight * scale * r * iv;          // dL / dO_i
            if (OBS == 0) {
                cot.p[0][i] = ob; cot.p[1][i] = 0.f; cot.p[2][i] = 0.f; cot.p[3][i] = 0.f; cot.p[4][i] = 0.f;
            } else {
                cot.p[0][i] = ob * 0.5f * (m[0] * m[0] + m[1] * m[1] + m[2] * m[2]) * rinv * rinv;
                cot.p[1][i] = -ob * m[0] * rinv; cot.p[2][i] = -ob * m[1] * rinv; cot.p[3][i] = -ob * m[2] * rinv;
                cot.p[4][i] = ob;
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) atomicAdd(loss, (double)weight * v);
    }
}

int launch_data_term(dh_ctx* c, int observable, const float* const gas[5], const float* data, const float* noise_var,
                     float scale, float weight, float* const cot[5], double* loss_dev) {
    Gas5c g; Gas5m q;
    for (int k = 0; k < 5; ++k) { g.p[k] = gas[k]; q.p[k] = cot ? cot[k] : nullptr; }
    const int64_t n = c->n3;
    int64_t blocks = (n + 255) / 256;
    const int64_t cap = (int64_t)c->sm_count * 8;
    const unsigned grid = (unsigned)(blocks < cap ? blocks : cap);
    if (observable == 0) {
        if (cot) data_term_kernel<0, true><<<grid, 256, 0, c->stream>>>(g, data, noise_var, q, n, scale, weight, loss_dev);
        else data_term_kernel<0, false><<<grid, 256, 0, c->stream>>>(g, data, noise_var, q, n, scale, weight, loss_dev);
    } else {
        if (cot) data_term_kernel<1, true><<<grid, 256, 0, c->stream>>>(g, data, noise_var, q, n, scale, weight, loss_dev);
        else data_term_kernel<1, false><<<grid, 256, 0, c->stream>>>(g, data, noise_var, q, n, scale, weight, loss_dev);
    }
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

// out[k] += sum_i a_k[i], k < NA: fp64 accumulation per thread, warp and block, one atomic per block and array
struct SumPtrs { const float* p[8]; };
__global__ void __launch_bounds__(256) sum_arrays_kernel(SumPtrs a, int na, int64_t n, double* out) {
    __shared__ double sm[8][8];
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        for (int k = 0; k < na; ++k) acc[k] += (double)__ldg(a.p[k] + i);
    for (int k = 0; k < na; ++k) {
        double v = acc[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) sm[k][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        for (int k = 0; k < na; ++k) {
            double v = threadIdx.x < (blockDim.x >> 5) ? sm[k][threadIdx.x] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (threadIdx.x == 0) atomicAdd(out + k, v);
        }
    }
}

int launch_sum_arrays(dh_ctx* c, const float* const* arrays, int na, int64_t n, double* out_dev) {
    if (na <= 0 || n <= 0) return DH_OK;
    SumPtrs a;
    for (int k = 0; k < 8; ++k) a.p[k] = k < na ? arrays[k] : nullptr;
    int64_t blocks = (n + 255) / 256;
    const int64_t cap = (int64_t)c->sm_count * 8;
    sum_arrays_kernel<<<(unsigned)(blocks < cap ? blocks : cap), 256, 0, c->stream>>>(a, na, n, out_dev);
    c->launches++;
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}

}  // namespace dh
