// dh_conserved_sums_noalloc: the conserved-sums diagnostic (dh_conserved_sums, api.cu) for callers that may not
// allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It takes no context
// (dh_init allocates), calls no cudaMalloc / cudaFree / allocating library routine, does not synchronise, and keeps its
// scratch -- one 64-byte partial sum per block and a block counter -- in a file-scope device array of fixed size that
// every GPU loading this library holds until the process exits.
//
// One launch: block b < nbc sums chunk b (CHUNK cells) of the five gas fields, block nbc + j sums chunk j of the three
// particle velocities, each in fp64, and writes its eight partial sums to its own slot of the scratch; the block that
// finishes last (a counter in the scratch, __threadfence on both sides) adds the slots in slot order and writes the
// eight results.  The order of every addition is fixed by the sizes alone: the same bits on every call and every GPU,
// where dh_conserved_sums (one fp64 atomicAdd per block) is only reproducible to rounding.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "../../include/diffhydro.h"
#include "dh_internal.cuh"

namespace dh {
namespace {

constexpr int NA_THREADS = 256;
constexpr int64_t NA_CHUNK = 32768;                                              // elements of one array per block
constexpr int64_t NA_MAX_BLOCKS = 2 * (DH_NOALLOC_MAX_ELEMS / NA_CHUNK);         // cells + particles at the maximum: 8192
constexpr size_t NA_SLOT_DOUBLES = 8;
// [0, 8 * NA_MAX_BLOCKS): the slots; then one double-sized cell whose first 4 bytes are the counter of finished blocks
constexpr size_t NA_SCRATCH_DOUBLES = NA_SLOT_DOUBLES * NA_MAX_BLOCKS + 1;       // 512 KiB + 8 B

// In host code this name is a host-side stand-in, not a device address: the launch below passes what
// cudaGetSymbolAddress returned for it.
static __device__ __align__(256) double g_noalloc_scratch[NA_SCRATCH_DOUBLES];

struct NaPtrs { const float* gas[5]; const float* w[3]; };

__device__ __forceinline__ double block_sum_fixed(double v, double* sm /* [NA_THREADS / 32] */) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();                                     // the previous use of sm is over
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < NA_THREADS / 32; ++w) t += sm[w];
    return t;                                            // valid in thread 0
}

__global__ void __launch_bounds__(NA_THREADS) conserved_sums_noalloc_kernel(NaPtrs a, int64_t n_cells, int64_t n_part,
                                                                            int nbc, int nbp, double m_p,
                                                                            double* __restrict__ scratch,
                                                                            double* __restrict__ out) {
    __shared__ double sm[NA_THREADS / 32];
    __shared__ bool s_last;
    unsigned int* const counter = reinterpret_cast<unsigned int*>(scratch + NA_SLOT_DOUBLES * NA_MAX_BLOCKS);
    const int b = blockIdx.x;
    const bool cells = b < nbc;
    const int64_t n = cells ? n_cells : n_part;
    const int64_t i0 = (int64_t)(cells ? b : b - nbc) * NA_CHUNK;
    const int64_t i1 = i0 + NA_CHUNK < n ? i0 + NA_CHUNK : n;
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (cells) {
        for (int64_t i = i0 + threadIdx.x; i < i1; i += NA_THREADS)
#pragma unroll
            for (int k = 0; k < 5; ++k) acc[k] += (double)__ldg(a.gas[k] + i);
    } else {
        for (int64_t i = i0 + threadIdx.x; i < i1; i += NA_THREADS)
#pragma unroll
            for (int k = 0; k < 3; ++k) acc[k] += (double)__ldg(a.w[k] + i);
    }
    double* const slot = scratch + NA_SLOT_DOUBLES * (size_t)b;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const double t = block_sum_fixed(acc[k], sm);
        if (threadIdx.x == 0) slot[k] = t;               // a particle block fills [0, 3); [3, 5) are zeros nobody reads
    }
    // ---- the block that arrives last adds the slots, in slot order
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int done = atomicAdd(counter, 1u);
        s_last = (done == (unsigned int)(nbc + nbp) - 1u);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double tot[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int j = threadIdx.x; j < nbc; j += NA_THREADS) {
        const volatile double* s = scratch + NA_SLOT_DOUBLES * (size_t)j;
#pragma unroll
        for (int k = 0; k < 5; ++k) tot[k] += s[k];
    }
    for (int j = threadIdx.x; j < nbp; j += NA_THREADS) {
        const volatile double* s = scratch + NA_SLOT_DOUBLES * (size_t)(nbc + j);
#pragma unroll
        for (int k = 0; k < 3; ++k) tot[5 + k] += s[k];
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const double t = block_sum_fixed(tot[k], sm);
        if (threadIdx.x == 0) out[k] = k < 5 ? t : m_p * t;
    }
    if (threadIdx.x == 0) *counter = 0u;                 // the next call on this device starts from zero again
}

// set-up, once per device, with that device current: the device address of the scratch array
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
double* g_na_ptr[NA_MAX_DEVICES] = {};

int noalloc_scratch(double** ptr) {
    int dev = -1;
    DH_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) { set_error("dh_conserved_sums_noalloc: device ordinal %d not supported", dev); return DH_ERR_INVALID; }
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
        double* p = nullptr;
        DH_CUDA(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
        if (!p) { set_error("dh_conserved_sums_noalloc: cudaGetSymbolAddress returned a null address"); return DH_ERR_CUDA; }
        g_na_ptr[dev] = p;
    }
    *ptr = g_na_ptr[dev];
    return DH_OK;
}

}  // namespace
}  // namespace dh

extern "C" int dh_conserved_sums_noalloc(const float* const gas[5], int64_t n_cells, const float* const w[3], int64_t n_part,
                                         double m_p, double* out, void* cuda_stream) {
    using namespace dh;
    if (!gas || !out || n_cells <= 0 || n_part < 0 || (n_part > 0 && !w)) {
        set_error("dh_conserved_sums_noalloc: bad argument (gas, out non-null; n_cells > 0; n_part >= 0; w non-null when n_part > 0)");
        return DH_ERR_INVALID;
    }
    if (n_cells > DH_NOALLOC_MAX_ELEMS || n_part > DH_NOALLOC_MAX_ELEMS) {
        set_error("dh_conserved_sums_noalloc: %lld cells / %lld particles exceed the static scratch's maximum of %lld each "
                  "(DH_NOALLOC_MAX_ELEMS = 512^3); use dh_conserved_sums",
                  (long long)n_cells, (long long)n_part, (long long)DH_NOALLOC_MAX_ELEMS);
        return DH_ERR_INVALID;
    }
    NaPtrs a;
    for (int k = 0; k < 5; ++k) {
        if (!gas[k]) { set_error("dh_conserved_sums_noalloc: gas[%d] is null", k); return DH_ERR_INVALID; }
        a.gas[k] = gas[k];
    }
    for (int k = 0; k < 3; ++k) {
        a.w[k] = n_part > 0 ? w[k] : nullptr;
        if (n_part > 0 && !w[k]) { set_error("dh_conserved_sums_noalloc: w[%d] is null", k); return DH_ERR_INVALID; }
    }
    double* scratch = nullptr;
    DH_TRY(noalloc_scratch(&scratch));
    const int nbc = (int)((n_cells + NA_CHUNK - 1) / NA_CHUNK);
    const int nbp = (int)((n_part + NA_CHUNK - 1) / NA_CHUNK);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // the counter must start at zero whatever an earlier, failed call left behind (a memset node, no allocation)
    DH_CUDA(cudaMemsetAsync(scratch + NA_SLOT_DOUBLES * NA_MAX_BLOCKS, 0, sizeof(double), stream));
    conserved_sums_noalloc_kernel<<<(unsigned)(nbc + nbp), NA_THREADS, 0, stream>>>(a, n_cells, n_part, nbc, nbp, m_p, scratch, out);
    DH_CUDA(cudaGetLastError());
    return DH_OK;
}
