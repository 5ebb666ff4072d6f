// scan_static.cu -- mlp_row_offsets_static: the CSR row-offset step of the neighbour build (row counts -> row_ptr, the
// exclusive scan of nbr.cu) as an entry point that ALLOCATES NOTHING, for callers that may not call cudaMalloc (code under
// CUDA graph capture, tight serving loops, harnesses that forbid it).  The block totals the scan needs between its passes
// live in a file-scope device array of fixed size instead of a cudaMalloc'ed buffer.
//
//   - The array is 64 KiB + 256 B; every GPU that loads this library holds it until the process exits.
//   - Limit: n <= MLP_ROW_OFFSETS_STATIC_MAX (67,108,864 rows = 16,384 blocks of 4,096); larger n is MLP_ERR_ARG.
//   - All calls on one device share the array.  It keeps the last call's contents; nothing in it has to start at zero
//     except the 64-bit grand total, which the first kernel of every call clears.  Calls that overlap on the GPU (two
//     streams, two host threads without ordering between them) RACE on it.
//   - In host code `g_scan_scratch` is a host-side stand-in, not a device address.  The address the kernels receive comes
//     from cudaGetSymbolAddress, taken once per device with that device current (scratch_of_current_device()).
//
// mlp_debug_row_offsets runs the EXISTING path (painn::exclusive_scan of nbr.cu with a cudaMalloc'ed block buffer, exactly
// what mlp_compute launches) on caller buffers so that a test can compare the two.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/mlp.h"
#include "common.cuh"

namespace {

constexpr int SS_T = 1024, SS_I = 4, SS_B = SS_T * SS_I;           // same blocking as nbr.cu: 4,096 rows per block
constexpr int SS_MAX_BLOCKS = 16384;                                // 64 KiB of block totals
constexpr int SS_HEAD = 64;                                         // ints before the block totals (256 B): [0..1] = 64-bit total
constexpr long long SS_MAX_N = (long long)SS_MAX_BLOCKS * SS_B;
static_assert(SS_MAX_N == MLP_ROW_OFFSETS_STATIC_MAX, "header and kernel disagree on the limit");

static __device__ __align__(256) int g_scan_scratch[SS_HEAD + SS_MAX_BLOCKS];

constexpr int SS_MAX_DEVICES = 64;
std::mutex g_mu;
int* g_scratch_ptr[SS_MAX_DEVICES] = {};

// Device address of g_scan_scratch on the CURRENT device (one cudaGetSymbolAddress per device, no allocation).
int scratch_of_current_device(int** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= SS_MAX_DEVICES) return MLP_ERR_CUDA;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_scan_scratch) != cudaSuccess || !p) { cudaGetLastError(); return MLP_ERR_CUDA; }
        g_scratch_ptr[dev] = static_cast<int*>(p);
    }
    *out = g_scratch_ptr[dev];
    return MLP_OK;
}

__device__ __forceinline__ int ss_block_scan(int v, int* total) {   // exclusive scan over the 1024 threads of a block
    __shared__ int wsum[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
        int s = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
        wsum[lane] = s;
    }
    __syncthreads();
    const int base = w ? wsum[w - 1] : 0;
    *total = wsum[31];
    __syncthreads();                                                 // wsum is reused by the next call in the same kernel
    return base + x - v;
}

// pass 1: scan inside blocks of 4,096 rows; block totals -> scratch[SS_HEAD + block]
__global__ void __launch_bounds__(SS_T) k_ss_block(const int* __restrict__ in, int* __restrict__ out, long long n,
                                                   int* __restrict__ scratch) {
    if (blockIdx.x == 0 && threadIdx.x == 0) *reinterpret_cast<long long*>(scratch) = 0;   // the word that must start at zero
    const long long base = (long long)blockIdx.x * SS_B + (long long)threadIdx.x * SS_I;
    int v[SS_I], s = 0;
#pragma unroll
    for (int k = 0; k < SS_I; k++) { v[k] = (base + k < n) ? in[base + k] : 0; s += v[k]; }
    int tot;
    int ex = ss_block_scan(s, &tot);
#pragma unroll
    for (int k = 0; k < SS_I; k++) { if (base + k < n) out[base + k] = ex; ex += v[k]; }
    if (threadIdx.x == 0) scratch[SS_HEAD + blockIdx.x] = tot;
}
// pass 2 (one block): exclusive scan of the block totals in place, 64-bit grand total -> scratch[0..1] and *total
__global__ void __launch_bounds__(SS_T) k_ss_tops(int* __restrict__ scratch, int nb, long long* __restrict__ total) {
    __shared__ long long carry_s;
    if (threadIdx.x == 0) carry_s = *reinterpret_cast<long long*>(scratch);   // 0, written by pass 1 of this call
    __syncthreads();
    int* block_tot = scratch + SS_HEAD;
    for (int b0 = 0; b0 < nb; b0 += SS_T) {
        const int b = b0 + threadIdx.x;
        const int v = b < nb ? block_tot[b] : 0;
        int tot;
        const int ex = ss_block_scan(v, &tot);
        const long long carry = carry_s;
        if (b < nb) block_tot[b] = (int)(carry + ex);
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *reinterpret_cast<long long*>(scratch) = carry_s;
        if (total) *total = carry_s;
    }
}
// pass 3: add the scanned block totals; out[n] = grand total
__global__ void k_ss_add(int* __restrict__ out, long long n, const int* __restrict__ scratch) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) out[i] += scratch[SS_HEAD + i / SS_B];
    if (i == n) out[n] = (int)*reinterpret_cast<const long long*>(scratch);
}

}  // namespace

#define MLP_EXPORT extern "C" __attribute__((visibility("default")))

MLP_EXPORT int mlp_row_offsets_static(const int* counts, int* offsets, long long n, long long* total, void* cuda_stream) {
    if (n < 0 || !offsets || (n > 0 && !counts)) return MLP_ERR_ARG;
    if (n > SS_MAX_N) return MLP_ERR_ARG;                            // beyond the static scratch: see mlp.h
    int* scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != MLP_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    long long nb = (n + SS_B - 1) / SS_B;
    if (nb < 1) nb = 1;
    k_ss_block<<<(unsigned)nb, SS_T, 0, st>>>(counts, offsets, n, scratch);
    k_ss_tops<<<1, SS_T, 0, st>>>(scratch, (int)nb, total);
    k_ss_add<<<(unsigned)((n + 1 + 255) / 256), 256, 0, st>>>(offsets, n, scratch);
    return cudaGetLastError() == cudaSuccess ? MLP_OK : MLP_ERR_CUDA;
}

MLP_EXPORT int mlp_debug_row_offsets(const int* counts, int* offsets, long long n, long long* total, void* cuda_stream) {
    if (n < 0 || !offsets || !total || (n > 0 && !counts)) return MLP_ERR_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int* tmp = nullptr;
    if (cudaMalloc(&tmp, (size_t)(n / SS_B + 2) * sizeof(int)) != cudaSuccess) { cudaGetLastError(); return MLP_ERR_NOMEM; }
    long long launches = 0;
    painn::Launch L{st, &launches};
    painn::exclusive_scan(L, counts, offsets, n, tmp, total);        // the three kernels mlp_compute launches (nbr.cu)
    const cudaError_t e1 = cudaGetLastError(), e2 = cudaStreamSynchronize(st);
    cudaFree(tmp);
    return (e1 == cudaSuccess && e2 == cudaSuccess) ? MLP_OK : MLP_ERR_CUDA;
}
