// gemm_tc.cu -- tcgen05 / TMEM / TMA path of the per-atom linear layers (sm_100a only).
//
//   C[M x N] (+)= A[M x K] . W[N x K]^T + bias            A, C fp32 row-major, W fixed weights
//
// Precision: the F = 128 PaiNN models of BASELINE.json are badly conditioned with N(0, 1/fan_in) weights (feature
// growth through un-normalised neighbour sums); single-pass TF32 or BF16 operands miss the force tolerance by
// ~10x (measured).  The tensor-core path therefore runs error-compensated "3xTF32":
//   a = a_hi + a_lo (both exactly representable in TF32, round-to-nearest),  w likewise (split once at create),
//   a.w ~= a_hi w_hi + a_hi w_lo + a_lo w_hi      (fp32 accumulation in TMEM; dropped term ~2^-22 relative).
// Structure (one persistent CTA per SM, warp-specialised, mbarrier pipelines):
//   warp 0      TMA producer : A tile (raw fp32), W_hi, W_lo tiles, 32-wide K blocks, SWIZZLE_128B, 3-4 stages
//   warps 2-5   converter    : A raw -> A_hi (in place) and A_lo (second buffer), element-wise (layout-agnostic),
//                              then fence.proxy.async so the tensor core sees the generic-proxy writes
//   warp 1      MMA issuer   : one elected thread, tcgen05.mma.kind::tf32 M=128 x N=BN x K=8, 12 MMAs per K block,
//                              tcgen05.commit frees the smem stage / publishes the accumulator
//   warps 6-9   epilogue     : tcgen05.ld 32x32b (one TMEM lane = one output row per thread), + bias (+ C), st.global
// The accumulator is double-buffered in TMEM (2 x BN columns), so the epilogue of tile t overlaps the MMAs of t+1.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>

#include "common.cuh"
#include "tc_common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

namespace tc {

constexpr int BM = 128, BK = 32;                       // 32 fp32 = 128 B = one swizzle row
constexpr int NUM_THREADS = 320;                       // 10 warps
constexpr int CONV_WARP0 = 2, EPI_WARP0 = 6;
constexpr int A_TILE_BYTES = BM * BK * 4;              // 16 KB

// K-major, SWIZZLE_128B shared-memory matrix descriptor: rows of 128 B, 8-row groups 1024 B apart
__device__ __forceinline__ uint64_t make_desc_sw128(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3ffff) >> 4) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
__device__ __forceinline__ float rn_tf32(float x) {
    uint32_t u = __float_as_uint(x);
    u += 0xfffu + ((u >> 13) & 1u);
    return __uint_as_float(u & 0xffffe000u);
}

struct Params {
    float* C;
    const float* bias;
    long long M;
    int N, K, ldc, accumulate;
};

template <int BN, int STAGES>
struct Smem {
    static constexpr int B_TILE = BN * BK * 4;
    static constexpr int STAGE = 2 * A_TILE_BYTES + 2 * B_TILE;
    static constexpr int BYTES = STAGES * STAGE + 1024 /*align*/ + 256 /*barriers*/;
};

template <int BN, int STAGES>
__global__ void __launch_bounds__(NUM_THREADS, 1)
    k_gemm_3xtf32(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapWhi,
                  const __grid_constant__ CUtensorMap mapWlo, Params p) {
    using S = Smem<BN, STAGES>;
    // declared aligned (no run-time pointer rounding: that would hide the shared address space from the compiler
    // and turn every LDS / STS into a generic LD / ST)
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t* bars = (uint64_t*)(smem + STAGES * S::STAGE);
    uint64_t* full = bars;                   // TMA landed            (count 1 + tx)
    uint64_t* conv = bars + STAGES;          // A converted           (count 128)
    uint64_t* empty = bars + 2 * STAGES;     // MMAs of the stage done (count 1, tcgen05.commit)
    uint64_t* tfull = bars + 3 * STAGES;     // accumulator ready     (count 1, tcgen05.commit)  [2]
    uint64_t* tempty = tfull + 2;            // accumulator drained   (count 4)                  [2]
    uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_tiles = p.N / BN;
    const long long m_tiles = (p.M + BM - 1) / BM;
    const long long total = m_tiles * n_tiles;
    const int kblocks = p.K / BK;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; s++) { mbar_init(&full[s], 1); mbar_init(&conv[s], 128); mbar_init(&empty[s], 1); }
        for (int b = 0; b < 2; b++) { mbar_init(&tfull[b], 1); mbar_init(&tempty[b], 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                     "r"(2 * BN));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (long long t = blockIdx.x; t < total; t += gridDim.x) {
                const int m0 = (int)(t / n_tiles) * BM, n0 = (int)(t % n_tiles) * BN;
                for (int kb = 0; kb < kblocks; kb++) {
                    mbar_wait(&empty[stage], phase ^ 1);
                    uint8_t* st = smem + stage * S::STAGE;
                    mbar_expect_tx(&full[stage], A_TILE_BYTES + 2 * S::B_TILE);
                    tma_load_2d(st, &mapA, &full[stage], kb * BK, m0);
                    tma_load_2d(st + 2 * A_TILE_BYTES, &mapWhi, &full[stage], kb * BK, n0);
                    tma_load_2d(st + 2 * A_TILE_BYTES + S::B_TILE, &mapWlo, &full[stage], kb * BK, n0);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
            int stage = 0;
            uint32_t phase = 0;
            int buf = 0;
            uint32_t bphase = 0;
            for (long long t = blockIdx.x; t < total; t += gridDim.x) {
                mbar_wait(&tempty[buf], bphase ^ 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t d = tmem_base + buf * BN;
                for (int kb = 0; kb < kblocks; kb++) {
                    mbar_wait(&conv[stage], phase);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint32_t sa = smem_u32(smem + stage * S::STAGE);
                    const uint64_t a_hi = make_desc_sw128(sa), a_lo = make_desc_sw128(sa + A_TILE_BYTES);
                    const uint64_t w_hi = make_desc_sw128(sa + 2 * A_TILE_BYTES),
                                   w_lo = make_desc_sw128(sa + 2 * A_TILE_BYTES + S::B_TILE);
#pragma unroll
                    for (int kk = 0; kk < BK / 8; kk++) {
                        const uint64_t o = (uint64_t)(kk * 2);   // 32 B along K inside the swizzle row, >> 4
                        umma_tf32(d, a_lo + o, w_hi + o, idesc, (kb | kk) != 0);
                        umma_tf32(d, a_hi + o, w_lo + o, idesc, 1);
                        umma_tf32(d, a_hi + o, w_hi + o, idesc, 1);
                    }
                    umma_commit(&empty[stage]);
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
                umma_commit(&tfull[buf]);
                if (++buf == 2) { buf = 0; bphase ^= 1; }
            }
        }
    } else if (warp < EPI_WARP0) {
        // ===================== converter: A -> (A_hi in place, A_lo) =====================
        const int ct = threadIdx.x - CONV_WARP0 * 32;   // 0..127
        int stage = 0;
        uint32_t phase = 0;
        for (long long t = blockIdx.x; t < total; t += gridDim.x) {
            for (int kb = 0; kb < kblocks; kb++) {
                mbar_wait(&full[stage], phase);
                float4* a = (float4*)(smem + stage * S::STAGE);
                float4* al = (float4*)(smem + stage * S::STAGE + A_TILE_BYTES);
#pragma unroll
                for (int i = 0; i < A_TILE_BYTES / 16 / 128; i++) {
                    const int idx = ct + i * 128;
                    float4 x = a[idx], h, l;
                    h.x = rn_tf32(x.x); h.y = rn_tf32(x.y); h.z = rn_tf32(x.z); h.w = rn_tf32(x.w);
                    l.x = rn_tf32(x.x - h.x); l.y = rn_tf32(x.y - h.y); l.z = rn_tf32(x.z - h.z); l.w = rn_tf32(x.w - h.w);
                    a[idx] = h;
                    al[idx] = l;
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_arrive(&conv[stage]);
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // ===================== epilogue =====================
        const int q = warp & 3;                      // TMEM lane quadrant this warp may access
        int buf = 0;
        uint32_t bphase = 0;
        for (long long t = blockIdx.x; t < total; t += gridDim.x) {
            const long long m0 = (t / n_tiles) * BM;
            const int n0 = (int)(t % n_tiles) * BN;
            mbar_wait(&tfull[buf], bphase);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const long long row = m0 + q * 32 + lane;
            float* crow = p.C + row * p.ldc + n0;
#pragma unroll 1
            for (int c0 = 0; c0 < BN; c0 += 32) {
                uint32_t r[32];
                float4 o[8];
                // accumulate: issue all residual loads of this 32-column chunk BEFORE waiting on TMEM, so they are
                // in flight together (a load -> add -> store chain per float4 serialises on DRAM latency)
                if (p.accumulate && row < p.M) {
#pragma unroll
                    for (int c = 0; c < 8; c++) o[c] = __ldcs((const float4*)(crow + c0) + c);
                }
                tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + buf * BN + c0, r);
                if (row < p.M) {
#pragma unroll
                    for (int c = 0; c < 32; c += 4) {
                        float4 v = make_float4(__uint_as_float(r[c]), __uint_as_float(r[c + 1]), __uint_as_float(r[c + 2]),
                                               __uint_as_float(r[c + 3]));
                        if (p.bias) {
                            const float4 b = *(const float4*)(p.bias + n0 + c0 + c);
                            v.x += b.x; v.y += b.y; v.z += b.z; v.w += b.w;
                        }
                        if (p.accumulate) { v.x += o[c / 4].x; v.y += o[c / 4].y; v.z += o[c / 4].z; v.w += o[c / 4].w; }
                        *(float4*)(crow + c0 + c) = v;
                    }
                }
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&tempty[buf]);
            if (++buf == 2) { buf = 0; bphase ^= 1; }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 1) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(2 * BN));
    }
}

// ---- host side: tensor maps through the driver entry point (no link-time dependency on libcuda) ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}
static bool make_map(CUtensorMap* map, const float* ptr, long long rows, int cols, int ld, int box_rows) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)ld * 4};
    cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int BN, int STAGES>
static bool launch(const Launch& L, const CUtensorMap& a, const CUtensorMap& whi, const CUtensorMap& wlo, Params p,
                   int n_sm) {
    using S = Smem<BN, STAGES>;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_gemm_3xtf32<BN, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::BYTES) != cudaSuccess)
            return false;
        attr_set = true;
    }
    const long long total = ((p.M + BM - 1) / BM) * (p.N / BN);
    int grid = (int)(total < n_sm ? total : n_sm);
    k_gemm_3xtf32<BN, STAGES><<<grid, NUM_THREADS, S::BYTES, L.stream>>>(a, whi, wlo, p);
    KLAUNCH(L);
    return true;
}

}  // namespace tc

// Returns false when the shape is not covered (caller falls back to the SIMT path).
bool gemm_nt_tc(const Launch& L, const float* A, int lda, const float* Whi, const float* Wlo, int ldw, float* C, int ldc,
                long long M, int N, int K, const float* bias, bool accumulate) {
    using namespace tc;
    if (M <= 0 || K % BK != 0 || K < BK || (lda % 4) || (ldw % 4) || (ldc % 4)) return false;
    if (((uintptr_t)A | (uintptr_t)Whi | (uintptr_t)Wlo | (uintptr_t)C) & 15) return false;
    const int BN = (N % 128 == 0) ? 128 : (N % 64 == 0 ? 64 : 0);
    if (!BN) return false;
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    CUtensorMap ma, mh, ml;
    if (!make_map(&ma, A, M, K, lda, BM) || !make_map(&mh, Whi, N, K, ldw, BN) || !make_map(&ml, Wlo, N, K, ldw, BN))
        return false;
    Params p{C, bias, M, N, K, ldc, accumulate ? 1 : 0};
    if (BN == 128) return launch<128, 3>(L, ma, mh, ml, p, n_sm);
    return launch<64, 4>(L, ma, mh, ml, p, n_sm);
}

}  // namespace painn
