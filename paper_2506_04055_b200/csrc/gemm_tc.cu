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
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <unordered_map>
#include <vector>
#include <algorithm>

#include "common.cuh"
#include "tc_common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

namespace tc {

constexpr int BM = 128, BK = 32;                       // 32 fp32 = 128 B = one swizzle row
constexpr int NUM_THREADS = 320;                       // 10 warps
constexpr int CONV_WARP0 = 2, EPI_WARP0 = 6;
constexpr int A_TILE_BYTES = BM * BK * 4;              // 16 KB
constexpr int EPI_LD = 36;                             // staging row stride in floats: 16-byte rows of a quarter-warp fall into distinct banks

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
    const float* dsilu_pre;    // optional [M x N] (row stride ld_pre): C = (A W^T + bias) * SiLU'(pre), fused adjoint of the activation
    int ld_pre;
    const float* resid;        // accumulate: the term added to A W^T (row stride ldc); C itself for an in-place accumulation
};
__device__ __forceinline__ float dsilu_x(float x) {
    const float sg = __fdividef(1.0f, 1.0f + __expf(-x));     // adjoint only: 2 ulp (forces carry a relative tolerance)
    return sg * (1.0f + x * (1.0f - sg));
}

template <int BN, int STAGES>
struct Smem {
    static constexpr int B_TILE = BN * BK * 4;
    static constexpr int STAGE = 2 * A_TILE_BYTES + 2 * B_TILE;
    static constexpr int EPI = 4 * 32 * EPI_LD * 4;     // epilogue staging: one [32 rows][32 columns (+4)] fp32 tile per warp
    static constexpr int BYTES = STAGES * STAGE + 1024 /*align*/ + 256 /*barriers*/ + EPI;
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
                    // the same block of this CTA's next unit goes to L2 now: only STAGES blocks (48 KB) can be in
                    // flight to shared memory, too few to cover the DRAM latency at full bandwidth
                    if (t + gridDim.x < total) {
                        const int m1 = (int)((t + gridDim.x) / n_tiles) * BM;
                        if (m1 != m0)
                            asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global [%0, {%1, %2}];" ::"l"(&mapA), "r"(kb * BK),
                                         "r"(m1)
                                         : "memory");
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer: converged warp, one elected lane issues =====================
        {
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
                    if (elect_one()) {
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
                        if (kb == kblocks - 1) umma_commit(&tfull[buf]);
                    }
                    __syncwarp();
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
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
        // tcgen05.ld hands every thread one ROW of the tile; global accesses in that layout touch 32 different lines per
        // instruction (32 LSU wavefronts each, measured: the LSU data pipe was the busiest unit of this kernel).  Each
        // warp therefore turns its 32 x 32 chunk through a private shared-memory tile and does all global traffic
        // (residual / SiLU' argument loads, stores) with a quarter-warp per 128-byte row segment.
        const int q = warp & 3;                      // TMEM lane quadrant this warp may access
        float* stg = (float*)(smem + STAGES * S::STAGE + 256) + q * 32 * EPI_LD;
        const int sub = lane >> 3, c4 = (lane & 7) * 4;          // coalesced phase: row i * 4 + sub, columns c4 .. c4 + 3
        int buf = 0;
        uint32_t bphase = 0;
        for (long long t = blockIdx.x; t < total; t += gridDim.x) {
            const long long m0 = (t / n_tiles) * BM;
            const int n0 = (int)(t % n_tiles) * BN;
            mbar_wait(&tfull[buf], bphase);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const long long row0 = m0 + q * 32 + sub;
#pragma unroll 1
            for (int c0 = 0; c0 < BN; c0 += 32) {
                uint32_t r[32];
                float4 o[8];
                // issue all residual loads of this chunk BEFORE waiting on TMEM, so they are in flight together
                if (p.accumulate) {
#pragma unroll
                    for (int i = 0; i < 8; i++)
                        if (row0 + 4 * i < p.M) o[i] = __ldcs((const float4*)(p.resid + (row0 + 4 * i) * p.ldc + n0 + c0 + c4));
                } else if (p.dsilu_pre) {     // (never combined with accumulate)
#pragma unroll
                    for (int i = 0; i < 8; i++)
                        if (row0 + 4 * i < p.M)
                            o[i] = __ldcs((const float4*)(p.dsilu_pre + (row0 + 4 * i) * p.ld_pre + n0 + c0 + c4));
                }
                float4 b4 = make_float4(0.f, 0.f, 0.f, 0.f);
                if (p.bias) b4 = *(const float4*)(p.bias + n0 + c0 + c4);
                tmem_ld32(tmem_base + ((uint32_t)(q * 32) << 16) + buf * BN + c0, r);
#pragma unroll
                for (int c = 0; c < 8; c++)
                    *(float4*)(stg + lane * EPI_LD + 4 * c) = make_float4(__uint_as_float(r[4 * c]), __uint_as_float(r[4 * c + 1]),
                                                                          __uint_as_float(r[4 * c + 2]), __uint_as_float(r[4 * c + 3]));
                __syncwarp();
#pragma unroll
                for (int i = 0; i < 8; i++) {
                    float4 v = *(const float4*)(stg + (4 * i + sub) * EPI_LD + c4);
                    v.x += b4.x; v.y += b4.y; v.z += b4.z; v.w += b4.w;
                    if (row0 + 4 * i < p.M) {
                        if (p.accumulate) { v.x += o[i].x; v.y += o[i].y; v.z += o[i].z; v.w += o[i].w; }
                        else if (p.dsilu_pre) {
                            v.x *= dsilu_x(o[i].x); v.y *= dsilu_x(o[i].y); v.z *= dsilu_x(o[i].z); v.w *= dsilu_x(o[i].w);
                        }
                        *(float4*)(p.C + (row0 + 4 * i) * p.ldc + n0 + c0 + c4) = v;
                    }
                }
                __syncwarp();
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

// =================================================================================================================
// k_gemm_exact: error-free tensor-core GEMM for the FORWARD linear layers (K = 128 per launch).
//
// tcgen05.mma truncates its fp32 accumulator toward zero after every instruction (B3), a systematic bias the
// energy cannot absorb.  Truncation is harmless when every partial sum is exactly representable, so the operands are
// cut into INTEGER slices (block floating point per row, Ozaki-style):
//     x'_mk = x_mk / 2^e_m  in (-1, 1)      x' ~= (s1 + s2 2^-8 + s3 2^-16) / 128 ,   s_i integers in [-128, 128]
// (weights likewise, sliced once at create: t1, t2, t3 and 2^f_n).  Every slice value is exact in TF32, every product
// |s t| <= 2^14, a K = 128 chain of up to three slice pairs stays below 2^24: each accumulator holds an exact integer.
//     y_mn = 2^(e_m + f_n - 14) ( S2 + S3 2^-8 + S4 2^-16 ),   S_g = sum over slice pairs i + j = g of  s_i . t_j
// (pairs with i + j >= 5 are dropped: relative 2^-22 of row max x column max, unbiased).  Three accumulators per
// output tile; 24 MMAs (M = 128, N = 64, K = 8) per 32-wide K block.
// Each output tile walks its K blocks twice: pass 0 streams A through the ring to find the row maxima (exponents
// e_m), pass 1 streams A (an L2 hit) and the weight slices again, converts A into its three slices in shared memory
// and runs the MMAs.  Same warp roles and barriers as k_gemm_3xtf32; ACT applies SiLU to A while converting.
constexpr int XBN = 32, XWST = 4, XRAW = 3;
constexpr int XTHREADS = NUM_THREADS + 32;                              // + warp 10: second TMA producer (raw A blocks)
constexpr int XW_TILE = XBN * 128;                                      // 4 KB: 32 rows x 64 fp16 (one slice, one K half)
constexpr int XW_STAGE = 3 * 2 * XW_TILE;                               // 24 KB: the three weight slices of one N tile, K = 128
constexpr int XNMAX = 512;                                              // widest N (column scale and bias are staged in shared memory)
constexpr int XSMEM = XRAW * A_TILE_BYTES + XWST * XW_STAGE + 4 * BM * 4 + 2 * XNMAX * 4 + 256 + 4 * 32 * EPI_LD * 4 + 1024;
constexpr int XTM_A = 0;                                                // TMEM columns 0..255: A slices [4][64 columns = 128 fp16]
constexpr int XTM_ACC = 256, XACC = 4 * XBN;                            // TMEM columns 256..511: 2 accumulator sets (S2..S5 x 32)

struct XParams {
    float* C;
    const float* bias;
    const float* colscale;     // [N] 2^f_n
    long long M;
    int N, ldc, accumulate;
};

// x sigmoid(x) with the approximate reciprocal (2 ulp, same order as __expf): the converter warps evaluate it twice per
// element (row maximum, then slicing) and the IEEE division made them the bottleneck of the act launches (1.14 -> 0.8 ms)
__device__ __forceinline__ float silu_x(float x) { return __fdividef(x, 1.0f + __expf(-x)); }
__device__ __forceinline__ void tmem_st16x(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
        "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void umma_f16_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(tmem_d),
        "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(acc)
        : "memory");
}

// Work unit = one 128-row block of A with ALL its N tiles.  The raw fp32 blocks of A stream twice through a small
// ring (pass 0: row maxima -> exponents; pass 1: conversion, an L2 hit).  The fp16 integer slices of the whole block
// (K = 128) are written straight into TENSOR MEMORY (one row per lane, tcgen05.st) and stay there while the N tiles
// run: the MMAs take A from TMEM and only the small weight-slice tiles from shared memory (with A in shared memory the
// kernel was bound by re-reading 4 KB of A for every N = 64 MMA: 85 cycles per MMA instead of 32).
template <bool ACT>
__global__ void __launch_bounds__(XTHREADS, 1)
    k_gemm_exact(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapW1,
                 const __grid_constant__ CUtensorMap mapW2, const __grid_constant__ CUtensorMap mapW3, XParams p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* raw = smem;                                              // [XRAW] raw A blocks (128 rows x 32 fp32, SWIZZLE_128B)
    uint8_t* wst = raw + XRAW * A_TILE_BYTES;                         // [XWST] weight-slice stages
    float* rowscale = (float*)(wst + XWST * XW_STAGE);                // [4][BM]  2^(e_m - 14) of the last four units
    float* s_cs = rowscale + 4 * BM;                                  // [N] column scales 2^f_n
    float* s_bias = s_cs + XNMAX;                                     // [N] bias (zeros when absent)
    uint64_t* bars = (uint64_t*)(s_bias + XNMAX);
    uint64_t* rfull = bars;                   // [XRAW] raw block landed          (count 1 + tx)
    uint64_t* rempty = rfull + XRAW;          // [XRAW] raw block consumed        (count 128)
    uint64_t* wfull = rempty + XRAW;          // [XWST] weight slices landed      (count 1 + tx)
    uint64_t* wempty = wfull + XWST;          // [XWST] MMAs of the stage done    (count 1, tcgen05.commit)
    uint64_t* sl_ready = wempty + XWST;       // [1] A slices of the unit written (count 128)
    uint64_t* sl_free = sl_ready + 1;         // [1] all MMAs of the unit done    (count 1, tcgen05.commit)
    uint64_t* tfull = sl_free + 1;            // [2] accumulators ready           (count 1)
    uint64_t* tempty = tfull + 2;             // [2] accumulators drained         (count 4)
    uint32_t* tmem_slot = (uint32_t*)(tempty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_tiles = p.N / XBN;
    const long long units = (p.M + BM - 1) / BM;
    constexpr int kblocks = 128 / BK;         // 4 raw blocks per pass

    if (threadIdx.x == 0) {
        for (int s = 0; s < XRAW; s++) { mbar_init(&rfull[s], 1); mbar_init(&rempty[s], 128); }
        for (int s = 0; s < XWST; s++) { mbar_init(&wfull[s], 1); mbar_init(&wempty[s], 1); }
        mbar_init(sl_ready, 128); mbar_init(sl_free, 1);
        for (int b = 0; b < 2; b++) { mbar_init(&tfull[b], 1); mbar_init(&tempty[b], 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) tmem_alloc(tmem_slot, 512);
    for (int i = threadIdx.x; i < p.N; i += XTHREADS) { s_cs[i] = p.colscale[i]; s_bias[i] = p.bias ? p.bias[i] : 0.0f; }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {
            // ===================== TMA producer 1: weight slices =====================
            int ws = 0;
            uint32_t wphase = 0;
            for (long long u = blockIdx.x; u < units; u += gridDim.x)
                for (int nt = 0; nt < n_tiles; nt++) {
                    mbar_wait(&wempty[ws], wphase ^ 1);
                    uint8_t* st = wst + ws * XW_STAGE;
                    mbar_expect_tx(&wfull[ws], XW_STAGE);
#pragma unroll
                    for (int kh = 0; kh < 2; kh++) {
                        tma_load_2d(st + (0 * 2 + kh) * XW_TILE, &mapW1, &wfull[ws], kh * 64, nt * XBN);
                        tma_load_2d(st + (1 * 2 + kh) * XW_TILE, &mapW2, &wfull[ws], kh * 64, nt * XBN);
                        tma_load_2d(st + (2 * 2 + kh) * XW_TILE, &mapW3, &wfull[ws], kh * 64, nt * XBN);
                    }
                    if (++ws == XWST) { ws = 0; wphase ^= 1; }
                }
        }
    } else if (warp == 10) {
        // The two TMA producers must not share a warp: UTMALDG / SYNCS run on the warp's uniform datapath, and two
        // divergent spinning lanes of one warp clobbered each other's uniform registers (measured: ~2 % of the pass-0
        // blocks landed with wrong coordinates).
        if (lane == 0) {
            // ===================== TMA producer 2: raw A blocks, twice per unit =====================
            int rs = 0;
            uint32_t rphase = 0;
            for (long long u = blockIdx.x; u < units; u += gridDim.x)
                for (int e = 0; e < 2 * kblocks; e++) {
                    // pull the next unit's rows into L2 while this unit is processed (its pass 0 is then an L2 hit too)
                    if (e < kblocks && u + gridDim.x < units)
                        asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global [%0, {%1, %2}];" ::"l"(&mapA), "r"(e * BK),
                                     "r"((int)(u + gridDim.x) * BM)
                                     : "memory");
                    mbar_wait(&rempty[rs], rphase ^ 1);
                    mbar_expect_tx(&rfull[rs], A_TILE_BYTES);
                    tma_load_2d(raw + rs * A_TILE_BYTES, &mapA, &rfull[rs], (e & (kblocks - 1)) * BK, (int)u * BM);
                    if (++rs == XRAW) { rs = 0; rphase ^= 1; }
                }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer: the warp stays converged, one elected lane issues =====================
        {
            const uint32_t idesc = (1u << 4) | ((uint32_t)(XBN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);   // f16 x f16 -> f32
            const uint32_t ta = tmem_base + XTM_A;
            int ws = 0;
            uint32_t wphase = 0, uphase = 0;
            int buf = 0;
            uint32_t bphase = 0;
            for (long long u = blockIdx.x; u < units; u += gridDim.x) {
                mbar_wait(sl_ready, uphase);
                tc_fence_after();
                for (int nt = 0; nt < n_tiles; nt++) {
                    mbar_wait(&tempty[buf], bphase ^ 1);
                    mbar_wait(&wfull[ws], wphase);
                    tc_fence_after();
                    const uint32_t d = tmem_base + XTM_ACC + buf * XACC;
                    const uint32_t sw = smem_u32(wst + ws * XW_STAGE);
                    if (elect_one()) {
#pragma unroll
                        for (int kh = 0; kh < 2; kh++) {
                            uint64_t w[3];
#pragma unroll
                            for (int i = 0; i < 3; i++) w[i] = make_desc_sw128(sw + (i * 2 + kh) * XW_TILE);
#pragma unroll
                            for (int kk = 0; kk < 4; kk++) {             // 16 fp16 along K = 8 TMEM columns of A, 32 B of a W row
                                const uint64_t o = (uint64_t)(kk * 2);
                                const uint32_t a0 = ta + kh * 32 + kk * 8, a1 = a0 + 64, a2 = a0 + 128, a3 = a0 + 192;
                                const uint32_t acc = (kh | kk) != 0;
                                // S2: (1,1)   S3: (1,2) (2,1)   S4: (1,3) (2,2) (3,1)   S5: (2,3) (3,2) (4,1)
                                umma_f16_ts(d, a0, w[0] + o, idesc, acc);
                                umma_f16_ts(d + XBN, a0, w[1] + o, idesc, acc);
                                umma_f16_ts(d + 2 * XBN, a0, w[2] + o, idesc, acc);
                                umma_f16_ts(d + 3 * XBN, a1, w[2] + o, idesc, acc);
                                umma_f16_ts(d + XBN, a1, w[0] + o, idesc, 1);
                                umma_f16_ts(d + 2 * XBN, a1, w[1] + o, idesc, 1);
                                umma_f16_ts(d + 3 * XBN, a2, w[1] + o, idesc, 1);
                                umma_f16_ts(d + 2 * XBN, a2, w[0] + o, idesc, 1);
                                umma_f16_ts(d + 3 * XBN, a3, w[0] + o, idesc, 1);
                            }
                        }
                        umma_commit(&wempty[ws]);
                        umma_commit(&tfull[buf]);
                        if (nt == n_tiles - 1) umma_commit(sl_free);
                    }
                    __syncwarp();
                    if (++ws == XWST) { ws = 0; wphase ^= 1; }
                    if (++buf == 2) { buf = 0; bphase ^= 1; }
                }
                uphase ^= 1;
            }
        }
    } else if (warp < EPI_WARP0) {
        // ===================== converter: one row per thread (= TMEM lane) =====================
        // SWIZZLE_128B stores logical 16-byte chunk c of row r at chunk c ^ (r & 7): reading the chunks in logical order is
        // conflict-free for the 8 consecutive rows of a quarter-warp.
        const int row = (warp & 3) * 32 + lane;
        const uint32_t trow = tmem_base + XTM_A + ((uint32_t)((warp & 3) * 32) << 16);
        const int rx = row & 7;
        int rs = 0;
        uint32_t rphase = 0, uphase = 0;
        uint32_t ucount = 0;
        const float MAGIC = 12582912.0f;                // 1.5 * 2^23: (t + MAGIC) - MAGIC = round-to-nearest-even integer
        for (long long u = blockIdx.x; u < units; u += gridDim.x, ucount++) {
            float mx = 0.f;
            for (int kb = 0; kb < kblocks; kb++) {
                mbar_wait(&rfull[rs], rphase);
                const float4* a = (const float4*)(raw + rs * A_TILE_BYTES + row * 128);
#pragma unroll
                for (int c = 0; c < 8; c++) {
                    float4 x = a[c ^ rx];
                    if (ACT) { x.x = silu_x(x.x); x.y = silu_x(x.y); x.z = silu_x(x.z); x.w = silu_x(x.w); }
                    mx = fmaxf(mx, fmaxf(fmaxf(fabsf(x.x), fabsf(x.y)), fmaxf(fabsf(x.z), fabsf(x.w))));
                }
                // Release to the TMA producer.  The refill is an ASYNC-proxy write to bytes this thread has just read through
                // the generic proxy: without a proxy fence the two are not ordered even across the mbarrier (measured: ~2 %
                // of the rows saw part of the next block in pass 0 and got a different, still valid, exponent run to run).
                asm volatile("" ::"f"(mx) : "memory");
                fence_async_smem();
                mbar_arrive(&rempty[rs]);
                if (++rs == XRAW) { rs = 0; rphase ^= 1; }
            }
            // 2^e = smallest power of two > max |x|; non-finite / huge rows fall through as garbage / NaN downstream
            const uint32_t E = (__float_as_uint(mx) >> 23) & 0xffu;      // mx in [2^(E-127), 2^(E-126))
            const uint32_t Ec = E < 20u ? 20u : (E > 230u ? 230u : E);   // keep every scale a normal number
            const float q128 = __uint_as_float((260u - Ec) << 23);       // 128 / 2^e
            rowscale[(ucount & 3) * BM + row] = __uint_as_float((Ec - 13u) << 23);   // 2^(e - 14)
            mbar_wait(sl_free, uphase ^ 1);              // the previous unit's MMAs no longer read the slices
            uphase ^= 1;
            tc_fence_after();
            for (int kb = 0; kb < kblocks; kb++) {
                mbar_wait(&rfull[rs], rphase);
                const float4* a = (const float4*)(raw + rs * A_TILE_BYTES + row * 128);
                uint32_t h1[16], h2[16], h3[16], h4[16];   // 32 K values x 4 slices, two fp16 per TMEM column
#pragma unroll
                for (int c = 0; c < 8; c++) {
                    const float4 v = a[c ^ rx];
                    const float x[4] = {v.x, v.y, v.z, v.w};
                    float s1[4], s2[4], s3[4], s4[4];
#pragma unroll
                    for (int j = 0; j < 4; j++) {
                        const float xv = ACT ? silu_x(x[j]) : x[j];
                        const float t1 = xv * q128;
                        s1[j] = (t1 + MAGIC) - MAGIC;
                        const float t2 = (t1 - s1[j]) * 256.0f;
                        s2[j] = (t2 + MAGIC) - MAGIC;
                        const float t3 = (t2 - s2[j]) * 256.0f;
                        s3[j] = (t3 + MAGIC) - MAGIC;
                        const float t4 = (t3 - s3[j]) * 256.0f;
                        s4[j] = (t4 + MAGIC) - MAGIC;
                    }
#pragma unroll
                    for (int j = 0; j < 2; j++) {
                        __half2 p1 = __floats2half2_rn(s1[2 * j], s1[2 * j + 1]), p2 = __floats2half2_rn(s2[2 * j], s2[2 * j + 1]),
                                p3 = __floats2half2_rn(s3[2 * j], s3[2 * j + 1]), p4 = __floats2half2_rn(s4[2 * j], s4[2 * j + 1]);
                        h1[2 * c + j] = *(uint32_t*)&p1; h2[2 * c + j] = *(uint32_t*)&p2; h3[2 * c + j] = *(uint32_t*)&p3;
                        h4[2 * c + j] = *(uint32_t*)&p4;
                    }
                }
                fence_async_smem();                      // cross-proxy release of the raw block (see pass 0)
                mbar_arrive(&rempty[rs]);
                if (++rs == XRAW) { rs = 0; rphase ^= 1; }
                tmem_st16x(trow + kb * 16, h1);
                tmem_st16x(trow + 64 + kb * 16, h2);
                tmem_st16x(trow + 128 + kb * 16, h3);
                tmem_st16x(trow + 192 + kb * 16, h4);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            tc_fence_before();
            mbar_arrive(sl_ready);
        }
    } else if (warp < 10) {
        // ===================== epilogue =====================
        // combine and scale in the TMEM layout (thread = row), then turn the 32 x 32 tile through a private shared-memory
        // tile so that the residual loads and the stores are coalesced (see k_gemm_3xtf32)
        const int q = warp & 3;                      // TMEM lane quadrant this warp may access
        float* stg = (float*)((uint8_t*)bars + 256) + q * 32 * EPI_LD;
        const int sub = lane >> 3, c4 = (lane & 7) * 4;
        int buf = 0;
        uint32_t bphase = 0;
        uint32_t ucount = 0;
        for (long long u = blockIdx.x; u < units; u += gridDim.x, ucount++) {
            const long long row0 = u * BM + q * 32 + sub;
            for (int nt = 0; nt < n_tiles; nt++) {
                const int n0 = nt * XBN;
                float4 o[8];
                if (p.accumulate) {
#pragma unroll
                    for (int i = 0; i < 8; i++)
                        if (row0 + 4 * i < p.M) o[i] = __ldcs((const float4*)(p.C + (row0 + 4 * i) * p.ldc + n0 + c4));
                }
                mbar_wait(&tfull[buf], bphase);
                tc_fence_after();
                const float rs = rowscale[(ucount & 3) * BM + q * 32 + lane];
                const uint32_t tb = tmem_base + XTM_ACC + ((uint32_t)(q * 32) << 16) + buf * XACC;
#pragma unroll
                for (int c0 = 0; c0 < XBN; c0 += 16) {
                    uint32_t r2[16], r3[16], r4[16], r5[16];
                    tmem_ld16_nowait(tb + c0, r2);
                    tmem_ld16_nowait(tb + XBN + c0, r3);
                    tmem_ld16_nowait(tb + 2 * XBN + c0, r4);
                    tmem_ld16_nowait(tb + 3 * XBN + c0, r5);
                    tmem_wait_ld();
                    if (c0 + 16 == XBN) {                // last read of this accumulator set: hand it back before the stores
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&tempty[buf]);
                    }
#pragma unroll
                    for (int c = 0; c < 16; c += 4) {
                        const float4 cs = *(const float4*)(s_cs + n0 + c0 + c);
                        float v[4];
#pragma unroll
                        for (int j = 0; j < 4; j++) {
                            const float lo = fmaf(__uint_as_float(r5[c + j]), 1.0f / 256.0f, __uint_as_float(r4[c + j]));
                            v[j] = fmaf(lo, 1.0f / 65536.0f, fmaf(__uint_as_float(r3[c + j]), 1.0f / 256.0f, __uint_as_float(r2[c + j])));
                        }
                        float4 y = make_float4(v[0] * (rs * cs.x), v[1] * (rs * cs.y), v[2] * (rs * cs.z), v[3] * (rs * cs.w));
                        const float4 b = *(const float4*)(s_bias + n0 + c0 + c);
                        y.x += b.x; y.y += b.y; y.z += b.z; y.w += b.w;
                        *(float4*)(stg + lane * EPI_LD + c0 + c) = y;
                    }
                }
                __syncwarp();
#pragma unroll
                for (int i = 0; i < 8; i++) {
                    float4 y = *(const float4*)(stg + (4 * i + sub) * EPI_LD + c4);
                    if (row0 + 4 * i < p.M) {
                        if (p.accumulate) { y.x += o[i].x; y.y += o[i].y; y.z += o[i].z; y.w += o[i].w; }
                        *(float4*)(p.C + (row0 + 4 * i) * p.ldc + n0 + c4) = y;
                    }
                }
                __syncwarp();
                if (++buf == 2) { buf = 0; bphase ^= 1; }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, 512);
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

// fp16 weight-slice plane [rows x 128], box = 64 halfs (128 B, one swizzle row) x box_rows
static bool make_map16(CUtensorMap* map, const __half* ptr, int rows, int box_rows) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t dims[2] = {128, (cuuint64_t)rows};
    cuuint64_t strides[1] = {128 * 2};
    cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, (void*)ptr, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
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

// ---- exact integer-slice path: weight slices are cut once, at create ----
// (ExactW in common.cuh: planes = device [K / 128][3][N][128] integer-valued fp16 slices t1, t2, t3; cs = device
//  [K / 128][N] column scales 2^f_n.)  The registry belongs to the model.
void gemm_register_exact(GemmRegistry& reg, const float* Wdev, const float* Whost, int N, int K) {
    if (K % 128 != 0 || N % tc::XBN != 0 || reg.exact.count(Wdev)) return;
    const int nc = K / 128;
    std::vector<__half> pl((size_t)nc * 3 * N * 128);
    std::vector<float> cs((size_t)nc * N);
    for (int c = 0; c < nc; c++)
        for (int n = 0; n < N; n++) {
            const float* w = Whost + (size_t)n * K + c * 128;
            float m = 0.f;
            for (int k = 0; k < 128; k++) m = std::fmax(m, std::fabs(w[k]));
            int ex = 0;
            if (m > 0.f) std::frexp(m, &ex);               // m = f 2^ex, f in [0.5, 1)  ->  |w| < 2^ex
            ex = std::min(104, std::max(-106, ex));
            const float q128 = std::ldexp(1.0f, 7 - ex);
            cs[(size_t)c * N + n] = std::ldexp(1.0f, ex);
            for (int k = 0; k < 128; k++) {
                const float t1 = w[k] * q128;
                const float s1 = std::nearbyint(t1);
                const float t2 = (t1 - s1) * 256.0f;
                const float s2 = std::nearbyint(t2);
                const float s3 = std::nearbyint((t2 - s2) * 256.0f);
                pl[(((size_t)c * 3 + 0) * N + n) * 128 + k] = __float2half_rn(s1);      // |s| <= 128: exact in fp16
                pl[(((size_t)c * 3 + 1) * N + n) * 128 + k] = __float2half_rn(s2);
                pl[(((size_t)c * 3 + 2) * N + n) * 128 + k] = __float2half_rn(s3);
            }
        }
    ExactW e{N, K, nullptr, nullptr};
    if (cudaMalloc(&e.planes, pl.size() * 2) != cudaSuccess) return;
    if (cudaMalloc(&e.cs, cs.size() * 4) != cudaSuccess) { cudaFree(e.planes); return; }
    cudaMemcpy(e.planes, pl.data(), pl.size() * 2, cudaMemcpyHostToDevice);
    cudaMemcpy(e.cs, cs.data(), cs.size() * 4, cudaMemcpyHostToDevice);
    reg.exact[Wdev] = e;
}
void gemm_registry_free(GemmRegistry& reg) {
    for (auto& kv : reg.exact) { cudaFree(kv.second.planes); cudaFree(kv.second.cs); }
    reg.exact.clear();
    reg.split.clear();
}

// C (+)= act(A) . W^T + bias on tensor cores with exact accumulation (k_gemm_exact).  Returns false when W has no
// slices registered or the shape is not covered; the caller then uses the fp32 FFMA kernel.
bool gemm_nt_exact(const Launch& L, const float* A, int lda, const float* W, float* C, int ldc, long long M, int N, int K,
                   const float* bias, bool accumulate, bool act_a) {
    using namespace tc;
    if (!L.reg) return false;
    auto it = L.reg->exact.find(W);
    if (it == L.reg->exact.end() || it->second.N != N || it->second.K != K) return false;
    if (M <= 0 || N > XNMAX || (lda % 4) || (ldc % 4) || (((uintptr_t)A | (uintptr_t)C | (uintptr_t)bias) & 15)) return false;
    static int n_sm = 0;
    static bool attr = false;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    if (!attr) {
        if (cudaFuncSetAttribute(k_gemm_exact<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, XSMEM) != cudaSuccess ||
            cudaFuncSetAttribute(k_gemm_exact<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, XSMEM) != cudaSuccess)
            return false;
        attr = true;
    }
    const ExactW& e = it->second;
    const long long units = (M + BM - 1) / BM;
    const int grid = (int)(units < n_sm ? units : n_sm);
    for (int c = 0; c < K / 128; c++) {
        CUtensorMap ma, m1, m2, m3;
        const __half* pl = (const __half*)e.planes + (size_t)c * 3 * N * 128;
        if (!make_map(&ma, A + c * 128, M, 128, lda, BM) || !make_map16(&m1, pl, N, XBN) ||
            !make_map16(&m2, pl + (size_t)N * 128, N, XBN) || !make_map16(&m3, pl + (size_t)2 * N * 128, N, XBN))
            return false;   // (only possible before the first launch: the driver entry point is missing)
        XParams p{C, c == 0 ? bias : nullptr, e.cs + (size_t)c * N, M, N, ldc, (accumulate || c > 0) ? 1 : 0};
        if (act_a) k_gemm_exact<true><<<grid, XTHREADS, XSMEM, L.stream>>>(ma, m1, m2, m3, p);
        else k_gemm_exact<false><<<grid, XTHREADS, XSMEM, L.stream>>>(ma, m1, m2, m3, p);
        KLAUNCH(L);
    }
    return true;
}

// Returns false when the shape is not covered (caller falls back to the SIMT path).
bool gemm_nt_tc(const Launch& L, const float* A, int lda, const float* Whi, const float* Wlo, int ldw, float* C, int ldc,
                long long M, int N, int K, const float* bias, bool accumulate, const float* dsilu_pre, int ld_pre,
                const float* resid) {
    using namespace tc;
    if (dsilu_pre && (accumulate || (ld_pre % 4) || ((uintptr_t)dsilu_pre & 15))) return false;
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
    if (resid && (((uintptr_t)resid & 15) || dsilu_pre)) return false;
    Params p{C, bias, M, N, K, ldc, (accumulate || resid) ? 1 : 0, dsilu_pre, ld_pre, resid ? resid : C};
    if (BN == 128) return launch<128, 3>(L, ma, mh, ml, p, n_sm);
    return launch<64, 4>(L, ma, mh, ml, p, n_sm);
}

}  // namespace painn
