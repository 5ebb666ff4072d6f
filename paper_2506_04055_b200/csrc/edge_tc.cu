// edge_tc.cu -- message pass with the per-edge filter on tensor cores (F = 128 models).
//
//   w_e = fc(d_e) (Wf rho(d_e) + bf)  is a [3F x (K+1)] . [(K+1) x edges] GEMM: per 32-edge tile one warp group
//   computes R_e = fc (1, rho_1..rho_K) on the fly (sincospi + rotation recurrence), writes it as the B operand into
//   shared memory, one thread issues tcgen05.mma (A = Wf|bf resident in shared memory, M = 128 channels per chunk,
//   N = 32 edges), and the accumulator D[channel, edge] lands in TMEM with ONE CHANNEL PER LANE.  The four consumer
//   warps then read their own channel's filter values (tcgen05.ld 32x32b) and run the segment sum over the sorted
//   CSR rows with plain FMAs: no atomics, no shuffles, coalesced 512 B gathers of the sender rows.
//
// Precision: fp16 operands alone miss the force tolerance (measured), so both operands are
// split x = hi + lo (two fp16 numbers, ~22 bits) and three product terms are accumulated:
//   hi(W) hi(R)  +  [hi(W) 2^-11][lo(R) 2^11]  +  [lo(W) 2^11][hi(R) 2^-11]           (K dimension 3 x 32 = 96)
// The two small terms are issued first so the fp32 accumulator (which truncates toward zero after every MMA) sees
// only two full-magnitude additions.
#include <cuda_fp16.h>

#include <algorithm>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "tc_common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

namespace etc {

constexpr int F = 128;
constexpr int NE = 32;                        // edges per tile (MMA N)
constexpr int KP = 96;                        // 3 terms x 32 basis slots
constexpr int LBO = 128, SBO = (KP / 8) * 128;          // 1536
constexpr int A_CHUNK_BYTES = (F / 8) * SBO;            // 24576
constexpr int B_BYTES = (NE / 8) * SBO;                 // 6144
constexpr int NTHREADS = 256;

// host: A operand image of one layer (3 chunks), see header comment; W[f][0] = bf, W[f][b] = Wf[f][b-1]
void build_filter_image(const float* Wf, const float* bf, int K, std::vector<unsigned short>& img) {
    img.assign(3 * A_CHUNK_BYTES / 2, 0);
    for (int c = 0; c < 3; c++)
        for (int r = 0; r < F; r++)
            for (int b = 0; b <= K; b++) {
                const float w = b == 0 ? bf[c * F + r] : Wf[(size_t)(c * F + r) * K + (b - 1)];
                const __half hi = __float2half_rn(w);
                const float hif = __half2float(hi);
                const __half t1 = __float2half_rn(hif * (1.0f / 2048.0f));
                const __half t2 = __float2half_rn((w - hif) * 2048.0f);
                const __half vals[3] = {hi, t1, t2};
                for (int t = 0; t < 3; t++) {
                    const int k = t * 32 + b;
                    const size_t off = (size_t)c * A_CHUNK_BYTES + (r / 8) * SBO + (k / 8) * LBO + (r % 8) * 16 + (k % 8) * 2;
                    unsigned short bits;
                    memcpy(&bits, &vals[t], 2);
                    img[off / 2] = bits;
                }
            }
}

// gather rows: Q4[j][f] = (phi^s, phi^vs, phi^vv v_x, phi^vv v_y), Q1[j][f] = phi^vv v_z ; layer 0 (v = 0): Q2 = (phi^s, phi^vs)
__global__ void k_make_gather(long long N, const float* __restrict__ phi, const float* __restrict__ v,
                              float4* __restrict__ Q4, float* __restrict__ Q1, float2* __restrict__ Q2, int has_v) {
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F) return;
    const long long j = idx / F;
    const int f = (int)(idx - j * F);
    const float ps = phi[j * 3 * F + f], pvs = phi[j * 3 * F + F + f];
    if (has_v) {
        const float pvv = phi[j * 3 * F + 2 * F + f];
        Q4[idx] = make_float4(ps, pvs, pvv * v[j * 3 * F + f], pvv * v[j * 3 * F + F + f]);
        Q1[idx] = pvv * v[j * 3 * F + 2 * F + f];
    } else {
        Q2[idx] = make_float2(ps, pvs);
    }
}

struct FwdParams {
    long long N;
    const int* row_ptr;
    const float4* ej;
    const float* s;
    const float* v;
    const float4* Q4;
    const float* Q1;
    const float2* Q2;
    const uint4* A_img;
    float* sn;     // s' written with row stride 2F
    float* v1;
    float inv_rc;
    int K;
    int atoms_per_unit;
};

template <bool HAS_V>
__global__ void __launch_bounds__(NTHREADS, 2) k_message_fwd_tc(FwdParams p) {
    constexpr int NCH = HAS_V ? 3 : 2;
    constexpr int TCOLS = NCH * NE;                 // TMEM columns per buffer
    constexpr int TALLOC = HAS_V ? 256 : 128;
    // declared aligned (no run-time pointer rounding: that would hide the shared address space from the compiler
    // and turn every LDS / STS into a generic LD / ST)
    extern __shared__ __align__(128) uint8_t smem[];
    uint8_t* sA = smem;
    uint8_t* sB = sA + NCH * A_CHUNK_BYTES;
    float4* sMeta = (float4*)(sB + 2 * B_BYTES);
    uint64_t* bars = (uint64_t*)(sMeta + 2 * NE);
    uint64_t* b_full = bars;          // [2] producer -> MMA      (count 96)
    uint64_t* t_full = bars + 2;      // [2] MMA commit -> consumers (count 1)
    uint64_t* t_empty = bars + 4;     // [2] consumers -> producer   (count 4)
    uint32_t* tmem_slot = (uint32_t*)(bars + 6);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    using namespace tc;

    // ---- one-time setup: filter operand into smem, zero B (padding slots stay zero), barriers, TMEM ----
    {
        const uint4* src = p.A_img;
        uint4* dst = (uint4*)sA;
        for (int i = tid; i < NCH * A_CHUNK_BYTES / 16; i += NTHREADS) dst[i] = src[i];
        uint4* zb = (uint4*)sB;
        for (int i = tid; i < 2 * B_BYTES / 16; i += NTHREADS) zb[i] = make_uint4(0, 0, 0, 0);
    }
    if (tid == 0) {
        for (int b = 0; b < 2; b++) { mbar_init(&b_full[b], 96); mbar_init(&t_full[b], 1); mbar_init(&t_empty[b], 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 7) tmem_alloc(tmem_slot, TALLOC);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const long long n_units = (p.N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    // register re-partition per warpgroup: consumers (warps 0-3) 168, producer / MMA warps (4-7) 88  (2 CTAs per SM)
    if (warp < 4) reg_inc<168>(); else reg_dec<88>();

    if (warp < 4) {
        // ===================== consumers: one channel per thread =====================
        const int f = tid;
        const uint32_t lane_base = tmem_base + ((uint32_t)(warp * 32) << 16);
        uint32_t it = 0;
        for (long long u = blockIdx.x; u < n_units; u += gridDim.x) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NE - 1) / NE;
            long long a_cur = a0;
            int row_end = p.row_ptr[a0 + 1];
            float accS = p.s[a_cur * F + f];
            float acc0 = p.v[a_cur * 3 * F + f], acc1 = p.v[a_cur * 3 * F + F + f], acc2 = p.v[a_cur * 3 * F + 2 * F + f];
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                mbar_wait(&t_full[buf], (it >> 1) & 1);
                tc_fence_after();
                const float4* meta = sMeta + buf * NE;
#pragma unroll 1
                for (int g = 0; g < NE / 16; g++) {
                    // 16 sender rows in flight per thread before the first use (the pass is bound by gather latency)
                    float4 q4[16];
                    float q1[16];
                    float2 q2[16];
#pragma unroll
                    for (int i = 0; i < 16; i++) {
                        const size_t row = (size_t)__float_as_int(meta[g * 16 + i].w) * F + f;
                        if (HAS_V) { q4[i] = __ldg(p.Q4 + row); q1[i] = __ldg(p.Q1 + row); }
                        else q2[i] = __ldg(p.Q2 + row);
                    }
                    uint32_t ws[16], wvs[16], wvv[16];
                    tmem_ld16_nowait(lane_base + buf * TCOLS + g * 16, ws);
                    tmem_ld16_nowait(lane_base + buf * TCOLS + NE + g * 16, wvs);
                    if (HAS_V) tmem_ld16_nowait(lane_base + buf * TCOLS + 2 * NE + g * 16, wvv);
                    tmem_wait_ld();
#pragma unroll
                    for (int i = 0; i < 16; i++) {
                        const int E = e_begin + t * NE + g * 16 + i;
                        if (E < e_end) {
                            while (E >= row_end) {   // uniform: finish receiver a_cur, start the next row
                                p.sn[a_cur * 2 * F + f] = accS;
                                p.v1[a_cur * 3 * F + f] = acc0; p.v1[a_cur * 3 * F + F + f] = acc1; p.v1[a_cur * 3 * F + 2 * F + f] = acc2;
                                a_cur++;
                                row_end = p.row_ptr[a_cur + 1];
                                accS = p.s[a_cur * F + f];
                                acc0 = p.v[a_cur * 3 * F + f]; acc1 = p.v[a_cur * 3 * F + F + f]; acc2 = p.v[a_cur * 3 * F + 2 * F + f];
                            }
                            const float4 m = meta[g * 16 + i];
                            const float w_s = __uint_as_float(ws[i]), w_vs = __uint_as_float(wvs[i]);
                            if (HAS_V) {
                                const float w_vv = __uint_as_float(wvv[i]);
                                accS = fmaf(w_s, q4[i].x, accS);
                                const float tv = w_vs * q4[i].y;
                                acc0 = fmaf(tv, m.x, fmaf(w_vv, q4[i].z, acc0));
                                acc1 = fmaf(tv, m.y, fmaf(w_vv, q4[i].w, acc1));
                                acc2 = fmaf(tv, m.z, fmaf(w_vv, q1[i], acc2));
                            } else {
                                accS = fmaf(w_s, q2[i].x, accS);
                                const float tv = w_vs * q2[i].y;
                                acc0 = fmaf(tv, m.x, acc0);
                                acc1 = fmaf(tv, m.y, acc1);
                                acc2 = fmaf(tv, m.z, acc2);
                            }
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&t_empty[buf]);
            }
            // finish the last receiver with edges, then pass trailing edge-less atoms through (s' = s, v' = v)
            for (;;) {
                p.sn[a_cur * 2 * F + f] = accS;
                p.v1[a_cur * 3 * F + f] = acc0; p.v1[a_cur * 3 * F + F + f] = acc1; p.v1[a_cur * 3 * F + 2 * F + f] = acc2;
                if (++a_cur >= a1) break;
                accS = p.s[a_cur * F + f];
                acc0 = p.v[a_cur * 3 * F + f]; acc1 = p.v[a_cur * 3 * F + F + f]; acc2 = p.v[a_cur * 3 * F + 2 * F + f];
            }
        }
    } else if (warp < 7) {
        // ===================== producers: B operand R_e = fc (1, rho_1 .. rho_K) split into fp16 hi / lo =====================
        const int pt = tid - 128, e = pt & 31, h = pt >> 5;   // h: basis slots 8h .. 8h+7 (slot 0 = bias, slot n = rho_n)
        uint32_t it = 0;
        for (long long u = blockIdx.x; u < n_units; u += gridDim.x) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NE - 1) / NE;
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                const int E = e_begin + t * NE + e;
                float4 r = make_float4(1.f, 0.f, 0.f, __int_as_float(0));
                const bool valid = E < e_end;
                if (valid) r = __ldg(p.ej + E);
                const bool real = valid && __float_as_int(r.w) >= 0;     // padding slots carry sender index ~self
                if (valid && !real) r.w = __int_as_float(~__float_as_int(r.w));
                const float d2 = r.x * r.x + r.y * r.y + r.z * r.z;
                const float inv_d = rsqrtf(d2);
                const float x = d2 * inv_d * p.inv_rc;
                float s1, c1;
                sincospif(x, &s1, &c1);
                const float fc = real ? 0.5f * (1.0f + c1) : 0.0f;
                const float amp = fc * inv_d;
                float sn_, cn_;
                const int n0 = h == 0 ? 1 : 8 * h;
                if (h == 0) { sn_ = s1; cn_ = c1; } else sincospif((float)n0 * x, &sn_, &cn_);
                __half2 hi2[4], t1[4], t2[4];
                float vals[8];
#pragma unroll
                for (int i = 0; i < 8; i++) {
                    const int b = h * 8 + i;
                    float R;
                    if (b == 0) R = fc;
                    else {
                        R = b <= p.K ? amp * sn_ : 0.0f;
                        const float tt = sn_ * c1 + cn_ * s1;
                        cn_ = cn_ * c1 - sn_ * s1;
                        sn_ = tt;
                    }
                    vals[i] = R;
                }
#pragma unroll
                for (int i = 0; i < 4; i++) {
                    const __half h0 = __float2half_rn(vals[2 * i]), h1 = __float2half_rn(vals[2 * i + 1]);
                    const float f0 = __half2float(h0), f1 = __half2float(h1);
                    hi2[i] = __halves2half2(h0, h1);
                    t1[i] = __halves2half2(__float2half_rn((vals[2 * i] - f0) * 2048.0f), __float2half_rn((vals[2 * i + 1] - f1) * 2048.0f));
                    t2[i] = __halves2half2(__float2half_rn(f0 * (1.0f / 2048.0f)), __float2half_rn(f1 * (1.0f / 2048.0f)));
                }
                mbar_wait_relaxed(&t_empty[buf], ((it >> 1) & 1) ^ 1);
                uint8_t* bb = sB + buf * B_BYTES + (e >> 3) * SBO + (e & 7) * 16 + h * LBO;
                *(uint4*)(bb) = *(uint4*)hi2;                       // term 0: k = b
                *(uint4*)(bb + 4 * LBO) = *(uint4*)t1;              // term 1: k = 32 + b   (lo(R) 2^11)
                *(uint4*)(bb + 8 * LBO) = *(uint4*)t2;              // term 2: k = 64 + b   (hi(R) 2^-11)
                if (h == 0) sMeta[buf * NE + e] = make_float4(r.x * inv_d, r.y * inv_d, r.z * inv_d, r.w);
                fence_async_smem();
                mbar_arrive(&b_full[buf]);
            }
        }
    } else {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            const uint32_t idesc = (1u << 4) | ((uint32_t)(NE >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);   // f16 x f16 -> f32
            const uint32_t a_base = smem_u32(sA), b_base = smem_u32(sB);
            uint32_t it = 0;
            for (long long u = blockIdx.x; u < n_units; u += gridDim.x) {
                const long long a0 = u * p.atoms_per_unit;
                const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
                const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
                const int ntiles = (e_end - e_begin + NE - 1) / NE;
                for (int t = 0; t < ntiles; t++, it++) {
                    const int buf = it & 1;
                    mbar_wait_relaxed(&b_full[buf], (it >> 1) & 1);
                    tc_fence_after();
#pragma unroll
                    for (int c = 0; c < NCH; c++) {
                        const uint32_t d = tmem_base + buf * TCOLS + c * NE;
#pragma unroll
                        for (int o = 0; o < 6; o++) {
                            const int kk = (o + 2) % 6;          // small terms (k-steps 2..5) first, main term last
                            const uint64_t ad = make_desc_nosw(a_base + c * A_CHUNK_BYTES + kk * 2 * LBO, LBO, SBO);
                            const uint64_t bd = make_desc_nosw(b_base + buf * B_BYTES + kk * 2 * LBO, LBO, SBO);
                            umma_f16(d, ad, bd, idesc, o != 0);
                        }
                    }
                    umma_commit(&t_full[buf]);
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 7) tmem_dealloc(tmem_base, TALLOC);
}

constexpr int fwd_smem_bytes(bool has_v) { return (has_v ? 3 : 2) * A_CHUNK_BYTES + 2 * B_BYTES + 2 * NE * 16 + 64 + 128; }

// ================================================================================================ adjoint (a12)
// One thread per channel again, walking the SENDER's own row (no-atomics gather form, painn_bwd.cu header).
// Per 16-edge tile the producers emit R_e (rows 0..15 of the B operand) and R'_e = d/dd [fc (1, rho)] (rows 16..31),
// so one N = 32 MMA per chunk yields both the filter w (columns 0..15) and its derivative w' (columns 16..31).
// The four per-edge scalars (db, ub_x, ub_y, ub_z) are reduced over the 128 channels with a butterfly
// transpose-reduce (31 shuffles per 8 edges per warp) + one shared-memory hop across the four warps.
constexpr int NEB = 16;

// gather rows of the adjoint pass: Gb[i][f] = (sb', vb'_x, vb'_y, vb'_z)
__global__ void k_make_gather_bwd(long long N, const float* __restrict__ s1b, const float* __restrict__ v1b,
                                  float4* __restrict__ Gb) {
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F) return;
    const long long j = idx / F;
    const int f = (int)(idx - j * F);
    Gb[idx] = make_float4(s1b[idx], v1b[j * 3 * F + f], v1b[j * 3 * F + F + f], v1b[j * 3 * F + 2 * F + f]);
}

struct BwdParams {
    long long N;
    const int* row_ptr;
    const float4* ej;
    const float4* Gb;
    const float* phi;
    const float* v_in;
    const float* v1b;
    const uint4* A_img;
    float* phib;
    float* vb_out;
    float4* G;
    float inv_rc;
    int K;
    int atoms_per_unit;
    int first;
};

__global__ void __launch_bounds__(NTHREADS, 2) k_message_bwd_tc(BwdParams p) {
    constexpr int NCH = 3;
    constexpr int TCOLS = NCH * 2 * NEB;            // 96 TMEM columns per buffer
    constexpr int TALLOC = 256;
    // declared aligned (no run-time pointer rounding: that would hide the shared address space from the compiler
    // and turn every LDS / STS into a generic LD / ST)
    extern __shared__ __align__(128) uint8_t smem[];
    uint8_t* sA = smem;
    uint8_t* sB = sA + NCH * A_CHUNK_BYTES;                  // 2 buffers x (32 rows x 96 halfs) = 2 x 6144
    float4* sMeta = (float4*)(sB + 2 * B_BYTES);            // [2][16] (u_e, i)
    float* sInvd = (float*)(sMeta + 2 * NEB);               // [2][16]
    float* sRed = sInvd + 2 * NEB;                          // [2][4][32]
    uint64_t* bars = (uint64_t*)(sRed + 2 * 4 * 32);
    uint64_t* b_full = bars;          // [2] (count 48)
    uint64_t* t_full = bars + 2;      // [2] (count 1)
    uint64_t* t_empty = bars + 4;     // [2] consumers (4) + finisher (1) -> producer
    uint64_t* r_full = bars + 6;      // [2] per-edge partial sums written (count 4)
    uint64_t* r_empty = bars + 8;     // [2] finisher done with the reduction buffer (count 1)
    uint32_t* tmem_slot = (uint32_t*)(bars + 10);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    using namespace tc;
    {
        const uint4* src = p.A_img;
        uint4* dst = (uint4*)sA;
        for (int i = tid; i < NCH * A_CHUNK_BYTES / 16; i += NTHREADS) dst[i] = src[i];
        uint4* zb = (uint4*)sB;
        for (int i = tid; i < 2 * B_BYTES / 16; i += NTHREADS) zb[i] = make_uint4(0, 0, 0, 0);
    }
    if (tid == 0) {
        for (int b = 0; b < 2; b++) {
            mbar_init(&b_full[b], 48); mbar_init(&t_full[b], 1); mbar_init(&t_empty[b], 5);
            mbar_init(&r_full[b], 4); mbar_init(&r_empty[b], 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 7) tmem_alloc(tmem_slot, TALLOC);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const long long n_units = (p.N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    // register re-partition per warpgroup: consumers (warps 0-3) 168, producer / MMA warps (4-7) 88  (2 CTAs per SM)
    if (warp < 4) reg_inc<168>(); else reg_dec<88>();

    if (warp < 4) {
        // ===================== consumers =====================
        const int f = tid;
        const uint32_t lane_base = tmem_base + ((uint32_t)(warp * 32) << 16);
        uint32_t it = 0, hc = 0;    // tile counter, 8-edge half counter (selects the reduction buffer)
        for (long long u = blockIdx.x; u < n_units; u += gridDim.x) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            long long j = a0;
            int row_end = p.row_ptr[a0 + 1];
            float phS = p.phi[j * 3 * F + f], phVS = p.phi[j * 3 * F + F + f], phVV = p.phi[j * 3 * F + 2 * F + f];
            float vj0 = p.v_in[j * 3 * F + f], vj1 = p.v_in[j * 3 * F + F + f], vj2 = p.v_in[j * 3 * F + 2 * F + f];
            float pbS = 0.f, pbVS = 0.f, Y0 = 0.f, Y1 = 0.f, Y2 = 0.f;
            auto finish_row = [&]() {
                p.phib[j * 3 * F + f] = pbS;
                p.phib[j * 3 * F + F + f] = pbVS;
                p.phib[j * 3 * F + 2 * F + f] = vj0 * Y0 + vj1 * Y1 + vj2 * Y2;
                p.vb_out[j * 3 * F + f] = p.v1b[j * 3 * F + f] + phVV * Y0;
                p.vb_out[j * 3 * F + F + f] = p.v1b[j * 3 * F + F + f] + phVV * Y1;
                p.vb_out[j * 3 * F + 2 * F + f] = p.v1b[j * 3 * F + 2 * F + f] + phVV * Y2;
            };
            auto start_row = [&]() {
                row_end = p.row_ptr[j + 1];
                phS = p.phi[j * 3 * F + f]; phVS = p.phi[j * 3 * F + F + f]; phVV = p.phi[j * 3 * F + 2 * F + f];
                vj0 = p.v_in[j * 3 * F + f]; vj1 = p.v_in[j * 3 * F + F + f]; vj2 = p.v_in[j * 3 * F + 2 * F + f];
                pbS = pbVS = Y0 = Y1 = Y2 = 0.f;
            };
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                mbar_wait(&t_full[buf], (it >> 1) & 1);
                tc_fence_after();
                const float4* meta = sMeta + buf * NEB;
#pragma unroll 1
                for (int h = 0; h < 2; h++, hc++) {
                    uint32_t w[3][8], dw[3][8];
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        tmem_ld8_nowait(lane_base + buf * TCOLS + c * 2 * NEB + h * 8, w[c]);
                        tmem_ld8_nowait(lane_base + buf * TCOLS + c * 2 * NEB + NEB + h * 8, dw[c]);
                    }
                    float4 m[8], gb[8];
#pragma unroll
                    for (int i = 0; i < 8; i++) {
                        m[i] = meta[h * 8 + i];
                        gb[i] = __ldg(p.Gb + (size_t)__float_as_int(m[i].w) * F + f);
                    }
                    tmem_wait_ld();
                    float part[32];
#pragma unroll
                    for (int i = 0; i < 8; i++) {
                        const int E = e_begin + t * NEB + h * 8 + i;
                        float db = 0.f, ub0 = 0.f, ub1 = 0.f, ub2 = 0.f;
                        if (E < e_end) {
                            while (E >= row_end) { finish_row(); j++; start_row(); }
                            const float wS = __uint_as_float(w[0][i]), wVS = __uint_as_float(w[1][i]), wVV = __uint_as_float(w[2][i]);
                            const float dS = __uint_as_float(dw[0][i]), dVS = __uint_as_float(dw[1][i]), dVV = __uint_as_float(dw[2][i]);
                            const float sb = gb[i].x, vb0 = gb[i].y, vb1 = gb[i].z, vb2 = gb[i].w;
                            const float X = vb0 * m[i].x + vb1 * m[i].y + vb2 * m[i].z;
                            const float Z = vb0 * vj0 + vb1 * vj1 + vb2 * vj2;
                            pbS = fmaf(wS, sb, pbS);
                            pbVS = fmaf(wVS, X, pbVS);
                            Y0 = fmaf(wVV, vb0, Y0); Y1 = fmaf(wVV, vb1, Y1); Y2 = fmaf(wVV, vb2, Y2);
                            db = phS * sb * dS + phVS * X * dVS + phVV * Z * dVV;
                            const float tt = wVS * phVS;
                            ub0 = tt * vb0; ub1 = tt * vb1; ub2 = tt * vb2;
                        }
                        part[4 * i] = db; part[4 * i + 1] = ub0; part[4 * i + 2] = ub1; part[4 * i + 3] = ub2;
                    }
                    // butterfly transpose-reduce: lane l ends with the warp total of part[l]
#pragma unroll
                    for (int o = 16, n = 16; o >= 1; o >>= 1, n >>= 1) {
                        const bool up = (lane & o) != 0;
#pragma unroll
                        for (int k = 0; k < 16; k++) {
                            if (k < n) {
                                const float keep = up ? part[k + n] : part[k];
                                const float send = up ? part[k] : part[k + n];
                                part[k] = keep + __shfl_xor_sync(0xffffffffu, send, o);
                            }
                        }
                    }
                    // hand the 32 warp totals to the finisher warp (cross-warp sum, g_e, G update) without a CTA barrier
                    float* red = sRed + (hc & 1) * 128;
                    mbar_wait(&r_empty[hc & 1], ((hc >> 1) & 1) ^ 1);
                    red[warp * 32 + lane] = part[0];
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&r_full[hc & 1]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&t_empty[buf]);
            }
            for (;;) {
                finish_row();
                if (++j >= a1) break;
                start_row();
            }
        }
    } else if (warp < 6) {
        // ===================== producers: rows 0..15 R_e, rows 16..31 R'_e =====================
        const int pt = tid - 128, e = pt & 15, h = pt >> 4;   // h = 0..3 (h == 3 idle)
        uint32_t it = 0;
        const float a1c = 3.14159265358979323846f * p.inv_rc;
        for (long long u = blockIdx.x; u < n_units; u += gridDim.x) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            for (int t = 0; t < ntiles; t++, it++) {
                if (h == 3) continue;
                const int buf = it & 1;
                const int E = e_begin + t * NEB + e;
                float4 r = make_float4(1.f, 0.f, 0.f, __int_as_float(0));
                const bool valid = E < e_end;
                if (valid) r = __ldg(p.ej + E);
                const bool real = valid && __float_as_int(r.w) >= 0;     // padding slots carry sender index ~self
                if (valid && !real) r.w = __int_as_float(~__float_as_int(r.w));
                const float d2 = r.x * r.x + r.y * r.y + r.z * r.z;
                const float inv_d = rsqrtf(d2);
                const float x = d2 * inv_d * p.inv_rc;
                float s1, c1;
                sincospif(x, &s1, &c1);
                const float fc = real ? 0.5f * (1.0f + c1) : 0.0f;
                const float dfc = real ? -0.5f * a1c * s1 : 0.0f;
                float sn_, cn_;
                const int n0 = h == 0 ? 1 : 8 * h;
                if (h == 0) { sn_ = s1; cn_ = c1; } else sincospif((float)n0 * x, &sn_, &cn_);
                float vals[8], dvals[8];
#pragma unroll
                for (int i = 0; i < 8; i++) {
                    const int b = h * 8 + i;
                    if (b == 0) { vals[i] = fc; dvals[i] = dfc; }
                    else {
                        const float rho = sn_ * inv_d;
                        const float drho = ((float)b * a1c * cn_ - rho) * inv_d;
                        vals[i] = b <= p.K ? fc * rho : 0.0f;
                        dvals[i] = b <= p.K ? dfc * rho + fc * drho : 0.0f;
                        const float tt = sn_ * c1 + cn_ * s1;
                        cn_ = cn_ * c1 - sn_ * s1;
                        sn_ = tt;
                    }
                }
                __half2 q[6][4];
#pragma unroll
                for (int i = 0; i < 4; i++) {
#pragma unroll
                    for (int z = 0; z < 2; z++) {
                        const float v0 = z ? dvals[2 * i] : vals[2 * i], v1 = z ? dvals[2 * i + 1] : vals[2 * i + 1];
                        const __half h0 = __float2half_rn(v0), h1 = __float2half_rn(v1);
                        const float f0 = __half2float(h0), f1 = __half2float(h1);
                        q[3 * z + 0][i] = __halves2half2(h0, h1);
                        q[3 * z + 1][i] = __halves2half2(__float2half_rn((v0 - f0) * 2048.0f), __float2half_rn((v1 - f1) * 2048.0f));
                        q[3 * z + 2][i] = __halves2half2(__float2half_rn(f0 * (1.0f / 2048.0f)), __float2half_rn(f1 * (1.0f / 2048.0f)));
                    }
                }
                mbar_wait_relaxed(&t_empty[buf], ((it >> 1) & 1) ^ 1);
#pragma unroll
                for (int z = 0; z < 2; z++) {
                    const int row = z * NEB + e;
                    uint8_t* bb = sB + buf * B_BYTES + (row >> 3) * SBO + (row & 7) * 16 + h * LBO;
                    *(uint4*)(bb) = *(uint4*)q[3 * z + 0];
                    *(uint4*)(bb + 4 * LBO) = *(uint4*)q[3 * z + 1];
                    *(uint4*)(bb + 8 * LBO) = *(uint4*)q[3 * z + 2];
                }
                if (h == 0) {
                    sMeta[buf * NEB + e] = make_float4(-r.x * inv_d, -r.y * inv_d, -r.z * inv_d, r.w);   // u_e of edge (i <- j)
                    sInvd[buf * NEB + e] = inv_d;
                }
                fence_async_smem();
                mbar_arrive(&b_full[buf]);
            }
        }
    } else if (warp == 6) {
        // ===================== finisher: sum the four warps' partials, assemble g_e, accumulate G =====================
        uint32_t it = 0, hc = 0;
        for (long long u = blockIdx.x; u < n_units; u += gridDim.x) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                for (int h = 0; h < 2; h++, hc++) {
                    mbar_wait_relaxed(&r_full[hc & 1], (hc >> 1) & 1);
                    const float* red = sRed + (hc & 1) * 128;
                    const int E = e_begin + t * NEB + h * 8 + lane;
                    if (lane < 8 && E < e_end) {
                        float db = 0.f, ub0 = 0.f, ub1 = 0.f, ub2 = 0.f;
#pragma unroll
                        for (int wq = 0; wq < 4; wq++) {
                            db += red[wq * 32 + 4 * lane]; ub0 += red[wq * 32 + 4 * lane + 1];
                            ub1 += red[wq * 32 + 4 * lane + 2]; ub2 += red[wq * 32 + 4 * lane + 3];
                        }
                        const float4 mm = sMeta[buf * NEB + h * 8 + lane];
                        const float inv_d = sInvd[buf * NEB + h * 8 + lane];
                        const float uu = ub0 * mm.x + ub1 * mm.y + ub2 * mm.z;
                        float4 g = make_float4(db * mm.x + (ub0 - uu * mm.x) * inv_d, db * mm.y + (ub1 - uu * mm.y) * inv_d,
                                               db * mm.z + (ub2 - uu * mm.z) * inv_d, 0.f);
                        if (!p.first) { const float4 o = p.G[E]; g.x += o.x; g.y += o.y; g.z += o.z; }
                        p.G[E] = g;
                    }
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(&r_empty[hc & 1]);
                        if (h == 1) mbar_arrive(&t_empty[buf]);
                    }
                }
            }
        }
    } else if (warp == 7) {
        if (lane == 0) {
            const uint32_t idesc = (1u << 4) | ((uint32_t)((2 * NEB) >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
            const uint32_t a_base = smem_u32(sA), b_base = smem_u32(sB);
            uint32_t it = 0;
            for (long long u = blockIdx.x; u < n_units; u += gridDim.x) {
                const long long a0 = u * p.atoms_per_unit;
                const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
                const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
                const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
                for (int t = 0; t < ntiles; t++, it++) {
                    const int buf = it & 1;
                    mbar_wait_relaxed(&b_full[buf], (it >> 1) & 1);
                    tc_fence_after();
#pragma unroll
                    for (int c = 0; c < NCH; c++) {
                        const uint32_t d = tmem_base + buf * TCOLS + c * 2 * NEB;
#pragma unroll
                        for (int o = 0; o < 6; o++) {
                            const int kk = (o + 2) % 6;
                            const uint64_t ad = make_desc_nosw(a_base + c * A_CHUNK_BYTES + kk * 2 * LBO, LBO, SBO);
                            const uint64_t bd = make_desc_nosw(b_base + buf * B_BYTES + kk * 2 * LBO, LBO, SBO);
                            umma_f16(d, ad, bd, idesc, o != 0);
                        }
                    }
                    umma_commit(&t_full[buf]);
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 7) tmem_dealloc(tmem_base, TALLOC);
}

constexpr int bwd_smem_bytes() { return 3 * A_CHUNK_BYTES + 2 * B_BYTES + 2 * NEB * 16 + 2 * NEB * 4 + 2 * 4 * 32 * 4 + 96 + 128; }

}  // namespace etc

void edge_build_filter_image(const float* Wf, const float* bf, int K, std::vector<unsigned short>& img) {
    etc::build_filter_image(Wf, bf, K, img);
}
size_t edge_filter_image_bytes() { return 3 * etc::A_CHUNK_BYTES; }

void make_gather_rows(const Launch& L, long long N, const float* phi, const float* v, float* Q4, float* Q1, bool has_v) {
    if (N == 0) return;
    etc::k_make_gather<<<(unsigned)((N * etc::F + 255) / 256), 256, 0, L.stream>>>(N, phi, v, (float4*)Q4, Q1, (float2*)Q4,
                                                                                  has_v ? 1 : 0);
    KLAUNCH(L);
}

// F = 128, K <= 23 only.  Q4/Q1 from make_gather_rows (layer 0: Q4 holds float2 rows).
bool message_fwd_tc(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* s,
                    const float* v, const float* Q4, const float* Q1, const void* A_img, float* sn, float* v1, bool has_v) {
    using namespace etc;
    if (N == 0) return true;
    if (K > 23) return false;
    static int n_sm = 0;
    static bool attr = false;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    if (!attr) {
        if (cudaFuncSetAttribute(k_message_fwd_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, fwd_smem_bytes(true)) != cudaSuccess ||
            cudaFuncSetAttribute(k_message_fwd_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, fwd_smem_bytes(false)) != cudaSuccess)
            return false;
        attr = true;
    }
    FwdParams p{N, row_ptr, ej, s, v, (const float4*)Q4, Q1, (const float2*)Q4, (const uint4*)A_img, sn, v1, 1.0f / rc, K, 16};
    const long long n_units = (N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    const int grid = (int)std::min<long long>(n_units, 2LL * n_sm);
    if (has_v) k_message_fwd_tc<true><<<grid, NTHREADS, fwd_smem_bytes(true), L.stream>>>(p);
    else k_message_fwd_tc<false><<<grid, NTHREADS, fwd_smem_bytes(false), L.stream>>>(p);
    KLAUNCH(L);
    return true;
}

void make_gather_rows_bwd(const Launch& L, long long N, const float* s1b, const float* v1b, float* Gb) {
    if (N == 0) return;
    etc::k_make_gather_bwd<<<(unsigned)((N * etc::F + 255) / 256), 256, 0, L.stream>>>(N, s1b, v1b, (float4*)Gb);
    KLAUNCH(L);
}

bool message_bwd_tc(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* Gb,
                    const float* phi, const float* v_in, const float* v1b, const void* A_img, float* phib, float* vb_out,
                    float4* G, bool first) {
    using namespace etc;
    if (N == 0) return true;
    if (K > 23) return false;
    static int n_sm = 0;
    static bool attr = false;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    if (!attr) {
        if (cudaFuncSetAttribute(k_message_bwd_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, bwd_smem_bytes()) != cudaSuccess)
            return false;
        attr = true;
    }
    BwdParams p{N, row_ptr, ej, (const float4*)Gb, phi, v_in, v1b, (const uint4*)A_img, phib, vb_out, G, 1.0f / rc, K, 16,
                first ? 1 : 0};
    const long long n_units = (N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    const int grid = (int)std::min<long long>(n_units, 2LL * n_sm);
    k_message_bwd_tc<<<grid, NTHREADS, bwd_smem_bytes(), L.stream>>>(p);
    KLAUNCH(L);
    return true;
}

}  // namespace painn
