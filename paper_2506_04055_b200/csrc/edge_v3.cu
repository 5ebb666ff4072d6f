// edge_v3.cu -- message / adjoint-message kernels of the F = 128 models.
//
//   w_e = fc(d_e) (Wf rho(d_e) + bf)  is a [3F x (K+1)] . [(K+1) x edges] GEMM: per tile of edges the producer warps
//   compute R_e = fc (1, rho_1..rho_K) on the fly (sincospi + rotation recurrence) and write it as the B operand into
//   shared memory, one elected thread issues tcgen05.mma (A = (bf | Wf), resident in TMEM / shared memory, M = 128
//   channels per chunk), and the accumulator D[channel, edge] lands in TMEM with ONE CHANNEL PER LANE.  The consumer
//   warps read their own channel's filter values (tcgen05.ld 32x32b) and run the CSR segment sum in registers: no
//   atomics, coalesced 512 B gathers of the sender rows.
//
// Precision: fp16 operands alone miss the force tolerance, so both operands are split
// x = hi + r (hi = RN_fp16(x), r the exact remainder) and THREE product terms are accumulated along K = 3 x 24 (+ 8 zero
// slots) = 80, five k-steps:
//   [hi(W) 2^-6][r(R) 2^6]  +  [r(W) 2^6][hi(R) 2^-6]  +  hi(W) hi(R)
// (split3b / filter_planes; K + 1 <= 24 basis slots per term).  The cross terms come first in K and the MMAs are issued
// in ascending K, so the fp32 accumulator (which truncates toward zero after every MMA, B3) sees only two
// full-magnitude additions.  Round 1 used 2^+-11 scales on 32-slot terms: the hi 2^-11 planes were fp16 subnormals for
// most operands and a cross term lost its bits -- 3.6x the per-atom energy noise of the plain fp32 kernels (DESIGN.md
// B1).  A fourth term r(W) r(R) was measured and changes nothing (2^-24 relative); without it the operand is 40 TMEM
// columns per chunk and ALL chunks are TMEM-resident: the tensor core reads only the small B operand from shared memory.
//
// Kernel structure (from the ncu captures, profiles/r01_edge_ncu.md):
//   * gathers are software-pipelined: two register banks of 8 edges (forward), a 16-row cp.async window per thread
//     (adjoint); the pipeline runs across tile and unit boundaries;
//   * rows are padded to 8 slots with zero-weight dummies, so nothing is predicated per edge: one uniform
//     row-boundary test per 8 edges; the receiver's own rows (residual / phi_j, v_j) are loaded one row ahead;
//   * the adjoint reduces its per-edge sums over the 128 channels through shared-memory planes and a reducer warp
//     (four planes per edge: db and the vector beta' vb'; u, 1/d and the projection are applied once per edge);
//   * one 512-thread CTA per SM = two independent 8-warp pipelines sharing one copy of the filter operand.
#include <cuda_fp16.h>

#include <algorithm>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "tc_common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

namespace ev3 {

using namespace tc;

constexpr int F = 128;
constexpr int KP = 96;                        // 4 split terms x 24 basis slots
constexpr int LBO = 128, SBO = (KP / 8) * 128;          // 1536

// -------------------------------------------------------------------------------------------------------------
// producer helper: R_e = fc (1, rho_1..rho_K) [and R'_e = d/dd of it] for basis slots 8h..8h+7 of one edge
// -------------------------------------------------------------------------------------------------------------
struct EdgeGeom {
    float4 r;        // (r_e, sender index bits)
    float inv_d, s1, c1, x;
    float xl;        // pi * x_lo of the compensated phase (0 without it)
    bool real;
};
// The record of the NEXT tile's edge is fetched while the current tile is evaluated (load_edge_raw / edge_geom): a
// producer thread that loads and uses the record in the same iteration spends a third of its time on that latency.
__device__ __forceinline__ float4 load_edge_raw(const float4* __restrict__ ej, int E, int e_end) {
    float4 r = make_float4(1.f, 0.f, 0.f, __int_as_float(0));
    if (E < e_end) r = __ldg(ej + E);
    return r;
}
// xp = (x_hi, x_lo) of nbr.cu::phase_pair, or x_hi < 0: no compensated phase, x from the fp32 record
__device__ __forceinline__ float2 load_phase(const float2* __restrict__ xph, int E, int e_end) {
    float2 x = make_float2(-1.f, 0.f);
    if (xph != nullptr && E < e_end) x = __ldg(xph + E);
    return x;
}
template <bool ACC = false>
__device__ __forceinline__ EdgeGeom edge_geom(const float4 raw, int E, int e_end, float inv_rc,
                                              const float2 xp = make_float2(-1.f, 0.f)) {
    EdgeGeom g;
    g.r = raw;
    const bool valid = E < e_end;
    g.real = valid && __float_as_int(g.r.w) >= 0;                 // padding slots carry sender index ~self
    if (valid && !g.real) g.r.w = __int_as_float(~__float_as_int(g.r.w));
    const float d2 = g.r.x * g.r.x + g.r.y * g.r.y + g.r.z * g.r.z;
    g.inv_d = ACC ? 1.0f / sqrtf(d2) : rsqrtf(d2);        // forward (energy) path: IEEE, rsqrtf's 2 ulp go straight into u and rho
    g.x = d2 * g.inv_d * inv_rc;
    g.xl = 0.f;
    if (xp.x >= 0.f) { g.x = xp.x; g.xl = xp.y * 3.14159265358979323846f; }
    sincospif(g.x, &g.s1, &g.c1);
    const float ts = fmaf(g.xl, g.c1, g.s1);                      // sin(pi (x_hi + x_lo)) to first order in x_lo
    g.c1 = fmaf(-g.xl, g.s1, g.c1);
    g.s1 = ts;
    return g;
}
// Split 8 fp32 values x = hi + r (hi = RN_fp16(x), r exact in fp32) into the three fp16 planes of the B operand, one per
// product term of (A_hi + A_r)(B_hi + B_r) without the r r term (filter_planes holds the matching A planes):
//   term 0 (hl): r * 2^6  (against A_hi * 2^-6)     term 1 (lh): hi * 2^-6  (against A_r * 2^6)     term 2 (hh): hi
// The 2^+-6 scales keep both factors of the cross terms inside fp16's normal range for the magnitudes that occur
// (|R| ~ 1e-3 .. 1, |W| ~ 1e-3 .. 2): with the 2^+-11 scales of round 1 hi * 2^-11 was a subnormal for |R| < 0.125 and the
// cross term lost most of its bits (B1).  What falls below the normal range only costs 2^-25 absolute times
// the other factor.  Packed conversions: one F2FP per pair; the 2^-6 plane is an exact exponent shift done in half2.
__device__ __forceinline__ void split3b(const float (&v)[8], uint4& p_hl, uint4& p_lh, uint4& p_hh) {
    __half2 a[4], b[4], c[4];
    const __half2 k = __floats2half2_rn(1.0f / 64.0f, 1.0f / 64.0f);
#pragma unroll
    for (int i = 0; i < 4; i++) {
        a[i] = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
        const float2 f = __half22float2(a[i]);
        b[i] = __floats2half2_rn((v[2 * i] - f.x) * 64.0f, (v[2 * i + 1] - f.y) * 64.0f);
        c[i] = __hmul2(a[i], k);
    }
    p_hh = *(uint4*)a; p_hl = *(uint4*)b; p_lh = *(uint4*)c;
}
// byte offset of the 8-slot group h (basis slots 8h .. 8h+7) of product term t inside a B row block: K index 24 t + 8 h + i
// (the row block keeps the 12-group stride of KP = 96; groups 9 .. 11 stay zero)
__device__ __forceinline__ int kgrp_off(int t, int h) { return (3 * t + h) * 128; }

// =============================================================================================================
// forward message pass
// =============================================================================================================
constexpr int NE = 32;                                  // edges per tile (MMA N)
constexpr int B_BYTES = (NE / 8) * SBO;                 // 6144

struct FwdParams {
    long long N;
    const int* row_ptr;
    const float4* ej;
    const float* s;
    const float* v;
    const float4* Q4;
    const float* Q1;
    const float2* Q2;
    const uint4* A_rows;   // [3][128][80] fp16 rows of the filter operand (edge_build_filter_rows), TMEM-resident
    float* sn;     // s' written with row stride 2F
    float* v1;
    float inv_rc;
    int K;
    int atoms_per_unit;
    // layer 0 (HAS_V = false): s^0 = Emb[z], so the sender rows (phi^s_j, phi^vs_j) depend on the SPECIES of j only; they
    // come from an n_species-row table in shared memory instead of a 55 GB gather through L2
    const int* types;      // [N] species of the (cell-sorted) atoms
    const float2* tab;     // [n_tab][F] (phi^s, phi^vs) per species
    int n_tab;
    const float2* xph;     // [edges] compensated phase x = d / rc as (hi, lo) from the fp64 neighbour build, or nullptr
};

constexpr int TAB_MAX = 16;                             // species rows the shared-memory table can hold
// three product terms (hl, lh, hh) on K = 3 x 24 + 8 zero slots = 80 = five k-steps; 40 TMEM columns per chunk, so all
// three chunks are TMEM-resident (four terms would need 48 columns per chunk: 16 more than TMEM has)
constexpr int KB = 80, KB_COLS = KB / 2;
constexpr int BWD_TMEM_A = 384;                         // TMEM columns of the filter operand (behind 2 x 2 x 96 accumulator columns)

// =============================================================================================================
// adjoint message pass (sender-row gather form, painn_bwd.cu header): one 512-thread CTA per SM = two independent
// 8-warp pipelines ("groups") that share one copy of the filter operand
// =============================================================================================================
constexpr int NEB = 16;                                 // edges per tile; B rows 0..15 = R_e, 16..31 = R'_e
constexpr int BB_BYTES = (2 * NEB / 8) * SBO;           // 6144
constexpr int BWD_THREADS = 512;
constexpr int P_ROW = 3 * F * 4 + 64;                   // per-edge partials: x | y | z planes of 128 floats (+64 B: the two rows
                                                        // read by one quarter-warp of the reducer fall into different banks)
constexpr int P_BYTES = 8 * P_ROW;                      // one 8-edge batch
constexpr int BWD_PD = 3;                               // consumer loop: shared-memory loads run this many edges ahead
constexpr int GW = 16;                                  // gather window (edges in flight per thread)
constexpr int RING_BYTES = GW * F * 16;                 // 32768
constexpr int G_OFF_B = 0, G_OFF_P = 2 * BB_BYTES, G_OFF_RING = G_OFF_P + 2 * P_BYTES, G_OFF_META = G_OFF_RING + RING_BYTES,
              G_OFF_BAR = G_OFF_META + 4 * NEB * 16;      // (layout of k_msg_bwd0's pipelines: GROUP0_BYTES below)
// k_msg_bwd reduces FOUR planes per edge (db | beta' vb_x | beta' vb_y | beta' vb_z, see its consumer loop); the layer-0
// species-table kernel k_msg_bwd0 keeps the three-plane layout above
constexpr int P4_ROW = 4 * F * 4 + 64;
constexpr int P4_BYTES = 8 * P4_ROW;
// k_msg_bwd: gather window of 24 edges per thread = three 8-edge slot groups (A/B at config 5: 16 -> 24 edges 45.2 -> 44.2 ms
// per step, 32 edges 44.9 ms)
constexpr int GWH = 24, NSG = GWH / 8;
constexpr int HRING_BYTES = GWH * F * 16;
constexpr int H_OFF_B = 0, H_OFF_P = 2 * BB_BYTES, H_OFF_RING = H_OFF_P + 2 * P4_BYTES, H_OFF_META = H_OFF_RING + HRING_BYTES,
              H_OFF_BAR = H_OFF_META + 4 * NEB * 16, HGROUP_BYTES = H_OFF_BAR + 128;
constexpr int bwd_smem_bytes(int) { return 2 * HGROUP_BYTES + 128; }


// two fp32 additions in one instruction (register pairs as they come out of a 16-byte shared-memory load): the reducer
// warps sit on the critical path of their pipeline and are bound by instruction issue
__device__ __forceinline__ unsigned long long fadd2(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ float hsum2(unsigned long long a) {
    return __uint_as_float((uint32_t)a) + __uint_as_float((uint32_t)(a >> 32));
}
// tcgen05.st: 16 consecutive 32-bit columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
        "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&r)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
                 "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                 : "memory");
}
// A operand from TMEM (lane = row, 8 columns = 16 fp16 along K), B from shared memory
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

// =============================================================================================================
// forward message pass, grouped form: one 512-thread CTA per SM = two independent 8-warp pipelines ("groups", as in the
// adjoint kernel below) that share ONE copy of the filter operand, chunks s and vs of which are TMEM-resident (A-from-
// TMEM MMA).  ncu on k_msg_fwd: the tensor core re-reads the 72 KB shared-memory image for every 32-edge tile (33 % of the
// L1 data stage, l1tex__data_pipe_tc_wavefronts) and collides with the consumers' loads on the data banks (arbitration
// conflicts in 23 % of the cycles, LSU wavefronts 74 %): the kernel is bound by the L1 data stage, not by L2 or DRAM.
// =============================================================================================================
constexpr int FWDG_THREADS = 512;
constexpr int FWDG_GROUP_BYTES = ((2 * B_BYTES + 2 * NE * 16 + 64) + 127) / 128 * 128;
constexpr int fwdg_smem_bytes(bool has_v) {
    return 2 * FWDG_GROUP_BYTES + 128 + (has_v ? 0 : TAB_MAX * F * 8);
}
template <bool HAS_V>
__global__ void __launch_bounds__(FWDG_THREADS, 1) k_msg_fwd_g(const FwdParams p) {
    constexpr int NCH = HAS_V ? 3 : 2;
    constexpr int TCOLS = NCH * NE;                 // TMEM columns per buffer
    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, grp = tid >> 8, ltid = tid & 255, lwarp = ltid >> 5, lane = tid & 31;
    uint8_t* gbase = smem + grp * FWDG_GROUP_BYTES;
    uint8_t* sB = gbase;
    float4* sMeta = (float4*)(sB + 2 * B_BYTES);   // [2][NE] (u_e, sender index)
    uint64_t* bars = (uint64_t*)(sMeta + 2 * NE);
    uint64_t* b_full = bars;          // [2] producers -> MMA (and consumers: sender indices readable)  (count 96)
    uint64_t* t_full = bars + 2;      // [2] MMA commit -> consumers (count 1)
    const int NB = 1 + grp * 2;       // named barriers NB + buf of this group (consumers -> producers: tile consumed)
    uint32_t* tmem_slot = (uint32_t*)(smem + 2 * FWDG_GROUP_BYTES);
    float2* sTab = (float2*)(tmem_slot + 32);          // [n_tab][F] species table (layer 0 only), shared by both groups

    {
        uint4* zb = (uint4*)sB;
        for (int i = ltid; i < 2 * B_BYTES / 16; i += 256) zb[i] = make_uint4(0, 0, 0, 0);
        if (!HAS_V)
            for (int i = tid; i < p.n_tab * F; i += FWDG_THREADS) sTab[i] = p.tab[i];
    }
    if (ltid == 0) {
        for (int b = 0; b < 2; b++) { mbar_init(&b_full[b], 96); mbar_init(&t_full[b], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid >> 5 == 15) tmem_alloc(tmem_slot, 512);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    // all chunks of the filter operand into TMEM (lane = channel row, KB_COLS = 40 columns = 80 fp16 per chunk: three
    // product terms, see KB): columns 384 .. behind the two groups' accumulators (2 x 2 x 96 columns)
    if (tid < 128) {
#pragma unroll
        for (int c = 0; c < NCH; c++) {
            const uint32_t abase = *tmem_slot + BWD_TMEM_A + c * KB_COLS + ((uint32_t)((tid >> 5) * 32) << 16);
            const uint4* src = p.A_rows + ((size_t)c * 128 + tid) * (KB_COLS / 4);
#pragma unroll
            for (int j = 0; j < 2; j++) {
                uint32_t r[16];
#pragma unroll
                for (int q = 0; q < 4; q++) { const uint4 v = src[j * 4 + q]; r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w; }
                tmem_st16(abase + j * 16, r);
            }
            uint32_t r8[8];
#pragma unroll
            for (int q = 0; q < 2; q++) { const uint4 v = src[8 + q]; r8[4 * q] = v.x; r8[4 * q + 1] = v.y; r8[4 * q + 2] = v.z; r8[4 * q + 3] = v.w; }
            tmem_st8(abase + 32, r8);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot + grp * 192;
    const uint32_t tmem_A = *tmem_slot + BWD_TMEM_A;

    const long long N = p.N;
    const int apu = p.atoms_per_unit;
    const int* __restrict__ row_ptr = p.row_ptr;
    const long long n_units = (N + apu - 1) / apu;
    const long long u0 = (long long)blockIdx.x * 2 + grp, ustride = (long long)gridDim.x * 2;
    if (lwarp < 4) reg_inc<168>(); else reg_dec<88>();

    if (lwarp < 4) {
        // ===================== consumers: one channel per thread =====================
        const int f = ltid;
        const float4* __restrict__ Q4 = p.Q4 + f;
        const float* __restrict__ Q1 = p.Q1 + f;
        const float* __restrict__ s_in = p.s + f;
        const float* __restrict__ v_in = p.v + f;
        float* __restrict__ sn = p.sn + f;
        float* __restrict__ v1 = p.v1 + f;
        const uint32_t lane_base = tmem_base + ((uint32_t)(lwarp * 32) << 16);
        float4 qa4[8], qb4[8];
        float qa1[8], qb1[8];
#define FWD_ISSUE(Q4R, Q1R, META8)                                                   \
    {                                                                                     \
        _Pragma("unroll") for (int i_ = 0; i_ < 8; i_++) {                                \
            const size_t row_ = (size_t)__float_as_int((META8)[i_].w) * F;                \
            if (HAS_V) { Q4R[i_] = __ldg(Q4 + row_); Q1R[i_] = __ldg(Q1 + row_); }        \
        }                                                                                 \
    }
        uint32_t it = 0;
        bool pre = false;                 // first batch of tile `it` already in flight (bank a)
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const int na = (int)min((long long)apu, N - a0);
            const int rp = __ldg(row_ptr + a0 + min(lane, na));           // lanes 0..na hold the unit's row pointers
            const int e_begin = __shfl_sync(0xffffffffu, rp, 0), e_end = __shfl_sync(0xffffffffu, rp, na);
            const int ntiles = (e_end - e_begin + NE - 1) / NE;
            bool next_has = false;                                        // does the CTA's next unit have a tile?
            {
                const long long un = u + ustride;
                if (un < n_units) {
                    const long long b0 = un * apu, b1 = min(N, b0 + apu);
                    next_has = __ldg(row_ptr + b1) > __ldg(row_ptr + b0);
                }
            }
            if (HAS_V && ntiles > 0 && !pre) {
                mbar_wait(&b_full[it & 1], (it >> 1) & 1);
                const float4* m0 = sMeta + (it & 1) * NE;
                FWD_ISSUE(qa4, qa1, m0);
            }
            pre = false;
            int a_rel = 0;
            int row_end = __shfl_sync(0xffffffffu, rp, 1);
            float accS = 0.f, acc0 = 0.f, acc1 = 0.f, acc2 = 0.f;
            // residual (s_i, v_i) of the current receiver: loaded at row start, added at row end
            float rs = s_in[(a0 + a_rel) * F], rv0 = 0.f, rv1 = 0.f, rv2 = 0.f;
            if (HAS_V) { rv0 = v_in[(a0 + a_rel) * 3 * F]; rv1 = v_in[(a0 + a_rel) * 3 * F + F]; rv2 = v_in[(a0 + a_rel) * 3 * F + 2 * F]; }
            auto store_row = [&]() {
                const long long a = a0 + a_rel;
                sn[a * 2 * F] = accS + rs;
                v1[a * 3 * F] = acc0 + rv0; v1[a * 3 * F + F] = acc1 + rv1; v1[a * 3 * F + 2 * F] = acc2 + rv2;
            };
            auto next_row = [&]() {
                store_row();
                a_rel++;
                row_end = __shfl_sync(0xffffffffu, rp, a_rel + 1);
                accS = acc0 = acc1 = acc2 = 0.f;
                const long long a = a0 + a_rel;
                rs = s_in[a * F];
                if (HAS_V) { rv0 = v_in[a * 3 * F]; rv1 = v_in[a * 3 * F + F]; rv2 = v_in[a * 3 * F + 2 * F]; }
            };
#define FWD_COMPUTE(BI, Q4R, Q1R)                                                                      \
    {                                                                                                       \
        const int E8_ = e_begin + t * NE + (BI) * 8;                                                        \
        if (E8_ < e_end) {                                                                                  \
            while (E8_ >= row_end) next_row();                                                              \
            uint32_t ws[8], wvs[8], wvv[8];                                                                 \
            tmem_ld8_nowait(lane_base + buf * TCOLS + (BI) * 8, ws);                                        \
            tmem_ld8_nowait(lane_base + buf * TCOLS + NE + (BI) * 8, wvs);                                  \
            if (HAS_V) tmem_ld8_nowait(lane_base + buf * TCOLS + 2 * NE + (BI) * 8, wvv);                   \
            tmem_wait_ld();                                                                                 \
            _Pragma("unroll") for (int i_ = 0; i_ < 8; i_++) {                                              \
                const float4 m_ = meta[(BI) * 8 + i_];                                                      \
                const float w_s = __uint_as_float(ws[i_]), w_vs = __uint_as_float(wvs[i_]);                 \
                if (HAS_V) {                                                                                \
                    const float w_vv = __uint_as_float(wvv[i_]);                                            \
                    accS = fmaf(w_s, Q4R[i_].x, accS);                                                      \
                    const float tv = w_vs * Q4R[i_].y;                                                      \
                    acc0 = fmaf(tv, m_.x, fmaf(w_vv, Q4R[i_].z, acc0));                                     \
                    acc1 = fmaf(tv, m_.y, fmaf(w_vv, Q4R[i_].w, acc1));                                     \
                    acc2 = fmaf(tv, m_.z, fmaf(w_vv, Q1R[i_], acc2));                                       \
                } else {                                                                                    \
                    const float2 q_ = sTab[__float_as_int(m_.w) * F + f];       /* species row of the sender */ \
                    accS = fmaf(w_s, q_.x, accS);                                                           \
                    const float tv = w_vs * q_.y;                                                           \
                    acc0 = fmaf(tv, m_.x, acc0);                                                            \
                    acc1 = fmaf(tv, m_.y, acc1);                                                            \
                    acc2 = fmaf(tv, m_.z, acc2);                                                            \
                }                                                                                           \
            }                                                                                               \
        }                                                                                                   \
    }
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                const float4* meta = sMeta + buf * NE;
                FWD_ISSUE(qb4, qb1, meta + 8);
                mbar_wait(&t_full[buf], (it >> 1) & 1);
                tc_fence_after();
                FWD_COMPUTE(0, qa4, qa1);
                FWD_ISSUE(qa4, qa1, meta + 16);
                FWD_COMPUTE(1, qb4, qb1);
                FWD_ISSUE(qb4, qb1, meta + 24);
                FWD_COMPUTE(2, qa4, qa1);
                if (HAS_V && (t + 1 < ntiles || next_has)) {       // first batch of the CTA's next tile
                    mbar_wait(&b_full[buf ^ 1], ((it + 1) >> 1) & 1);
                    const float4* mn = sMeta + (buf ^ 1) * NE;
                    FWD_ISSUE(qa4, qa1, mn);
                    pre = t + 1 == ntiles;
                }
                FWD_COMPUTE(3, qb4, qb1);
                tc_fence_before();
                bar_arrive(NB + buf, 224);              // tile consumed: 128 consumers arrive, 96 producers wait (named barrier)
            }
            // finish the last receiver with edges, then pass trailing edge-less atoms through (s' = s, v' = v)
            for (;;) {
                store_row();
                if (a_rel + 1 >= na) break;
                a_rel++;
                accS = acc0 = acc1 = acc2 = 0.f;
                const long long a = a0 + a_rel;
                rs = s_in[a * F];
                if (HAS_V) { rv0 = v_in[a * 3 * F]; rv1 = v_in[a * 3 * F + F]; rv2 = v_in[a * 3 * F + 2 * F]; }
            }
        }
#undef FWD_ISSUE
#undef FWD_COMPUTE
    } else if (lwarp < 7) {
        // ===================== producers: B operand R_e = fc (1, rho_1 .. rho_K), three fp16 planes =====================
        const int pt = ltid - 128, e = pt & 31, h = pt >> 5;   // h: basis slots 8h .. 8h+7 (slot 0 = bias, slot n = rho_n)
        const float inv_rc = p.inv_rc;
        const int K = p.K;
        uint32_t it = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const long long a1 = min(N, a0 + (long long)apu);
            const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
            const int ntiles = (e_end - e_begin + NE - 1) / NE;
            float4 raw_n = load_edge_raw(p.ej, e_begin + e, e_end);
            float2 xp_n = load_phase(p.xph, e_begin + e, e_end);
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                const float4 raw = raw_n;
                const float2 xp = xp_n;
                if (t + 1 < ntiles) {
                    raw_n = load_edge_raw(p.ej, e_begin + (t + 1) * NE + e, e_end);
                    xp_n = load_phase(p.xph, e_begin + (t + 1) * NE + e, e_end);
                }
                const EdgeGeom g = edge_geom<true>(raw, e_begin + t * NE + e, e_end, inv_rc, xp);
                const float fc = g.real ? 0.5f * (1.0f + g.c1) : 0.0f;
                const float amp = fc * g.inv_d;
                float sn_, cn_;
                if (h == 0) { sn_ = g.s1; cn_ = g.c1; }
                else {
                    sincospif((float)(8 * h) * g.x, &sn_, &cn_);
                    const float dl = (float)(8 * h) * g.xl;              // first-order phase correction (pi x_lo)
                    const float ts = fmaf(dl, cn_, sn_);
                    cn_ = fmaf(-dl, sn_, cn_);
                    sn_ = ts;
                }
                float vals[8];
#pragma unroll
                for (int i = 0; i < 8; i++) {
                    const int b = h * 8 + i;
                    float R;
                    if (b == 0) R = fc;
                    else {
                        R = b <= K ? amp * sn_ : 0.0f;
                        const float tt = sn_ * g.c1 + cn_ * g.s1;
                        cn_ = cn_ * g.c1 - sn_ * g.s1;
                        sn_ = tt;
                    }
                    vals[i] = R;
                }
                uint4 p0, p1, p2;
                split3b(vals, p0, p1, p2);
                if (it >= 2) bar_sync(NB + buf, 224);   // tile it - 2 consumed (hardware-blocking wait, no spin)
                uint8_t* bb = sB + buf * B_BYTES + (e >> 3) * SBO + (e & 7) * 16;
                *(uint4*)(bb + kgrp_off(0, h)) = p0;      // term 0: k = b        lo(R) 2^6
                *(uint4*)(bb + kgrp_off(1, h)) = p1;      // term 1: k = 24 + b   hi(R) 2^-6
                *(uint4*)(bb + kgrp_off(2, h)) = p2;      // term 2: k = 48 + b   hi(R)
                if (h == 0) {
                    float mw = g.r.w;                                             // sender index ...
                    if (!HAS_V) mw = __int_as_float(__ldg(p.types + __float_as_int(g.r.w)));   // ... or its species (layer 0)
                    sMeta[buf * NE + e] = make_float4(g.r.x * g.inv_d, g.r.y * g.inv_d, g.r.z * g.inv_d, mw);
                }
                fence_async_smem();
                mbar_arrive(&b_full[buf]);
            }
        }
    } else {
        // ===================== MMA issuer: the warp stays converged, one elected lane issues (descriptors in uniform registers) =====================
        {
            const uint32_t idesc = (1u << 4) | ((uint32_t)(NE >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);   // f16 x f16 -> f32
            const uint32_t b_base = smem_u32(sB);
            uint32_t it = 0;
            for (long long u = u0; u < n_units; u += ustride) {
                const long long a0 = u * apu;
                const long long a1 = min(N, a0 + (long long)apu);
                const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
                const int ntiles = (e_end - e_begin + NE - 1) / NE;
                for (int t = 0; t < ntiles; t++, it++) {
                    const int buf = it & 1;
                    mbar_wait_sleep(&b_full[buf], (it >> 1) & 1, 128);
                    tc_fence_after();
                    if (elect_one()) {
#pragma unroll
                        for (int c = 0; c < NCH; c++) {
                            const uint32_t d = tmem_base + buf * TCOLS + c * NE;
#pragma unroll
                            for (int kk = 0; kk < KB_COLS / 8; kk++) {     // ascending K: the cross terms first, the main term (hh) last
                                const uint64_t bd = make_desc_nosw(b_base + buf * B_BYTES + kk * 2 * LBO, LBO, SBO);
                                umma_f16_ts(d, tmem_A + c * KB_COLS + kk * 8, bd, idesc, kk != 0);
                            }
                        }
                        umma_commit(&t_full[buf]);
                    }
                    __syncwarp();
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (tid >> 5 == 15) tmem_dealloc(*tmem_slot, 512);
}



struct BwdParams {
    long long N;
    const int* row_ptr;
    const float4* ej;
    const float4* Gb;      // gather rows (sb', vb'_x, vb'_y, vb'_z)
    const float* phi;
    const float* v_in;
    const float* v1b;
    const uint4* A_rows;   // [3][128][80] fp16 rows of the filter operand, TMEM-resident
    float* phib;
    float* vb_out;
    float4* G;
    float inv_rc;
    int K;
    int atoms_per_unit;
    int first;
};

// L0: layer 0 -- v_in = 0 and the embedding is constant, so only the geometry gradient G is produced
// (chunks s and vs of the filter; no phib / vb_out).
template <bool L0>
__global__ void __launch_bounds__(BWD_THREADS, 1) k_msg_bwd(const BwdParams p) {
    constexpr int NCH = L0 ? 2 : 3;
    constexpr int TCOLS = NCH * 2 * NEB;            // TMEM columns per accumulator buffer
    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, grp = tid >> 8, ltid = tid & 255, lwarp = ltid >> 5, lane = tid & 31;
    uint8_t* gbase = smem + grp * HGROUP_BYTES;
    uint8_t* sB = gbase + H_OFF_B;
    uint8_t* sP = gbase + H_OFF_P;                 // [2][8] rows of P4_ROW bytes: four planes of 128 floats per edge
    float4* sMeta = (float4*)(gbase + H_OFF_META); // [4][NEB] (u of edge (i <- j), 1/d): ring of 4 tiles
    uint64_t* bars = (uint64_t*)(gbase + H_OFF_BAR);
    uint64_t* t_full = bars;          // [2] MMA commit -> consumers (mbarrier, count 1)
    uint64_t* p_empty = bars + 2;     // [2] reducer -> consumers: partials buffer read (mbarrier, count 1)
    // named barriers of this group (hardware-blocking waits): [2] each
    const int NB_TE = 1 + grp * 6;    // consumers (128, arrive) -> producer (32, sync): tile buffer consumed
    const int NB_BF = NB_TE + 2;      // producer (32, arrive) -> MMA warp (32, sync): B operand written
    const int NB_PF = NB_TE + 4;      // consumers (128, arrive) -> reducer (32, sync): partials of one batch written
    uint32_t* tmem_slot = (uint32_t*)(smem + 2 * HGROUP_BYTES);

    {
        uint4* zb = (uint4*)sB;
        for (int i = ltid; i < 2 * BB_BYTES / 16; i += 256) zb[i] = make_uint4(0, 0, 0, 0);
    }
    if (ltid == 0) {
        for (int b = 0; b < 2; b++) { mbar_init(&t_full[b], 1); mbar_init(&p_empty[b], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid >> 5 == 15) tmem_alloc(tmem_slot, 512);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    // ALL chunks of the filter operand into TMEM (lane = channel row, KB_COLS = 40 columns = 80 fp16 per chunk, three
    // product terms: edge_build_filter_rows_bwd): columns 384 .. 384 + 40 NCH behind the two groups' accumulators (2 x 2 x
    // 96 columns).  The forward kernel keeps chunk vv in shared memory (its four terms need 48 columns per chunk, 16 more
    // than TMEM has); here the tensor core re-read those 24 KB for every 16-edge tile: 12 of the kernel's 84 shared-memory
    // wavefronts per edge on an LSU data pipe that is 75 % busy (profiles/r02_edge_ncu.md).
    if (tid < 128) {
#pragma unroll
        for (int c = 0; c < NCH; c++) {
            const uint32_t abase = *tmem_slot + BWD_TMEM_A + c * KB_COLS + ((uint32_t)((tid >> 5) * 32) << 16);
            const uint4* src = p.A_rows + ((size_t)c * 128 + tid) * (KB_COLS / 4);
#pragma unroll
            for (int j = 0; j < 2; j++) {
                uint32_t r[16];
#pragma unroll
                for (int q = 0; q < 4; q++) { const uint4 v = src[j * 4 + q]; r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w; }
                tmem_st16(abase + j * 16, r);
            }
            uint32_t r8[8];
#pragma unroll
            for (int q = 0; q < 2; q++) { const uint4 v = src[8 + q]; r8[4 * q] = v.x; r8[4 * q + 1] = v.y; r8[4 * q + 2] = v.z; r8[4 * q + 3] = v.w; }
            tmem_st8(abase + 32, r8);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot + grp * 192;
    const uint32_t tmem_A = *tmem_slot + BWD_TMEM_A;
    const long long N = p.N;
    const int apu = p.atoms_per_unit;
    const int* __restrict__ row_ptr = p.row_ptr;
    const long long n_units = (N + apu - 1) / apu;
    const long long u0 = (long long)blockIdx.x * 2 + grp, ustride = (long long)gridDim.x * 2;
    if (lwarp < 4) reg_inc<168>(); else reg_dec<88>();

    if (lwarp < 4) {
        // ===================== consumers: one channel per thread =====================
        const int f = ltid;
        const float4* __restrict__ Gb = p.Gb + f;
        const float* __restrict__ phi = p.phi + f;
        const float* __restrict__ v_in = p.v_in + f;
        const float* __restrict__ v1b = p.v1b + f;
        float* __restrict__ phib = p.phib + f;
        float* __restrict__ vb_out = p.vb_out + f;
        const uint32_t lane_base = tmem_base + ((uint32_t)(lwarp * 32) << 16);
        // Rolling gather window: the W = 16 next neighbour rows of this thread's channel are always in flight as
        // cp.async copies into private 16-byte shared-memory slots (one commit group per edge, wait_group W-1 before
        // an edge is consumed).  ptxas tracks register-landing loads of different pipeline stages on one scoreboard
        // (measured: the "ping-pong" LDG banks serialised), cp.async groups complete in order by construction.
        float4* ring = (float4*)(gbase + H_OFF_RING) + f;             // slot s of this thread: ring[s * F]
        const float4* __restrict__ ejp = p.ej;
        uint32_t it = 0, hc = 0;          // tile counter, active 8-edge batch counter (selects the partials buffer)
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const int na = (int)min((long long)apu, N - a0);
            const int rp = __ldg(row_ptr + a0 + min(lane, na));
            const int e_begin = __shfl_sync(0xffffffffu, rp, 0), e_end = __shfl_sync(0xffffffffu, rp, na);
            const int n_e = e_end - e_begin;
            const int ntiles = (n_e + NEB - 1) / NEB;
            // sender indices of the unit's edges, 32 per register (lane l <-> edge 32 blk + l); padding slots -> own row
            // (returned raw: padding slots carry ~own row; the sign is folded one batch after the load was issued, so
            // that nothing waits for the load where it is issued)
            auto load_idx = [&](int blk) -> int {
                const int E = e_begin + 32 * blk + lane;
                return E < e_end ? __float_as_int(__ldg(ejp + E).w) : 0;
            };
            int idx0 = load_idx(0), idx1 = load_idx(1);
            idx0 ^= idx0 >> 31;
            idx1 ^= idx1 >> 31;
            int idxn = 0;
            if (ntiles > 0) {
#pragma unroll
                for (int i = 0; i < GWH; i++) {
                    const int j = __shfl_sync(0xffffffffu, idx0, i);
                    if (i < n_e) cp_async16(ring + i * F, Gb + (size_t)j * F);
                    if ((i & 7) == 7) cp_async_commit();            // one commit group per 8-edge batch
                }
            }
            int j_rel = 0;
            int sg = 0;                       // ring slot group of the next batch (batch b of the unit lives in group b % NSG)
            int row_end = __shfl_sync(0xffffffffu, rp, 1);
            // own rows of sender j (current) and j + 1 (prefetched)
            float phS, phVS, phVV = 0.f, vj0 = 0.f, vj1 = 0.f, vj2 = 0.f, r0 = 0.f, r1 = 0.f, r2 = 0.f;
            float nphS = 0.f, nphVS = 0.f, nphVV = 0.f, nvj0 = 0.f, nvj1 = 0.f, nvj2 = 0.f, nr0 = 0.f, nr1 = 0.f, nr2 = 0.f;
            float pbS = 0.f, pbVS = 0.f, Y0 = 0.f, Y1 = 0.f, Y2 = 0.f;
            float vp0 = 0.f, vp1 = 0.f, vp2 = 0.f;                     // phi^vv_j v_j: the vv share of db takes one dot product with it
            auto load_own = [&](long long j, float& a, float& b, float& c, float& x, float& y, float& z, float& q0, float& q1, float& q2) {
                a = phi[j * 3 * F]; b = phi[j * 3 * F + F];
                if (!L0) {
                    c = phi[j * 3 * F + 2 * F];
                    x = v_in[j * 3 * F]; y = v_in[j * 3 * F + F]; z = v_in[j * 3 * F + 2 * F];
                    q0 = v1b[j * 3 * F]; q1 = v1b[j * 3 * F + F]; q2 = v1b[j * 3 * F + 2 * F];
                }
            };
            load_own(a0, phS, phVS, phVV, vj0, vj1, vj2, r0, r1, r2);
            vp0 = phVV * vj0; vp1 = phVV * vj1; vp2 = phVV * vj2;
            if (na > 1) load_own(a0 + 1, nphS, nphVS, nphVV, nvj0, nvj1, nvj2, nr0, nr1, nr2);
            auto store_row = [&]() {
                if (L0) return;
                const long long j = a0 + j_rel;
                phib[j * 3 * F] = pbS;
                phib[j * 3 * F + F] = pbVS;
                phib[j * 3 * F + 2 * F] = vj0 * Y0 + vj1 * Y1 + vj2 * Y2;
                vb_out[j * 3 * F] = r0 + phVV * Y0;
                vb_out[j * 3 * F + F] = r1 + phVV * Y1;
                vb_out[j * 3 * F + 2 * F] = r2 + phVV * Y2;
            };
            auto next_row = [&]() {
                store_row();
                j_rel++;
                row_end = __shfl_sync(0xffffffffu, rp, j_rel + 1);
                phS = nphS; phVS = nphVS; phVV = nphVV; vj0 = nvj0; vj1 = nvj1; vj2 = nvj2; r0 = nr0; r1 = nr1; r2 = nr2;
                vp0 = phVV * vj0; vp1 = phVV * vj1; vp2 = phVV * vj2;
                pbS = pbVS = Y0 = Y1 = Y2 = 0.f;
                if (j_rel + 1 < na) load_own(a0 + j_rel + 1, nphS, nphVS, nphVV, nvj0, nvj1, nvj2, nr0, nr1, nr2);
            };
#define BWD_COMPUTE(H)                                                                                            \
    {                                                                                                             \
        const int k0_ = t * NEB + (H) * 8;                                                                        \
        const int E8_ = e_begin + k0_;                                                                            \
        if (E8_ < e_end) {                                                                                        \
            while (E8_ >= row_end) next_row();                                                                    \
            /* prefetch targets: edges k0 + 16 .. k0 + 23 of the unit, all in index block tb_ */                  \
            const int tb_ = (k0_ + GWH) >> 5, l0_ = (k0_ + GWH) & 31;                                             \
            /* the next index block lands in its own register and is folded into idx0 / idx1 one batch later: */ \
            /* the select below then never reads a register with a load in flight                              */ \
            if (l0_ == 0) idxn = load_idx(tb_ + 1);                                                               \
            if (l0_ == 8) { if (tb_ & 1) idx0 = idxn ^ (idxn >> 31); else idx1 = idxn ^ (idxn >> 31); }           \
            const int isel_ = (tb_ & 1) ? idx1 : idx0;                                                            \
            const bool pf_ = k0_ + GWH < n_e;                                                                     \
            float4* rslot_ = ring + sg * 8 * F;              /* slot group of this batch */                       \
            uint32_t wS_[8], wVS_[8], wVV_[8], dS_[8], dVS_[8], dVV_[8];                                          \
            tmem_ld8_nowait(lane_base + buf * TCOLS + (H) * 8, wS_);                                              \
            tmem_ld8_nowait(lane_base + buf * TCOLS + NEB + (H) * 8, dS_);                                        \
            tmem_ld8_nowait(lane_base + buf * TCOLS + 2 * NEB + (H) * 8, wVS_);                                   \
            tmem_ld8_nowait(lane_base + buf * TCOLS + 3 * NEB + (H) * 8, dVS_);                                   \
            if (!L0) {                                                                                            \
                tmem_ld8_nowait(lane_base + buf * TCOLS + 4 * NEB + (H) * 8, wVV_);                               \
                tmem_ld8_nowait(lane_base + buf * TCOLS + 5 * NEB + (H) * 8, dVV_);                               \
            }                                                                                                     \
            mbar_wait(&p_empty[hc & 1], ((hc >> 1) & 1) ^ 1);           /* partials buffer free again */          \
            tmem_wait_ld();                                                                                       \
            cp_async_wait<NSG - 1>();        /* this batch's rows have landed; the next batches' stay in flight */ \
            uint8_t* pdst_ = sP + (hc & 1) * P4_BYTES;                                                             \
            /* the loads of edge i + BWD_PD are issued before the partials of edge i are stored: ptxas cannot */  \
            /* prove that the stores to sP do not alias the ring, and would otherwise expose the full LDS     */  \
            /* latency once per edge (measured: 25 % of the consumers' time)                                  */  \
            float4 mq_[8], gq_[8];                                                                                \
            _Pragma("unroll") for (int i_ = 0; i_ < BWD_PD; i_++) {                                               \
                mq_[i_] = meta[(H) * 8 + i_];                                                                     \
                gq_[i_] = rslot_[i_ * F];                                                                         \
            }                                                                                                     \
            _Pragma("unroll") for (int i_ = 0; i_ < 8; i_++) {                                                    \
                if (i_ + BWD_PD < 8) {                                                                            \
                    mq_[i_ + BWD_PD] = meta[(H) * 8 + i_ + BWD_PD];                                               \
                    gq_[i_ + BWD_PD] = rslot_[(i_ + BWD_PD) * F];                                                 \
                }                                                                                                 \
                const float4 m_ = mq_[i_];                                                                        \
                const float4 g_ = gq_[i_];                                                                        \
                const float sb_ = g_.x, vb0_ = g_.y, vb1_ = g_.z, vb2_ = g_.w;                                    \
                const float X_ = fmaf(vb0_, m_.x, fmaf(vb1_, m_.y, vb2_ * m_.z));                                 \
                const float wVSf_ = __uint_as_float(wVS_[i_]);                                                    \
                float db_ = (phS * sb_) * __uint_as_float(dS_[i_]);                                               \
                db_ = fmaf(phVS * X_, __uint_as_float(dVS_[i_]), db_);                                            \
                if (!L0) {                                                                                        \
                    const float wVVf_ = __uint_as_float(wVV_[i_]);                                                \
                    const float Z_ = fmaf(vb0_, vp0, fmaf(vb1_, vp1, vb2_ * vp2));      /* phi^vv (vb' . v_j) */  \
                    db_ = fmaf(Z_, __uint_as_float(dVV_[i_]), db_);                                               \
                    pbS = fmaf(__uint_as_float(wS_[i_]), sb_, pbS);                                               \
                    pbVS = fmaf(wVSf_, X_, pbVS);                                                                 \
                    Y0 = fmaf(wVVf_, vb0_, Y0); Y1 = fmaf(wVVf_, vb1_, Y1); Y2 = fmaf(wVVf_, vb2_, Y2);           \
                }                                                                                                 \
                /* this channel's share of g_e = db u + (ub - (ub.u) u) / d with ub = beta' vb', beta' = w^vs phi^vs: */ \
                /* the planes (db, ub) are summed over the channels first; u, 1/d and the projection are applied   */ \
                /* once per edge by the reducer (sum_c ub_c . u = u . sum_c ub_c)                                   */ \
                const float bq_ = wVSf_ * phVS;                                                                   \
                float* pd_ = (float*)(pdst_ + i_ * P4_ROW) + f;         /* four planes of 128 floats per edge */  \
                pd_[0] = db_;                                                                                     \
                pd_[F] = bq_ * vb0_;                                                                              \
                pd_[2 * F] = bq_ * vb1_;                                                                          \
                pd_[3 * F] = bq_ * vb2_;                                                                          \
            }                                                                                                     \
            /* re-arm the 8 slots with the rows of edges k0 + 16 .. k0 + 23 (one commit group, also when empty) */ \
            _Pragma("unroll") for (int i_ = 0; i_ < 8; i_++) {                                                    \
                const int jn_ = __shfl_sync(0xffffffffu, isel_, l0_ + i_);                                        \
                if (pf_) cp_async16(rslot_ + i_ * F, Gb + (size_t)jn_ * F);                                       \
            }                                                                                                     \
            cp_async_commit();                                                                                    \
            if (++sg == NSG) sg = 0;                                                                              \
            bar_arrive(NB_PF + (hc & 1), 160);                          /* hand the batch to the reducer warp */  \
            hc++;                                                                                                 \
        }                                                                                                         \
    }
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                const float4* meta = sMeta + (it & 3) * NEB;
                mbar_wait(&t_full[buf], (it >> 1) & 1);
                tc_fence_after();
                BWD_COMPUTE(0);
                BWD_COMPUTE(1);
                tc_fence_before();
                bar_arrive(NB_TE + buf, 160);
            }
            cp_async_wait<0>();           // slots are re-armed by the next unit's prologue
            for (;;) {
                store_row();
                if (j_rel + 1 >= na) break;
                // trailing edge-less senders: phib = 0, vb_out = v1b
                j_rel++;
                phS = nphS; phVS = nphVS; phVV = nphVV; vj0 = nvj0; vj1 = nvj1; vj2 = nvj2; r0 = nr0; r1 = nr1; r2 = nr2;
                pbS = pbVS = Y0 = Y1 = Y2 = 0.f;
                if (j_rel + 1 < na) load_own(a0 + j_rel + 1, nphS, nphVS, nphVV, nvj0, nvj1, nvj2, nr0, nr1, nr2);
            }
        }
#undef BWD_COMPUTE
    } else if (lwarp == 4 + grp) {
        // ===================== producer: rows 0..15 R_e, rows 16..31 R'_e =====================
        // (helper roles sit on different schedulers in the two pipelines: producer on 0 | 1, reducer on 2 | 3, MMA issuer on 3 | 2)
        // ONE warp per pipeline: lane = (edge e of the tile, half hh): basis slots 12 hh .. 12 hh + 11 (slot 0 = bias).  The
        // per-edge part (record, 1/d, sincospi, cutoff) is evaluated twice per edge instead of four times (round 1 / 2 used
        // two warps with one 8-slot group per thread and an idle quarter), and R' comes from the closed form
        //   R'_n = sin(n pi x) A + cos(n pi x) n B,   A = (fc' - fc / d) / d,   B = (pi / rc) fc / d,   R_n = sin(n pi x) fc / d
        // (3 instructions per slot instead of 6): 330 instead of 740 warp instructions per 16-edge tile -- the producers were
        // a sixth of all instructions this kernel issues (profiles/r02_edge_ncu.md).
        const int e = lane & 15, hh = lane >> 4;
        const float inv_rc = p.inv_rc;
        const float a1c = 3.14159265358979323846f * inv_rc;
        const int K = p.K;
        // the thread's 12 slots are three 8-byte pieces of a B row (4 fp16 each): piece j holds slots 12 hh + 4 j .. + 3,
        // i.e. bytes ((12 hh + 4 j) & 7) * 2 .. of the 16-byte chunk (12 hh + 4 j) >> 3 of every product term
        int poff[3];
#pragma unroll
        for (int j = 0; j < 3; j++) { const int sl = 12 * hh + 4 * j; poff[j] = (sl >> 3) * 128 + (sl & 7) * 2; }
        uint32_t it = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const long long a1 = min(N, a0 + (long long)apu);
            const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            float4 raw_n = load_edge_raw(p.ej, e_begin + e, e_end);
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                const float4 raw = raw_n;
                if (t + 1 < ntiles) raw_n = load_edge_raw(p.ej, e_begin + (t + 1) * NEB + e, e_end);
                const EdgeGeom g = edge_geom(raw, e_begin + t * NEB + e, e_end, inv_rc);
                const float fc = g.real ? 0.5f * (1.0f + g.c1) : 0.0f;
                const float dfc = g.real ? -0.5f * a1c * g.s1 : 0.0f;
                const float amp = fc * g.inv_d;                       // R_n = amp sin(n pi x)
                const float cA = (dfc - amp) * g.inv_d, cB = a1c * amp;
                float sn_, cn_;
                sincospif(12.0f * g.x, &sn_, &cn_);                   // first slot of the upper half (the lower half starts at slot 1)
                if (hh == 0) { sn_ = g.s1; cn_ = g.c1; }
                float nB = hh == 0 ? cB : 12.0f * cB;                 // n B of the current slot
                uint2 q[2][3][3];                                     // [R | R'][term][piece]
#pragma unroll
                for (int j = 0; j < 3; j++) {
                    float vals[4], dvals[4];
#pragma unroll
                    for (int i = 0; i < 4; i++) {
                        const int sl = 4 * j + i;                     // slot 12 hh + sl
                        if (sl == 0) {                                // (hh == 0: the bias slot; hh == 1: slot 12, an ordinary one)
                            const bool ok = 12 <= K;
                            vals[i] = hh == 0 ? fc : (ok ? amp * sn_ : 0.0f);
                            dvals[i] = hh == 0 ? dfc : (ok ? fmaf(sn_, cA, cn_ * nB) : 0.0f);
                            if (hh == 0) continue;                    // (uniform per half-warp; the rotation below is skipped for the bias)
                        } else {
                            const bool ok = 12 * hh + sl <= K;
                            vals[i] = ok ? amp * sn_ : 0.0f;
                            dvals[i] = ok ? fmaf(sn_, cA, cn_ * nB) : 0.0f;
                        }
                        const float tt = sn_ * g.c1 + cn_ * g.s1;
                        cn_ = cn_ * g.c1 - sn_ * g.s1;
                        sn_ = tt;
                        nB += cB;
                    }
#pragma unroll
                    for (int z = 0; z < 2; z++) {
                        const float* v = z ? dvals : vals;
                        const __half2 k64 = __floats2half2_rn(1.0f / 64.0f, 1.0f / 64.0f);
                        __half2 h_hh[2], h_hl[2], h_lh[2];
#pragma unroll
                        for (int w = 0; w < 2; w++) {                 // split3b on two values at a time
                            h_hh[w] = __floats2half2_rn(v[2 * w], v[2 * w + 1]);
                            const float2 f = __half22float2(h_hh[w]);
                            h_hl[w] = __floats2half2_rn((v[2 * w] - f.x) * 64.0f, (v[2 * w + 1] - f.y) * 64.0f);
                            h_lh[w] = __hmul2(h_hh[w], k64);
                        }
                        q[z][0][j] = make_uint2(*(uint32_t*)&h_hl[0], *(uint32_t*)&h_hl[1]);     // term 0: r 2^6
                        q[z][1][j] = make_uint2(*(uint32_t*)&h_lh[0], *(uint32_t*)&h_lh[1]);     // term 1: hi 2^-6
                        q[z][2][j] = make_uint2(*(uint32_t*)&h_hh[0], *(uint32_t*)&h_hh[1]);     // term 2: hi
                    }
                }
                __syncwarp();
                if (it >= 2) bar_sync(NB_TE + buf, 160);          // tile it - 2 consumed: B operand / TMEM buffer free
#pragma unroll
                for (int z = 0; z < 2; z++) {
                    const int row = z * NEB + e;
                    uint8_t* bb = sB + buf * BB_BYTES + (row >> 3) * SBO + (row & 7) * 16;
#pragma unroll
                    for (int tm = 0; tm < 3; tm++)
#pragma unroll
                        for (int j = 0; j < 3; j++) *(uint2*)(bb + tm * 3 * 128 + poff[j]) = q[z][tm][j];
                }
                if (hh == 0) sMeta[(it & 3) * NEB + e] = make_float4(-g.r.x * g.inv_d, -g.r.y * g.inv_d, -g.r.z * g.inv_d, g.inv_d);   // u_e of edge (i <- j), 1/d
                fence_async_smem();
                __syncwarp();
                bar_arrive(NB_BF + buf, 64);
            }
        }
    } else if (lwarp == 6 + grp) {
        // ===================== reducer: sum the partials over the 128 channels, assemble g_e, accumulate G =====================
        // lane = (edge of the batch, quarter of the channels): 32 conflict-free LDS.128 + two shuffle stages per batch
        const int re = lane >> 2, rsub = lane & 3;
        float4* __restrict__ Gout = p.G;
        const bool first = p.first != 0;
        uint32_t it = 0, hc = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const long long a1 = min(N, a0 + (long long)apu);
            const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            for (int t = 0; t < ntiles; t++, it++) {
                for (int h = 0; h < 2; h++) {
                    const int E8 = e_begin + t * NEB + h * 8;
                    if (E8 >= e_end) continue;
                    const int E = E8 + re;
                    float4 gold = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (rsub == 0 && !first) gold = Gout[E];                  // running sum over layers, fetched early
                    bar_sync(NB_PF + (hc & 1), 160);
                    // this lane adds a quarter (chunks rsub + 4 k) of each of the four 128-float planes of row re
                    const uint8_t* src = sP + (hc & 1) * P4_BYTES + re * P4_ROW + rsub * 16;
                    const float4 mt = sMeta[(it & 3) * NEB + h * 8 + re];      // (u_e, 1 / d_e)
                    unsigned long long ad = 0ull, ax = 0ull, ay = 0ull, az = 0ull;      // packed (+0.f, +0.f)
#pragma unroll
                    for (int k = 0; k < 8; k++) {
                        const ulonglong2 d = *(const ulonglong2*)(src + k * 64);
                        const ulonglong2 x = *(const ulonglong2*)(src + F * 4 + k * 64);
                        const ulonglong2 y = *(const ulonglong2*)(src + 2 * F * 4 + k * 64);
                        const ulonglong2 z = *(const ulonglong2*)(src + 3 * F * 4 + k * 64);
                        ad = fadd2(ad, fadd2(d.x, d.y));
                        ax = fadd2(ax, fadd2(x.x, x.y));
                        ay = fadd2(ay, fadd2(y.x, y.y));
                        az = fadd2(az, fadd2(z.x, z.y));
                    }
                    float db = hsum2(ad);
                    float3 ub = make_float3(hsum2(ax), hsum2(ay), hsum2(az));
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&p_empty[hc & 1]);
                    hc++;
#pragma unroll
                    for (int o = 2; o >= 1; o >>= 1) {
                        db += __shfl_xor_sync(0xffffffffu, db, o);
                        ub.x += __shfl_xor_sync(0xffffffffu, ub.x, o);
                        ub.y += __shfl_xor_sync(0xffffffffu, ub.y, o);
                        ub.z += __shfl_xor_sync(0xffffffffu, ub.z, o);
                    }
                    // g_e = db u + (ub - (ub . u) u) / d
                    ub.x *= mt.w; ub.y *= mt.w; ub.z *= mt.w;
                    const float al = db - (ub.x * mt.x + ub.y * mt.y + ub.z * mt.z);
                    const float3 acc = make_float3(fmaf(al, mt.x, ub.x), fmaf(al, mt.y, ub.y), fmaf(al, mt.z, ub.z));
                    if (rsub == 0) Gout[E] = make_float4(gold.x + acc.x, gold.y + acc.y, gold.z + acc.z, 0.f);
                }
            }
        }
    } else if (lwarp == 7 - grp) {
        // ===================== MMA issuer (lane 0; the whole warp waits on the producers' named barrier) =====================
        const uint32_t idesc = (1u << 4) | ((uint32_t)((2 * NEB) >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        const uint32_t b_base = smem_u32(sB);
        uint32_t it = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const long long a1 = min(N, a0 + (long long)apu);
            const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                bar_sync(NB_BF + buf, 64);
                tc_fence_after();
                if (elect_one()) {
#pragma unroll
                    for (int c = 0; c < NCH; c++) {
                        const uint32_t d = tmem_base + buf * TCOLS + c * 2 * NEB;
#pragma unroll
                        for (int kk = 0; kk < KB_COLS / 8; kk++) {     // ascending K: cross terms first, the hh term last
                            const uint64_t bd = make_desc_nosw(b_base + buf * BB_BYTES + kk * 2 * LBO, LBO, SBO);
                            umma_f16_ts(d, tmem_A + c * KB_COLS + kk * 8, bd, idesc, kk != 0);
                        }
                    }
                    umma_commit(&t_full[buf]);
                }
                __syncwarp();
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (tid >> 5 == 15) tmem_dealloc(*tmem_slot, 512);
}

// =============================================================================================================
// layer-0 adjoint: only the geometry gradient is wanted (the embedding is constant) and the sender rows
// (phi^s_j, phi^vs_j) depend on the species of j only.  The pass therefore walks the RECEIVER's row with the
// receiver's own (sb'_i, vb'_i) in registers and looks the sender up in the species table: no neighbour-row gather
// at all.  g of edge (i <- j) is produced at the slot of i's row; G is indexed by the slot of the sender's row
// (force_final: F_a = sum_x G[rev x] - G[x]), so the reducer scatters through the reverse-edge index.
// =============================================================================================================
struct Bwd0Params {
    long long N;
    const int* row_ptr;
    const float4* ej;
    const float4* Gb;      // (sb', vb'_x, vb'_y, vb'_z) per atom and channel
    const int* types;
    const float2* tab;     // [n_tab][F] (phi^s, phi^vs) per species
    const int* rev;
    const uint4* A_img;    // [>= 2 chunks][128 rows][80 fp16] rows (edge_build_filter_rows): TMEM-resident A operand
    float4* G;
    float inv_rc;
    int K;
    int atoms_per_unit;
    int first;
    int n_tab;
};
constexpr int G0_OFF_SPEC = G_OFF_BAR + 128, G0_OFF_TAB = G0_OFF_SPEC + 4 * NEB * 4, GROUP0_BYTES = G0_OFF_TAB;
constexpr int bwd0_smem_bytes() { return 2 * GROUP0_BYTES + TAB_MAX * F * 8 + 128; }
constexpr int BWD0_TMEM_A = 128;                        // TMEM columns 128..207: the filter operand (2 chunks x 40 columns)

__global__ void __launch_bounds__(BWD_THREADS, 1) k_msg_bwd0(const Bwd0Params p) {
    constexpr int NCH = 2;
    constexpr int TCOLS = NCH * 2 * NEB;
    extern __shared__ __align__(128) uint8_t smem[];
    const int tid = threadIdx.x, grp = tid >> 8, ltid = tid & 255, lwarp = ltid >> 5, lane = tid & 31;
    uint8_t* gbase = smem + grp * GROUP0_BYTES;
    uint8_t* sB = gbase + G_OFF_B;
    uint8_t* sP = gbase + G_OFF_P;
    float4* sMeta = (float4*)(gbase + G_OFF_META);  // [4][NEB] (u_e, 1/d_e)
    int* sSpec = (int*)(gbase + G0_OFF_SPEC);       // [4][NEB] species of the sender
    uint64_t* bars = (uint64_t*)(gbase + G_OFF_BAR);
    uint64_t* t_full = bars;
    uint64_t* p_empty = bars + 2;
    const int NB_TE = 1 + grp * 6, NB_BF = NB_TE + 2, NB_PF = NB_TE + 4;
    float2* sTab = (float2*)(smem + 2 * GROUP0_BYTES);
    uint32_t* tmem_slot = (uint32_t*)(sTab + TAB_MAX * F);
    {
        uint4* zb = (uint4*)sB;
        for (int i = ltid; i < 2 * BB_BYTES / 16; i += 256) zb[i] = make_uint4(0, 0, 0, 0);
        for (int i = tid; i < p.n_tab * F; i += BWD_THREADS) sTab[i] = p.tab[i];
    }
    if (ltid == 0) {
        for (int b = 0; b < 2; b++) { mbar_init(&t_full[b], 1); mbar_init(&p_empty[b], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid >> 5 == 15) tmem_alloc(tmem_slot, 512);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    // filter operand into TMEM (lane = channel row, KB_COLS = 40 columns = 80 fp16 per chunk): the MMAs read only the small
    // B operand from shared memory
    if (tid < 128) {
#pragma unroll
        for (int c = 0; c < NCH; c++) {
            const uint32_t abase = *tmem_slot + BWD0_TMEM_A + c * KB_COLS + ((uint32_t)((tid >> 5) * 32) << 16);
            const uint4* src = p.A_img + ((size_t)c * 128 + tid) * (KB_COLS / 4);
#pragma unroll
            for (int j = 0; j < 2; j++) {
                uint32_t r[16];
#pragma unroll
                for (int q = 0; q < 4; q++) { const uint4 v = src[j * 4 + q]; r[4 * q] = v.x; r[4 * q + 1] = v.y; r[4 * q + 2] = v.z; r[4 * q + 3] = v.w; }
                tmem_st16(abase + j * 16, r);
            }
            uint32_t r8[8];
#pragma unroll
            for (int q = 0; q < 2; q++) { const uint4 v = src[8 + q]; r8[4 * q] = v.x; r8[4 * q + 1] = v.y; r8[4 * q + 2] = v.z; r8[4 * q + 3] = v.w; }
            tmem_st8(abase + 32, r8);
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot + grp * 256;
    const uint32_t tmem_A = *tmem_slot + BWD0_TMEM_A;
    const long long N = p.N;
    const int apu = p.atoms_per_unit;
    const int* __restrict__ row_ptr = p.row_ptr;
    const long long n_units = (N + apu - 1) / apu;
    const long long u0 = (long long)blockIdx.x * 2 + grp, ustride = (long long)gridDim.x * 2;
    if (lwarp < 4) reg_inc<168>(); else reg_dec<88>();

    if (lwarp < 4) {
        // ===================== consumers: one channel per thread, receiver rows =====================
        const int f = ltid;
        const float4* __restrict__ Gb = p.Gb + f;
        const uint32_t lane_base = tmem_base + ((uint32_t)(lwarp * 32) << 16);
        uint32_t it = 0, hc = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const int na = (int)min((long long)apu, N - a0);
            const int rp = __ldg(row_ptr + a0 + min(lane, na));
            const int e_begin = __shfl_sync(0xffffffffu, rp, 0), e_end = __shfl_sync(0xffffffffu, rp, na);
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            int i_rel = 0;
            int row_end = __shfl_sync(0xffffffffu, rp, 1);
            float4 own = Gb[a0 * F], nown = na > 1 ? Gb[(a0 + 1) * F] : own;      // (sb', vb') of receiver i, i + 1
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                const float4* meta = sMeta + (it & 3) * NEB;
                const int* spec = sSpec + (it & 3) * NEB;
                mbar_wait(&t_full[buf], (it >> 1) & 1);
                tc_fence_after();
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const int E8 = e_begin + t * NEB + h * 8;
                    if (E8 < e_end) {
                        while (E8 >= row_end) {
                            i_rel++;
                            row_end = __shfl_sync(0xffffffffu, rp, i_rel + 1);
                            own = nown;
                            if (i_rel + 1 < na) nown = Gb[(a0 + i_rel + 1) * F];
                        }
                        uint32_t dS[8], wVS[8], dVS[8];
                        tmem_ld8_nowait(lane_base + buf * TCOLS + NEB + h * 8, dS);
                        tmem_ld8_nowait(lane_base + buf * TCOLS + 2 * NEB + h * 8, wVS);
                        tmem_ld8_nowait(lane_base + buf * TCOLS + 3 * NEB + h * 8, dVS);
                        mbar_wait(&p_empty[hc & 1], ((hc >> 1) & 1) ^ 1);
                        tmem_wait_ld();
                        uint8_t* pdst = sP + (hc & 1) * P_BYTES;
                        // all shared-memory reads of the batch before its first store (see BWD_PD in k_msg_bwd)
                        float4 mq[8];
                        float2 pq[8];
#pragma unroll
                        for (int i = 0; i < 8; i++) {
                            mq[i] = meta[h * 8 + i];
                            pq[i] = sTab[spec[h * 8 + i] * F + f];
                        }
#pragma unroll
                        for (int i = 0; i < 8; i++) {
                            const float4 m = mq[i];
                            const float2 ph = pq[i];
                            const float X = fmaf(own.y, m.x, fmaf(own.z, m.y, own.w * m.z));
                            float db = ph.x * (own.x * __uint_as_float(dS[i]));
                            db = fmaf(ph.y, X * __uint_as_float(dVS[i]), db);
                            const float beta = __uint_as_float(wVS[i]) * ph.y * m.w;
                            const float alpha = fmaf(-beta, X, db);
                            float* pd = (float*)(pdst + i * P_ROW) + f;
                            pd[0] = fmaf(alpha, m.x, beta * own.y);
                            pd[F] = fmaf(alpha, m.y, beta * own.z);
                            pd[2 * F] = fmaf(alpha, m.z, beta * own.w);
                        }
                        bar_arrive(NB_PF + (hc & 1), 160);
                        hc++;
                    }
                }
                tc_fence_before();
                bar_arrive(NB_TE + buf, 192);
            }
        }
    } else if (lwarp < 6) {
        // ===================== producers: rows 0..15 R_e, rows 16..31 R'_e; meta (u_e, 1/d), species =====================
        const int pt = ltid - 128, e = pt & 15, h = pt >> 4;
        const float inv_rc = p.inv_rc;
        const float a1c = 3.14159265358979323846f * inv_rc;
        const int K = p.K;
        uint32_t it = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const long long a1 = min(N, a0 + (long long)apu);
            const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            float4 raw_n = load_edge_raw(p.ej, e_begin + e, h < 3 ? e_end : 0);
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                uint4 q[6];
                float4 meta_v = make_float4(0.f, 0.f, 0.f, 0.f);
                const float4 raw = raw_n;
                if (t + 1 < ntiles) raw_n = load_edge_raw(p.ej, e_begin + (t + 1) * NEB + e, h < 3 ? e_end : 0);
                int spec_v = 0;
                if (h < 3) {
                    const EdgeGeom g = edge_geom(raw, e_begin + t * NEB + e, e_end, inv_rc);
                    if (h == 0) spec_v = __ldg(p.types + __float_as_int(g.r.w));
                    const float fc = g.real ? 0.5f * (1.0f + g.c1) : 0.0f;
                    const float dfc = g.real ? -0.5f * a1c * g.s1 : 0.0f;
                    float sn_, cn_;
                    if (h == 0) { sn_ = g.s1; cn_ = g.c1; } else sincospif((float)(8 * h) * g.x, &sn_, &cn_);
                    float vals[8], dvals[8];
#pragma unroll
                    for (int i = 0; i < 8; i++) {
                        const int b = h * 8 + i;
                        if (b == 0) { vals[i] = fc; dvals[i] = dfc; }
                        else {
                            const float rho = sn_ * g.inv_d;
                            const float drho = ((float)b * a1c * cn_ - rho) * g.inv_d;
                            vals[i] = b <= K ? fc * rho : 0.0f;
                            dvals[i] = b <= K ? dfc * rho + fc * drho : 0.0f;
                            const float tt = sn_ * g.c1 + cn_ * g.s1;
                            cn_ = cn_ * g.c1 - sn_ * g.s1;
                            sn_ = tt;
                        }
                    }
                    split3b(vals, q[0], q[1], q[2]);
                    split3b(dvals, q[3], q[4], q[5]);
                    meta_v = make_float4(g.r.x * g.inv_d, g.r.y * g.inv_d, g.r.z * g.inv_d, g.inv_d);
                }
                __syncwarp();
                if (it >= 2) bar_sync(NB_TE + buf, 192);
                if (h < 3) {
#pragma unroll
                    for (int z = 0; z < 2; z++) {
                        const int row = z * NEB + e;
                        uint8_t* bb = sB + buf * BB_BYTES + (row >> 3) * SBO + (row & 7) * 16;
#pragma unroll
                        for (int tm = 0; tm < 3; tm++) *(uint4*)(bb + kgrp_off(tm, h)) = q[3 * z + tm];
                    }
                    if (h == 0) { sMeta[(it & 3) * NEB + e] = meta_v; sSpec[(it & 3) * NEB + e] = spec_v; }
                }
                fence_async_smem();
                __syncwarp();
                bar_arrive(NB_BF + buf, 96);
            }
        }
    } else if (lwarp == 6) {
        // ===================== reducer: channel sums, scatter into the sender-row slot =====================
        // The scatter target rev[E] and the running sum G[rev[E]] (a random 16-byte row, usually from DRAM) are two
        // dependent global loads per batch: issued where they are needed, their latencies (~1.5 us per batch) were the
        // bound of the whole kernel (measured: consumers 46 % of their time waiting for the partials buffer).  The
        // reducer therefore runs them ahead: rev in coalesced 32-edge blocks (one register per lane, two blocks in
        // flight, the target of a batch taken by shuffle), G of batch b + 1 while batch b is reduced.  The loop is
        // unrolled over two blocks so that every register choice is static (a select between a landed and a pending
        // register would wait for both).
        const int re = lane >> 2, rsub = lane & 3;
        float4* __restrict__ Gout = p.G;
        const bool want_old = p.first == 0 && rsub == 0;
        const int* __restrict__ rev = p.rev;
        uint32_t hc = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const long long a1 = min(N, a0 + (long long)apu);
            const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
            const int nb = (e_end - e_begin + 7) >> 3;                 // 8-edge batches of the unit (rows are padded to 8)
            auto ld_blk = [&](int blk) -> int {
                const int E = e_begin + 32 * blk + lane;
                return E < e_end ? __ldg(rev + E) : 0;
            };
            int rA = ld_blk(0), rB = ld_blk(1);
            int tcur = __shfl_sync(0xffffffffu, rA, re);
            float4 gc = make_float4(0.f, 0.f, 0.f, 0.f);
            if (want_old && nb > 0) gc = Gout[tcur];
            for (int b0 = 0; b0 < nb; b0 += 8) {
#pragma unroll
                for (int i = 0; i < 8; i++) {
                    const int b = b0 + i;
                    if (b >= nb) break;
                    if (i == 0 && b0 > 0) rB = ld_blk((b0 >> 2) + 1);
                    if (i == 4) rA = ld_blk((b0 >> 2) + 2);
                    const int tnext = __shfl_sync(0xffffffffu, (((i + 1) >> 2) & 1) ? rB : rA, ((i + 1) & 3) * 8 + re);
                    float4 gn = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (want_old && b + 1 < nb) gn = Gout[tnext];
                    bar_sync(NB_PF + (hc & 1), 160);
                    const uint8_t* src = sP + (hc & 1) * P_BYTES + re * P_ROW + rsub * 16;
                    unsigned long long ax = 0ull, ay = 0ull, az = 0ull;      // packed (+0.f, +0.f)
#pragma unroll
                    for (int k = 0; k < 8; k++) {
                        const ulonglong2 x = *(const ulonglong2*)(src + k * 64);
                        const ulonglong2 y = *(const ulonglong2*)(src + F * 4 + k * 64);
                        const ulonglong2 z = *(const ulonglong2*)(src + 2 * F * 4 + k * 64);
                        ax = fadd2(ax, fadd2(x.x, x.y));
                        ay = fadd2(ay, fadd2(y.x, y.y));
                        az = fadd2(az, fadd2(z.x, z.y));
                    }
                    float3 acc = make_float3(hsum2(ax), hsum2(ay), hsum2(az));
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&p_empty[hc & 1]);
                    hc++;
#pragma unroll
                    for (int o = 2; o >= 1; o >>= 1) {
                        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o);
                        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
                        acc.z += __shfl_xor_sync(0xffffffffu, acc.z, o);
                    }
                    if (rsub == 0) Gout[tcur] = make_float4(gc.x + acc.x, gc.y + acc.y, gc.z + acc.z, 0.f);
                    tcur = tnext;
                    gc = gn;
                }
            }
        }
    } else if (lwarp == 7) {
        // ===================== MMA issuer =====================
        const uint32_t idesc = (1u << 4) | ((uint32_t)((2 * NEB) >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        const uint32_t b_base = smem_u32(sB);
        uint32_t it = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * apu;
            const long long a1 = min(N, a0 + (long long)apu);
            const int e_begin = __ldg(row_ptr + a0), e_end = __ldg(row_ptr + a1);
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                bar_sync(NB_BF + buf, 96);
                tc_fence_after();
                if (elect_one()) {
#pragma unroll
                    for (int c = 0; c < NCH; c++) {
                        const uint32_t d = tmem_base + buf * TCOLS + c * 2 * NEB;
#pragma unroll
                        for (int kk = 0; kk < KB_COLS / 8; kk++) {
                            const uint64_t bd = make_desc_nosw(b_base + buf * BB_BYTES + kk * 2 * LBO, LBO, SBO);
                            umma_f16_ts(d, tmem_A + c * KB_COLS + kk * 8, bd, idesc, kk != 0);
                        }
                    }
                    umma_commit(&t_full[buf]);
                }
                __syncwarp();
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (tid >> 5 == 15) tmem_dealloc(*tmem_slot, 512);
}

}  // namespace ev3

// gather rows: Q4[j][f] = (phi^s, phi^vs, phi^vv v_x, phi^vv v_y), Q1[j][f] = phi^vv v_z ; layer 0 (v = 0): Q2 = (phi^s, phi^vs)
__global__ void k_make_gather(long long N, const float* __restrict__ phi, const float* __restrict__ v,
                              float4* __restrict__ Q4, float* __restrict__ Q1, float2* __restrict__ Q2, int has_v) {
    constexpr int F = ev3::F;
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
// gather rows of the adjoint pass: Gb[i][f] = (sb', vb'_x, vb'_y, vb'_z)
__global__ void k_make_gather_bwd(long long N, const float* __restrict__ s1b, const float* __restrict__ v1b,
                                  float4* __restrict__ Gb) {
    constexpr int F = ev3::F;
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F) return;
    const long long j = idx / F;
    const int f = (int)(idx - j * F);
    Gb[idx] = make_float4(s1b[idx], v1b[j * 3 * F + f], v1b[j * 3 * F + F + f], v1b[j * 3 * F + 2 * F + f]);
}
void make_gather_rows(const Launch& L, long long N, const float* phi, const float* v, float* Q4, float* Q1, bool has_v) {
    if (N == 0) return;
    k_make_gather<<<(unsigned)((N * ev3::F + 255) / 256), 256, 0, L.stream>>>(N, phi, v, (float4*)Q4, Q1, (float2*)Q4, has_v ? 1 : 0);
    KLAUNCH(L);
}
void make_gather_rows_bwd(const Launch& L, long long N, const float* s1b, const float* v1b, float* Gb) {
    if (N == 0) return;
    k_make_gather_bwd<<<(unsigned)((N * ev3::F + 255) / 256), 256, 0, L.stream>>>(N, s1b, v1b, (float4*)Gb);
    KLAUNCH(L);
}

// host: the three fp16 planes of one filter weight w = hi + r, term order (hl, lh, hh) as in split3b:  hi 2^-6 | r 2^6 | hi
static void filter_planes(float w, unsigned short (&bits)[3]) {
    const __half hi = __float2half_rn(w);
    const float hif = __half2float(hi), r = w - hif;
    const __half vals[3] = {__float2half_rn(hif * (1.0f / 64.0f)), __float2half_rn(r * 64.0f), hi};
    for (int t = 0; t < 3; t++) memcpy(&bits[t], &vals[t], 2);
}
// host: filter operand (bf | Wf) of one layer as plain rows [3 chunks][128 channels][80 fp16], k = 24 term + basis slot
// (basis slot 0 = the bias bf), k >= 72 zero -- the TMEM-resident A operand of every tensor-core edge kernel
void edge_build_filter_rows(const float* Wf, const float* bf, int K, std::vector<unsigned short>& img) {
    img.assign((size_t)3 * ev3::F * ev3::KB, 0);
    for (int c = 0; c < 3; c++)
        for (int r = 0; r < ev3::F; r++)
            for (int b = 0; b <= K; b++) {
                const float w = b == 0 ? bf[c * ev3::F + r] : Wf[(size_t)(c * ev3::F + r) * K + (b - 1)];
                unsigned short bits[3];
                filter_planes(w, bits);
                for (int t = 0; t < 3; t++) img[((size_t)c * ev3::F + r) * ev3::KB + t * 24 + b] = bits[t];
            }
}

static int sm_count() {
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    return n_sm;
}

// F = 128, K <= 23 only.  Q4/Q1 from make_gather_rows; A_rows from edge_build_filter_rows.  has_v = false:
// layer 0 through the species table.
bool message_fwd_v3(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* s,
                    const float* v, const float* Q4, const float* Q1, const void* A_rows, float* sn, float* v1,
                    bool has_v, const int* types_s, const float* tab, int n_tab, const float2* xph) {
    using namespace ev3;
    if (N == 0) return true;
    if (K > 23 || !A_rows) return false;
    if (!has_v && (!tab || !types_s || n_tab > TAB_MAX)) return false;
    static bool attr = false;
    if (!attr) {
        if (cudaFuncSetAttribute(k_msg_fwd_g<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, fwdg_smem_bytes(true)) != cudaSuccess ||
            cudaFuncSetAttribute(k_msg_fwd_g<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, fwdg_smem_bytes(false)) != cudaSuccess)
            return false;
        attr = true;
    }
    FwdParams p{N, row_ptr, ej, s, v, (const float4*)Q4, Q1, (const float2*)Q4, (const uint4*)A_rows, sn, v1,
                1.0f / rc, K, L.apu_fwd, types_s, (const float2*)tab, n_tab, xph};
    const long long n_units = (N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    // one CTA per SM, two 8-warp pipelines sharing the TMEM-resident filter operand
    const int grid = (int)std::min<long long>((n_units + 1) / 2, (long long)sm_count());
    if (has_v) k_msg_fwd_g<true><<<grid, FWDG_THREADS, fwdg_smem_bytes(true), L.stream>>>(p);
    else k_msg_fwd_g<false><<<grid, FWDG_THREADS, fwdg_smem_bytes(false), L.stream>>>(p);
    KLAUNCH(L);
    return true;
}

// layer0: v_in = 0 and no sender adjoint wanted (phib / vb_out untouched)
bool message_bwd_v3(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* Gb,
                    const float* phi, const float* v_in, const float* v1b, const void* A_rows, float* phib,
                    float* vb_out, float4* G, bool first, bool layer0) {
    using namespace ev3;
    if (N == 0) return true;
    if (K > 23 || !A_rows) return false;
    static bool attr = false;
    if (!attr) {
        if (cudaFuncSetAttribute(k_msg_bwd<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bwd_smem_bytes(2)) != cudaSuccess ||
            cudaFuncSetAttribute(k_msg_bwd<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bwd_smem_bytes(3)) != cudaSuccess)
            return false;
        attr = true;
    }
    BwdParams p{N, row_ptr, ej, (const float4*)Gb, phi, v_in, v1b, (const uint4*)A_rows, phib, vb_out, G,
                1.0f / rc, K, L.apu_bwd, first ? 1 : 0};
    const long long n_units = (N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    const int grid = (int)std::min<long long>((n_units + 1) / 2, (long long)sm_count());
    if (layer0) k_msg_bwd<true><<<grid, BWD_THREADS, bwd_smem_bytes(2), L.stream>>>(p);
    else k_msg_bwd<false><<<grid, BWD_THREADS, bwd_smem_bytes(3), L.stream>>>(p);
    KLAUNCH(L);
    return true;
}

// layer-0 adjoint through the species table (see k_msg_bwd0); G indexed as everywhere else (slot of the sender's row)
bool message_bwd0_v3(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* Gb,
                     const int* types_s, const float* tab, int n_tab, const int* rev, const void* A_img, float4* G, bool first) {
    using namespace ev3;
    if (N == 0) return true;
    if (K > 23 || !tab || n_tab > TAB_MAX) return false;
    static bool attr = false;
    if (!attr) {
        if (cudaFuncSetAttribute(k_msg_bwd0, cudaFuncAttributeMaxDynamicSharedMemorySize, bwd0_smem_bytes()) != cudaSuccess) return false;
        attr = true;
    }
    Bwd0Params p{N, row_ptr, ej, (const float4*)Gb, types_s, (const float2*)tab, rev, (const uint4*)A_img, G, 1.0f / rc, K, L.apu_bwd,
                 first ? 1 : 0, n_tab};
    const long long n_units = (N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    const int grid = (int)std::min<long long>((n_units + 1) / 2, (long long)sm_count());
    k_msg_bwd0<<<grid, BWD_THREADS, bwd0_smem_bytes(), L.stream>>>(p);
    KLAUNCH(L);
    return true;
}

}  // namespace painn
