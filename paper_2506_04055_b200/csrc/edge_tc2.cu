// edge_tc2.cu -- second-generation adjoint message kernel (F = 128): same mathematics and thread mapping as
// edge_tc.cu::k_message_bwd_tc (one channel per TMEM lane, gather form, finisher warp), with two changes aimed at
// the measured bottleneck (gather latency, ncu: long-scoreboard stalls, 3.4 TB/s of L2->SM traffic):
//   * the neighbour rows (2 KB each) are staged into shared memory by the TMA engine (cp.async.bulk, one copy per
//     edge issued by the producer warp, mbarrier complete_tx), a whole 16-edge tile ahead of the consumers, so no
//     consumer register or LSU slot is spent on keeping loads in flight;
//   * two independent pipelines ("groups" of 8 warps) share ONE copy of the filter operand in a 512-thread CTA
//     (one CTA per SM), and the fp16 hi/lo split is stored unscaled (hi plane, lo plane; the MMA descriptors pick
//     the plane), which shrinks the operand from 72 KB to 48 KB: the freed shared memory holds the gather rings.
#include <cuda_fp16.h>

#include <algorithm>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "tc_common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

namespace etc2 {

constexpr int F = 128, NEB = 16;
constexpr int LBO = 128, SBO = 1024;                   // K = 64 halfs per row: [hi 0..31 | lo 32..63]
constexpr int A_CHUNK = (F / 8) * SBO;                 // 16384
constexpr int A_BYTES = 3 * A_CHUNK;                   // 49152
constexpr int B_BYTES = (2 * NEB / 8) * SBO;           // 4096 (rows 0..15 R_e, 16..31 R'_e)
constexpr int G_ROW = F * 16;                          // 2048 B per gathered row (float4 per channel)
constexpr int GT = 8, NS = 4;                          // gather ring: NS stages of GT edges (one 8-edge half each)
constexpr int G_STAGE = GT * G_ROW;                    // 16384
constexpr int OFF_B = 0, OFF_G = 2 * B_BYTES, OFF_META = OFF_G + NS * G_STAGE, OFF_INVD = OFF_META + 2 * NEB * 16,
              OFF_RED = OFF_INVD + 2 * NEB * 4, OFF_BAR = OFF_RED + 2 * 128 * 4, GROUP_BYTES = OFF_BAR + 256;
constexpr int NTHREADS = 512;
constexpr int SMEM_BYTES = A_BYTES + 2 * GROUP_BYTES + 16 + 128;

void build_filter_image2(const float* Wf, const float* bf, int K, std::vector<unsigned short>& img) {
    img.assign(A_BYTES / 2, 0);
    for (int c = 0; c < 3; c++)
        for (int r = 0; r < F; r++)
            for (int b = 0; b <= K; b++) {
                const float w = b == 0 ? bf[c * F + r] : Wf[(size_t)(c * F + r) * K + (b - 1)];
                const __half hi = __float2half_rn(w);
                const __half lo = __float2half_rn(w - __half2float(hi));
                const __half vals[2] = {hi, lo};
                for (int t = 0; t < 2; t++) {
                    const int k = t * 32 + b;
                    const size_t off = (size_t)c * A_CHUNK + (r / 8) * SBO + (k / 8) * LBO + (r % 8) * 16 + (k % 8) * 2;
                    unsigned short bits;
                    memcpy(&bits, &vals[t], 2);
                    img[off / 2] = bits;
                }
            }
}

__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     tc::smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(tc::smem_u32(bar))
                 : "memory");
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
    int need_sender;     // 0: layer 0 -- phib / vb_out are never used (the embedding is constant), skip their stores
};

__global__ void __launch_bounds__(NTHREADS, 1) k_message_bwd_tc2(BwdParams p) {
    constexpr int TCOLS = 3 * 2 * NEB;            // 96 TMEM columns per accumulator buffer
    // declared aligned (no run-time pointer rounding: that would hide the shared address space from the compiler
    // and turn every LDS / STS into a generic LD / ST)
    extern __shared__ __align__(128) uint8_t smem[];
    uint8_t* sA = smem;
    const int tid = threadIdx.x, grp = tid >> 8, ltid = tid & 255, lwarp = ltid >> 5, lane = tid & 31;
    uint8_t* gbase = smem + A_BYTES + grp * GROUP_BYTES;
    uint8_t* sB = gbase + OFF_B;
    uint8_t* sG = gbase + OFF_G;
    float4* sMeta = (float4*)(gbase + OFF_META);
    float* sInvd = (float*)(gbase + OFF_INVD);
    float* sRed = (float*)(gbase + OFF_RED);
    uint64_t* bars = (uint64_t*)(gbase + OFF_BAR);
    uint64_t* b_full = bars;          // [2] producers -> MMA                    (count 48)
    uint64_t* t_full = bars + 2;      // [2] MMA commit -> consumers             (count 1)
    uint64_t* t_empty = bars + 4;     // [2] consumers (4) + finisher (1) -> producers
    uint64_t* r_full = bars + 6;      // [2] per-edge partial sums written (count 4)
    uint64_t* r_empty = bars + 8;     // [2] finisher done with the reduction buffer (count 1)
    uint64_t* g_full = bars + 10;     // [NS] gathered rows landed (count 1 + 16 KB of complete_tx)
    uint64_t* g_empty = bars + 10 + NS;   // [NS] consumers done with the ring stage (count 4)
    uint32_t* tmem_slot = (uint32_t*)(smem + A_BYTES + 2 * GROUP_BYTES);
    using namespace tc;

    {
        const uint4* src = p.A_img;
        uint4* dst = (uint4*)sA;
        for (int i = tid; i < A_BYTES / 16; i += NTHREADS) dst[i] = src[i];
        uint4* zb = (uint4*)sB;
        for (int i = ltid; i < 2 * B_BYTES / 16; i += 256) zb[i] = make_uint4(0, 0, 0, 0);
    }
    if (ltid == 0) {
        for (int b = 0; b < 2; b++) {
            mbar_init(&b_full[b], 32); mbar_init(&t_full[b], 1); mbar_init(&t_empty[b], 5);
            mbar_init(&r_full[b], 4); mbar_init(&r_empty[b], 1);
        }
        for (int b = 0; b < NS; b++) { mbar_init(&g_full[b], 1); mbar_init(&g_empty[b], 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid >> 5 == 15) tmem_alloc(tmem_slot, 512);
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot + grp * 256;
    const long long n_units = (p.N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    const long long u0 = (long long)blockIdx.x * 2 + grp, ustride = (long long)gridDim.x * 2;
    if (lwarp < 4) reg_inc<168>(); else reg_dec<88>();

    if (lwarp < 4) {
        // ===================== consumers: one channel per thread =====================
        const int f = ltid;
        const uint32_t lane_base = tmem_base + ((uint32_t)(lwarp * 32) << 16);
        uint32_t it = 0, hc = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            long long j = a0;
            int row_end = p.row_ptr[a0 + 1];
            float phS, phVS, phVV, vj0, vj1, vj2, pbS, pbVS, Y0, Y1, Y2;
            auto start_row = [&]() {
                row_end = p.row_ptr[j + 1];
                phS = p.phi[j * 3 * F + f]; phVS = p.phi[j * 3 * F + F + f]; phVV = p.phi[j * 3 * F + 2 * F + f];
                vj0 = p.v_in[j * 3 * F + f]; vj1 = p.v_in[j * 3 * F + F + f]; vj2 = p.v_in[j * 3 * F + 2 * F + f];
                pbS = pbVS = Y0 = Y1 = Y2 = 0.f;
            };
            auto finish_row = [&]() {
                if (!p.need_sender) return;
                p.phib[j * 3 * F + f] = pbS;
                p.phib[j * 3 * F + F + f] = pbVS;
                p.phib[j * 3 * F + 2 * F + f] = vj0 * Y0 + vj1 * Y1 + vj2 * Y2;
                p.vb_out[j * 3 * F + f] = p.v1b[j * 3 * F + f] + phVV * Y0;
                p.vb_out[j * 3 * F + F + f] = p.v1b[j * 3 * F + F + f] + phVV * Y1;
                p.vb_out[j * 3 * F + 2 * F + f] = p.v1b[j * 3 * F + 2 * F + f] + phVV * Y2;
            };
            start_row();
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                const uint32_t ph = (it >> 1) & 1;
                mbar_wait(&t_full[buf], ph);
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
                    const int gs = hc & (NS - 1);
                    mbar_wait(&g_full[gs], (hc / NS) & 1);
                    const uint8_t* grow = sG + gs * G_STAGE + f * 16;
                    tmem_wait_ld();
                    float part[32];
#pragma unroll
                    for (int i = 0; i < 8; i++) {
                        const int E = e_begin + t * NEB + h * 8 + i;
                        float db = 0.f, ub0 = 0.f, ub1 = 0.f, ub2 = 0.f;
                        if (E < e_end) {
                            while (E >= row_end) { finish_row(); j++; start_row(); }
                            const float4 m = meta[h * 8 + i];
                            const float4 gb = *(const float4*)(grow + i * G_ROW);
                            const float wS = __uint_as_float(w[0][i]), wVS = __uint_as_float(w[1][i]), wVV = __uint_as_float(w[2][i]);
                            const float dS = __uint_as_float(dw[0][i]), dVS = __uint_as_float(dw[1][i]), dVV = __uint_as_float(dw[2][i]);
                            const float sb = gb.x, vb0 = gb.y, vb1 = gb.z, vb2 = gb.w;
                            const float X = vb0 * m.x + vb1 * m.y + vb2 * m.z;
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
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&g_empty[gs]);      // ring stage may be refilled
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
                    float* red = sRed + (hc & 1) * 128;
                    mbar_wait(&r_empty[hc & 1], ((hc >> 1) & 1) ^ 1);
                    red[lwarp * 32 + lane] = part[0];
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
    } else if (lwarp == 4) {
        // ===================== producer: filter operands R_e, R'_e (hi / lo fp16 planes), edge meta =====================
        const int e = lane & 15, hh = lane >> 4;        // thread = (edge, half of the 24 basis slots: 0..11 / 12..23)
        uint32_t it = 0;
        const float a1c = 3.14159265358979323846f * p.inv_rc;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            for (int t = 0; t < ntiles; t++, it++) {
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
                if (hh == 0) { sn_ = s1; cn_ = c1; } else sincospif(12.0f * x, &sn_, &cn_);
                __half hi[2][12], lo[2][12];
#pragma unroll
                for (int i = 0; i < 12; i++) {
                    const int b = hh * 12 + i;
                    float v, dv;
                    if (b == 0) { v = fc; dv = dfc; }
                    else {
                        const float rho = sn_ * inv_d;
                        const float drho = ((float)b * a1c * cn_ - rho) * inv_d;
                        v = b <= p.K ? fc * rho : 0.0f;
                        dv = b <= p.K ? dfc * rho + fc * drho : 0.0f;
                        const float tt = sn_ * c1 + cn_ * s1;
                        cn_ = cn_ * c1 - sn_ * s1;
                        sn_ = tt;
                    }
                    hi[0][i] = __float2half_rn(v);  lo[0][i] = __float2half_rn(v - __half2float(hi[0][i]));
                    hi[1][i] = __float2half_rn(dv); lo[1][i] = __float2half_rn(dv - __half2float(hi[1][i]));
                }
                // the stage (TMEM buffer, B operand, meta) is free once tile it-2 is fully consumed
                mbar_wait(&t_empty[buf], ((it >> 1) & 1) ^ 1);
#pragma unroll
                for (int z = 0; z < 2; z++) {
                    const int row = z * NEB + e;
                    uint8_t* bb = sB + buf * B_BYTES + (row >> 3) * SBO + (row & 7) * 16;   // + kc * LBO, + 4 * LBO for lo
                    if (hh == 0) {   // slots 0..7 -> chunk 0, slots 8..11 -> first half of chunk 1
                        *(uint4*)(bb) = *(uint4*)&hi[z][0];
                        *(uint4*)(bb + 4 * LBO) = *(uint4*)&lo[z][0];
                        *(uint2*)(bb + LBO) = *(uint2*)&hi[z][8];
                        *(uint2*)(bb + 5 * LBO) = *(uint2*)&lo[z][8];
                    } else {         // slots 12..15 -> second half of chunk 1, slots 16..23 -> chunk 2
                        *(uint2*)(bb + LBO + 8) = *(uint2*)&hi[z][0];
                        *(uint2*)(bb + 5 * LBO + 8) = *(uint2*)&lo[z][0];
                        *(uint4*)(bb + 2 * LBO) = *(uint4*)&hi[z][4];
                        *(uint4*)(bb + 6 * LBO) = *(uint4*)&lo[z][4];
                    }
                }
                if (hh == 0) {
                    sMeta[buf * NEB + e] = make_float4(-r.x * inv_d, -r.y * inv_d, -r.z * inv_d, r.w);   // u_e of edge (i <- j)
                    sInvd[buf * NEB + e] = inv_d;
                }
                fence_async_smem();
                mbar_arrive(&b_full[buf]);
            }
        }
    } else if (lwarp == 5) {
        // ===================== gather warp: TMA bulk copies of the neighbour rows into the ring =====================
        // Lane l serves edge (l & 7) of ring stage hc = 4 r + (l >> 3) in round r; every lane walks the same
        // (unit, tile, half) sequence as the consumers, four stages at a time, and loads its neighbour index one
        // round ahead so the index-load latency is hidden behind the ring back-pressure.
        const int le = lane & 7, lg = lane >> 3;
        long long u = u0;
        int e_begin = 0, e_end = 0, ntiles = 0, t = 0, h = 0;
        bool done = false;
        auto load_unit = [&]() {
            for (;;) {
                if (u >= n_units) { done = true; return; }
                const long long a0 = u * p.atoms_per_unit;
                const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
                e_begin = p.row_ptr[a0]; e_end = p.row_ptr[a1];
                ntiles = (e_end - e_begin + NEB - 1) / NEB;
                t = 0; h = 0;
                if (ntiles > 0) return;
                u += ustride;
            }
        };
        auto advance = [&]() {      // one stage forward
            if (done) return;
            if (++h == 2) { h = 0; if (++t == ntiles) { u += ustride; load_unit(); } }
        };
        auto fetch = [&]() -> int {   // neighbour index of this lane's edge in its current stage
            if (done) return -1;
            const int E = e_begin + t * NEB + h * GT + le;
            int ix = E < e_end ? __float_as_int(__ldg(p.ej + E).w) : 0;
            return ix < 0 ? ~ix : ix;                    // padding slot: gather the atom's own row (weight is zero)
        };
        load_unit();
        for (int k = 0; k < lg; k++) advance();
        int idx = fetch();
        uint32_t hc = 0;
        while (__any_sync(0xffffffffu, idx >= 0)) {
            for (int k = 0; k < 4; k++) advance();
            const int idx_next = fetch();
#pragma unroll
            for (int q = 0; q < 4; q++, hc++) {
                const int active = __shfl_sync(0xffffffffu, idx, q * 8) >= 0;   // does stage hc exist? (uniform)
                if (!active) break;
                const int gs = hc & (NS - 1);
                mbar_wait(&g_empty[gs], ((hc / NS) & 1) ^ 1);
                if (lane == q * 8) mbar_expect_tx(&g_full[gs], G_STAGE);
                __syncwarp();
                if (lg == q) bulk_g2s(sG + gs * G_STAGE + le * G_ROW, p.Gb + (size_t)idx * F, G_ROW, &g_full[gs]);
            }
            idx = idx_next;
        }
    } else if (lwarp == 6) {
        // ===================== finisher: cross-warp sums, g_e, G accumulation =====================
        uint32_t it = 0, hc = 0;
        for (long long u = u0; u < n_units; u += ustride) {
            const long long a0 = u * p.atoms_per_unit;
            const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
            const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
            const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
            for (int t = 0; t < ntiles; t++, it++) {
                const int buf = it & 1;
                for (int h = 0; h < 2; h++, hc++) {
                    const int E = e_begin + t * NEB + h * 8 + lane;
                    float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
                    const bool act = lane < 8 && E < e_end;
                    if (act && !p.first) o = p.G[E];                 // issue the read-modify-write load early
                    mbar_wait(&r_full[hc & 1], (hc >> 1) & 1);
                    const float* red = sRed + (hc & 1) * 128;
                    if (act) {
                        float db = 0.f, ub0 = 0.f, ub1 = 0.f, ub2 = 0.f;
#pragma unroll
                        for (int wq = 0; wq < 4; wq++) {
                            db += red[wq * 32 + 4 * lane]; ub0 += red[wq * 32 + 4 * lane + 1];
                            ub1 += red[wq * 32 + 4 * lane + 2]; ub2 += red[wq * 32 + 4 * lane + 3];
                        }
                        const float4 mm = sMeta[buf * NEB + h * 8 + lane];
                        const float inv_d = sInvd[buf * NEB + h * 8 + lane];
                        const float uu = ub0 * mm.x + ub1 * mm.y + ub2 * mm.z;
                        p.G[E] = make_float4(o.x + db * mm.x + (ub0 - uu * mm.x) * inv_d, o.y + db * mm.y + (ub1 - uu * mm.y) * inv_d,
                                             o.z + db * mm.z + (ub2 - uu * mm.z) * inv_d, 0.f);
                    }
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(&r_empty[hc & 1]);
                        if (h == 1) mbar_arrive(&t_empty[buf]);
                    }
                }
            }
        }
    } else {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            const uint32_t idesc = (1u << 4) | ((uint32_t)((2 * NEB) >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
            const uint32_t a_base = smem_u32(sA), b_base = smem_u32(sB);
            // (A k-step, B k-step) pairs; k-steps 0,1 = hi plane, 2,3 = lo plane; small terms first, main term last
            const int sa[6] = {2, 3, 0, 1, 0, 1}, sb[6] = {0, 1, 2, 3, 0, 1};
            uint32_t it = 0;
            for (long long u = u0; u < n_units; u += ustride) {
                const long long a0 = u * p.atoms_per_unit;
                const long long a1 = min(p.N, a0 + (long long)p.atoms_per_unit);
                const int e_begin = p.row_ptr[a0], e_end = p.row_ptr[a1];
                const int ntiles = (e_end - e_begin + NEB - 1) / NEB;
                for (int t = 0; t < ntiles; t++, it++) {
                    const int buf = it & 1;
                    mbar_wait(&b_full[buf], (it >> 1) & 1);
                    tc_fence_after();
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        const uint32_t d = tmem_base + buf * TCOLS + c * 2 * NEB;
#pragma unroll
                        for (int o = 0; o < 6; o++) {
                            const uint64_t ad = make_desc_nosw(a_base + c * A_CHUNK + sa[o] * 2 * LBO, LBO, SBO);
                            const uint64_t bd = make_desc_nosw(b_base + buf * B_BYTES + sb[o] * 2 * LBO, LBO, SBO);
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
    if (tid >> 5 == 15) tmem_dealloc(*tmem_slot, 512);
}

}  // namespace etc2

void edge_build_filter_image2(const float* Wf, const float* bf, int K, std::vector<unsigned short>& img) {
    etc2::build_filter_image2(Wf, bf, K, img);
}

bool message_bwd_tc2(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* Gb,
                     const float* phi, const float* v_in, const float* v1b, const void* A_img2, float* phib, float* vb_out,
                     float4* G, bool first, bool need_sender) {
    using namespace etc2;
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
        if (cudaFuncSetAttribute(k_message_bwd_tc2, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES) != cudaSuccess) return false;
        attr = true;
    }
    BwdParams p{N, row_ptr, ej, (const float4*)Gb, phi, v_in, v1b, (const uint4*)A_img2, phib, vb_out, G, 1.0f / rc, K, 16,
                first ? 1 : 0, need_sender ? 1 : 0};
    const long long n_units = (N + p.atoms_per_unit - 1) / p.atoms_per_unit;
    const int grid = (int)std::min<long long>((n_units + 1) / 2, (long long)n_sm);
    k_message_bwd_tc2<<<grid, NTHREADS, SMEM_BYTES, L.stream>>>(p);
    KLAUNCH(L);
    return true;
}

}  // namespace painn
