// edge_l0.cu -- layer-0 adjoint message pass with the channel contraction hoisted out of the edge loop.
//
// At layer 0 the sender features are the embedding: s^0_j = Emb[z_j], v^0_j = 0 (reading B6), so the sender rows
// (phi^s, phi^vs) of an edge depend on the SPECIES of j only.  The geometry gradient of edge (i <- j), written out from
// the adjoint of the PaiNN message (PAPER.md:58 semi-local message passing),
//
//     g_e = u [ sum_c db_c - (1/d) sum_c w^vs_c phi^vs_c (vb'_ic . u) ] + (1/d) sum_c w^vs_c phi^vs_c vb'_ic ,
//     db_c = phi^s_c sb'_ic dw^s_c/dd + phi^vs_c (vb'_ic . u) dw^vs_c/dd ,     w_c(d) = sum_k Wf[c][k] R_k(d) ,
//
// (R_0 = fc, R_k = fc rho_k, bias in slot 0) is linear in the filter, and everything that carries a channel index besides
// the filter weights belongs to the RECEIVER i and the species z of the sender.  Contracting the channels first,
//
//     B_iz[k] = sum_c Wf^vs[c][k] phi^vs_z[c] vb'_ic   (3-vector)        C_iz[k] = sum_c Wf^s[c][k] phi^s_z[c] sb'_ic ,
//
// is two plain GEMMs per step ([3N x F] and [N x F] against [n_species (K+1) x F] matrices built at create), after which
// an edge costs O(K) instead of O(F K):
//
//     P = sum_k R_k B_iz[k],  P' = sum_k R'_k B_iz[k],  c' = sum_k R'_k C_iz[k],
//     g_e = u [ c' + u . P' - (u . P) / d ] + P / d .
//
// One thread per edge, one warp per receiver row; the row's (B, C) vectors are staged in shared memory as float4
// (B_x, B_y, B_z, C) per (species, k).  G is indexed by the slot of the SENDER's row (force_final: F_a = sum_x G[rev x] -
// G[x]), so the result is scattered through the reverse-edge index, as in k_msg_bwd0.
#include "common.cuh"

namespace painn {
namespace el0 {

constexpr int WARPS = 8;
constexpr int KMAX1 = 24;          // K + 1 <= 24 (same limit as the tensor-core edge kernels)

#define KLAUNCH(L) (++*(L).counter)

__global__ void __launch_bounds__(WARPS * 32) k_l0_bwd(long long N, const int* __restrict__ row_ptr, const float4* __restrict__ ej,
                                                      const int* __restrict__ types, const int* __restrict__ rev,
                                                      const float* __restrict__ Bv, const float* __restrict__ Cs, int NP,
                                                      int n_used, int K, float inv_rc, float4* __restrict__ G, int first) {
    extern __shared__ float4 sm[];                       // [WARPS][n_used]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4* bc = sm + warp * n_used;
    const float a1c = 3.14159265358979323846f * inv_rc;
    const int KP1 = K + 1;
    for (long long i = (long long)blockIdx.x * WARPS + warp; i < N; i += (long long)gridDim.x * WARPS) {
        const int e0 = __ldg(row_ptr + i), e1 = __ldg(row_ptr + i + 1);
        __syncwarp();
        for (int n = lane; n < n_used; n += 32)
            bc[n] = make_float4(__ldg(Bv + (3 * i) * NP + n), __ldg(Bv + (3 * i + 1) * NP + n), __ldg(Bv + (3 * i + 2) * NP + n),
                                __ldg(Cs + i * NP + n));
        __syncwarp();
        for (int E = e0 + lane; E < e1; E += 32) {
            const float4 r = __ldg(ej + E);
            const int jb = __float_as_int(r.w);
            const int tgt = __ldg(rev + E);
            float gx = 0.f, gy = 0.f, gz = 0.f;
            if (jb >= 0) {                               // padding slots carry ~own row: zero weight
                const float d2 = r.x * r.x + r.y * r.y + r.z * r.z;
                const float inv_d = rsqrtf(d2);
                const float x = d2 * inv_d * inv_rc;
                float s1, c1;
                sincospif(x, &s1, &c1);
                const float fc = 0.5f * (1.0f + c1), dfc = -0.5f * a1c * s1;
                const float ux = r.x * inv_d, uy = r.y * inv_d, uz = r.z * inv_d;
                const float4* v = bc + __ldg(types + jb) * KP1;
                // slot 0: bias (R_0 = fc)
                float4 q = v[0];
                float Px = fc * q.x, Py = fc * q.y, Pz = fc * q.z;
                float Dx = dfc * q.x, Dy = dfc * q.y, Dz = dfc * q.z, cd = dfc * q.w;
                float sn = s1, cn = c1;
                for (int b = 1; b <= K; b++) {
                    if ((b & 7) == 0) sincospif((float)b * x, &sn, &cn);      // fresh start every 8 slots (as the producers do)
                    const float rho = sn * inv_d;
                    const float drho = ((float)b * a1c * cn - rho) * inv_d;
                    const float R = fc * rho, dR = fmaf(dfc, rho, fc * drho);
                    q = v[b];
                    Px = fmaf(R, q.x, Px); Py = fmaf(R, q.y, Py); Pz = fmaf(R, q.z, Pz);
                    Dx = fmaf(dR, q.x, Dx); Dy = fmaf(dR, q.y, Dy); Dz = fmaf(dR, q.z, Dz);
                    cd = fmaf(dR, q.w, cd);
                    const float tt = fmaf(sn, c1, cn * s1);
                    cn = fmaf(cn, c1, -sn * s1);
                    sn = tt;
                }
                const float uP = fmaf(ux, Px, fmaf(uy, Py, uz * Pz));
                const float uD = fmaf(ux, Dx, fmaf(uy, Dy, uz * Dz));
                const float a = cd + uD - uP * inv_d;
                gx = fmaf(a, ux, Px * inv_d);
                gy = fmaf(a, uy, Py * inv_d);
                gz = fmaf(a, uz, Pz * inv_d);
            }
            float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
            if (!first) o = G[tgt];
            G[tgt] = make_float4(o.x + gx, o.y + gy, o.z + gz, 0.f);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Forward counterpart.  With s^0_j = Emb[z_j] and v^0 = 0 the layer-0 message is
//     ds_i[c] = sum_z phi^s_z[c]  sum_k Wf^s[c][k]  Rs_iz[k] ,      Rs_iz[k] = sum_{j in N(i), z_j = z} R_k(d_ij)
//     dv_i[c] = sum_z phi^vs_z[c] sum_k Wf^vs[c][k] Q_iz[k]  ,      Q_iz[k]  = sum_{j in N(i), z_j = z} R_k(d_ij) u_ij
// i.e. an O(K) accumulation per edge into per-(receiver, species) radial sums, then two GEMMs against [F x n_species
// (K + 1)] matrices.  One warp per receiver, lane = radial slot k (each lane owns its column of the accumulators: no
// atomics, fixed summation order, bit-reproducible); the edges of the row are prepared 32 at a time by lane = edge.
// Writes As [N][NP] = Rs, Av [3N][NP] = Q (row 3 i + component) and copies s_i into the s' half of sn (ldsn floats per
// row), to which the first GEMM accumulates.
// ---------------------------------------------------------------------------------------------------------------
constexpr float PI_F = 3.14159265358979323846f;
constexpr int RLD = 25;            // row stride of the per-edge radial values (odd: conflict-free both ways)
__global__ void __launch_bounds__(WARPS * 32) k_l0_fwd(long long N, const int* __restrict__ row_ptr, const float4* __restrict__ ej,
                                                      const int* __restrict__ types, const float* __restrict__ s_in, int F,
                                                      float* __restrict__ sn, int ldsn, float* __restrict__ As,
                                                      float* __restrict__ Av, int NP, int n_used, int K, float inv_rc,
                                                      const float2* __restrict__ xph) {
    extern __shared__ float4 sm[];       // [WARPS][n_used] accumulators | [WARPS][32] (u, species offset) | [WARPS][32][RLD] R_k
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4* acc = sm + warp * n_used;
    float4* rec = sm + WARPS * n_used + warp * 32;
    float* Rb = (float*)(sm + WARPS * (n_used + 32)) + warp * 32 * RLD;
    const int KP1 = K + 1;
    for (long long i = (long long)blockIdx.x * WARPS + warp; i < N; i += (long long)gridDim.x * WARPS) {
        const int e0 = __ldg(row_ptr + i), e1 = __ldg(row_ptr + i + 1);
        for (int n = lane; n < n_used; n += 32) acc[n] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int c = lane * 4; c < F; c += 128) *(float4*)(sn + i * ldsn + c) = __ldg((const float4*)(s_in + i * F + c));
        for (int eb = e0; eb < e1; eb += 32) {
            // lane = edge: geometry and all K + 1 radial values of up to 32 edges (one sincospi + rotation recurrence per
            // 8 slots, as the producers of the tensor-core kernels do)
            const int E = eb + lane;
            float4 r = make_float4(1.f, 0.f, 0.f, __int_as_float(-1));
            if (E < e1) r = __ldg(ej + E);
            const int jb = __float_as_int(r.w);
            const float d2 = r.x * r.x + r.y * r.y + r.z * r.z;
            const float inv_d = 1.0f / sqrtf(d2);                 // IEEE: rsqrtf's 2 ulp would go straight into u and rho
            float x = d2 * inv_d * inv_rc, xl = 0.f;
            if (xph != nullptr && E < e1) { const float2 xp = __ldg(xph + E); x = xp.x; xl = xp.y * PI_F; }   // compensated phase (nbr.cu)
            float s1, c1;
            sincospif(x, &s1, &c1);
            { const float t = fmaf(xl, c1, s1); c1 = fmaf(-xl, s1, c1); s1 = t; }
            const float fc = jb >= 0 ? 0.5f * (1.0f + c1) : 0.0f;                  // padding slots: zero weight
            const int z = jb >= 0 ? __ldg(types + jb) : 0;
            __syncwarp();
            rec[lane] = make_float4(r.x * inv_d, r.y * inv_d, r.z * inv_d, __int_as_float(z * KP1));
            float* rb = Rb + lane * RLD;
            rb[0] = fc;
            const float amp = fc * inv_d;
            float sn_ = s1, cn_ = c1;
            for (int b = 1; b <= K; b++) {
                if ((b & 7) == 0) {
                    sincospif((float)b * x, &sn_, &cn_);
                    const float t = fmaf((float)b * xl, cn_, sn_);
                    cn_ = fmaf(-(float)b * xl, sn_, cn_);
                    sn_ = t;
                }
                rb[b] = amp * sn_;
                const float tt = fmaf(sn_, c1, cn_ * s1);
                cn_ = fmaf(cn_, c1, -sn_ * s1);
                sn_ = tt;
            }
            __syncwarp();
            // lane = radial slot: walk the edges in order (each lane owns its column of the accumulators)
            const int ne = min(32, e1 - eb);
            if (lane < KP1) {
                for (int e = 0; e < ne; e++) {
                    const float4 u = rec[e];
                    const float R = Rb[e * RLD + lane];
                    float4* q = acc + __float_as_int(u.w) + lane;
                    float4 v = *q;
                    v.x += R; v.y = fmaf(R, u.x, v.y); v.z = fmaf(R, u.y, v.z); v.w = fmaf(R, u.z, v.w);
                    *q = v;
                }
            }
        }
        __syncwarp();
        for (int n = lane; n < NP; n += 32) {
            const float4 v = n < n_used ? acc[n] : make_float4(0.f, 0.f, 0.f, 0.f);
            As[i * NP + n] = v.x;
            Av[(3 * i) * NP + n] = v.y; Av[(3 * i + 1) * NP + n] = v.z; Av[(3 * i + 2) * NP + n] = v.w;
        }
        __syncwarp();
    }
}

}  // namespace el0

bool message_fwd0_collapsed_accum(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej,
                                  const int* types_s, int n_species, const float* s_in, int F, float* sn, int ldsn, float* As,
                                  float* Av, int NP, const float2* xph) {
    using namespace el0;
    if (N == 0) return true;
    const int n_used = n_species * (K + 1);
    if (K + 1 > KMAX1 || n_used > NP || (F % 4) || (ldsn % 4)) return false;
    const size_t smem = (size_t)WARPS * (n_used + 32) * sizeof(float4) + (size_t)WARPS * 32 * RLD * sizeof(float);
    if (smem > 48 * 1024) return false;
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    const long long want = (N + WARPS - 1) / WARPS;
    const int grid = (int)(want < (long long)n_sm * 8 ? want : (long long)n_sm * 8);
    k_l0_fwd<<<grid, WARPS * 32, smem, L.stream>>>(N, row_ptr, ej, types_s, s_in, F, sn, ldsn, As, Av, NP, n_used, K, 1.0f / rc, xph);
    KLAUNCH(L);
    return true;
}

// Bv: [3N][NP] (row 3 i + component), Cs: [N][NP]; columns n = species (K + 1) + k, n < n_species (K + 1) <= NP
bool message_bwd0_collapsed(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej,
                            const int* types_s, int n_species, const int* rev, const float* Bv, const float* Cs, int NP,
                            float4* G, bool first) {
    using namespace el0;
    if (N == 0) return true;
    const int n_used = n_species * (K + 1);
    if (K + 1 > KMAX1 || n_used > NP) return false;
    const size_t smem = (size_t)WARPS * n_used * sizeof(float4);
    if (smem > 48 * 1024) return false;
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    const long long want = (N + WARPS - 1) / WARPS;
    const int grid = (int)(want < (long long)n_sm * 8 ? want : (long long)n_sm * 8);
    k_l0_bwd<<<grid, WARPS * 32, smem, L.stream>>>(N, row_ptr, ej, types_s, rev, Bv, Cs, NP, n_used, K, 1.0f / rc, G, first ? 1 : 0);
    KLAUNCH(L);
    return true;
}

}  // namespace painn
