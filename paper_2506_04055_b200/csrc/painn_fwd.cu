// painn_fwd.cu -- forward PaiNN kernels (north_star items 2-3).
//
// Equations: DESIGN.md section 2 "Forward" (the reading of PaiNN this build fixes; Eq. 6-7 give
// only the generic message / update frame, PAPER.md:212, 246 name the architecture).
//   rho_n(d) = sin(n pi d / rc) / d,  fc(d) = (1 + cos(pi d / rc)) / 2,  w_e = fc (Wf rho + bf) = [s | vs | vv]
//   s'_i = s_i + sum_e w^s o phi^s_j ;  v'_i[c] = v_i[c] + sum_e (w^vs o phi^vs_j u_e[c] + w^vv o phi^vv_j o v_j[c])
// Node layout: s [N][F], v [N][3][F], phi [N][3F], pq [N][3][2F] (p | q), sn [N][2F] (s' | n), a [N][3F].
// Thread mapping of the edge kernels: one thread per (receiver atom, channel f); a row of the CSR is walked
// sequentially, so the segment sum needs no atomics and consecutive threads gather consecutive channels
// (coalesced 4F-byte row reads).
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include "common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

__device__ __forceinline__ float sigmoidf_(float x) { return 1.0f / (1.0f + __expf(-x)); }
__device__ __forceinline__ float siluf_(float x) { return x * sigmoidf_(x); }
__device__ __forceinline__ float dsiluf_(float x) { float s = sigmoidf_(x); return s * (1.0f + x * (1.0f - s)); }

// ------------------------------------------------------------------------------------------------ a5
__global__ void k_embed(long long N, int F, const int* __restrict__ types_s, const float* __restrict__ Emb,
                        float* __restrict__ s0, float* __restrict__ v0) {
    const int F4 = F >> 2;                       // four channels per thread
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F4) return;
    long long a = idx / F4;
    int f = (int)(idx - a * F4) * 4;
    *(float4*)(s0 + a * F + f) = *(const float4*)(Emb + (size_t)types_s[a] * F + f);
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    *(float4*)(v0 + a * 3 * F + f) = z; *(float4*)(v0 + a * 3 * F + F + f) = z; *(float4*)(v0 + a * 3 * F + 2 * F + f) = z;
}
void embed(const Launch& L, long long N, int F, const int* types_s, const float* Emb, float* s0, float* v0) {
    if (N == 0) return;
    k_embed<<<(unsigned)((N * (F / 4) + 255) / 256), 256, 0, L.stream>>>(N, F, types_s, Emb, s0, v0);
    KLAUNCH(L);
}

__global__ void k_silu(long long n, const float* __restrict__ x, float* __restrict__ y) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) y[i] = siluf_(x[i]);
}
void silu_fwd(const Launch& L, long long n, const float* x, float* y) {
    if (n == 0) return;
    k_silu<<<(unsigned)((n + 255) / 256), 256, 0, L.stream>>>(n, x, y);
    KLAUNCH(L);
}
__global__ void k_mul_dsilu(long long n, const float* __restrict__ pre, float* __restrict__ g) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) g[i] *= dsiluf_(pre[i]);
}
void mul_dsilu(const Launch& L, long long n, const float* pre, float* g) {
    if (n == 0) return;
    k_mul_dsilu<<<(unsigned)((n + 255) / 256), 256, 0, L.stream>>>(n, pre, g);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ a4 + a7
template <int KMAX>
__global__ void __launch_bounds__(128) k_message_fwd(long long N, int F, int K, float inv_rc,
                                                     const int* __restrict__ row_ptr,
                                                     const float4* __restrict__ ej, const float* __restrict__ s,
                                                     const float* __restrict__ v, const float* __restrict__ phi,
                                                     const float* __restrict__ Wf, const float* __restrict__ bf,
                                                     float* __restrict__ sn, float* __restrict__ v1) {
    const long long a = blockIdx.x * (long long)blockDim.y + threadIdx.y;
    const int f = threadIdx.x;
    if (a >= N) return;
    float wS[KMAX], wVS[KMAX], wVV[KMAX];
#pragma unroll
    for (int n = 0; n < KMAX; n++) {
        wS[n] = n < K ? Wf[(size_t)(f)*K + n] : 0.0f;
        wVS[n] = n < K ? Wf[(size_t)(F + f) * K + n] : 0.0f;
        wVV[n] = n < K ? Wf[(size_t)(2 * F + f) * K + n] : 0.0f;
    }
    const float bS = bf[f], bVS = bf[F + f], bVV = bf[2 * F + f];
    const size_t F3 = 3 * (size_t)F;
    float accS = s[a * F + f];
    float accV0 = v[a * F3 + f], accV1 = v[a * F3 + F + f], accV2 = v[a * F3 + 2 * F + f];
    const int e0 = row_ptr[a], e1 = row_ptr[a + 1];
    for (int e = e0; e < e1; e++) {
        const float4 r = ej[e];
        const int j = __float_as_int(r.w);
        if (j < 0) continue;                         // padding slot
        const float d2 = r.x * r.x + r.y * r.y + r.z * r.z;
        const float inv_d = rsqrtf(d2);
        const float d = d2 * inv_d;
        float s1, c1;
        sincospif(d * inv_rc, &s1, &c1);
        float sn_ = s1, cn_ = c1;
        const float fc = 0.5f * (1.0f + c1);
        // w = fc (Wf rho + bf) = Wf (fc rho) + bf fc : the cutoff is folded into the GEMM operand
        float linS = fmaf(bS, fc, 0.f), linVS = fmaf(bVS, fc, 0.f), linVV = fmaf(bVV, fc, 0.f);
#pragma unroll
        for (int n = 0; n < KMAX; n++) {
            const float rho = fc * sn_ * inv_d;
            linS = fmaf(wS[n], rho, linS);
            linVS = fmaf(wVS[n], rho, linVS);
            linVV = fmaf(wVV[n], rho, linVV);
            const float t = sn_ * c1 + cn_ * s1;
            cn_ = cn_ * c1 - sn_ * s1;
            sn_ = t;
        }
        const float* pj = phi + (size_t)j * F3;
        const float* vj = v + (size_t)j * F3;
        const float pvv = pj[2 * F + f];
        const float xs = linS * pj[f];
        const float xvs = linVS * pj[F + f];
        accS += xs;
        accV0 += xvs * (r.x * inv_d) + linVV * pvv * vj[f];
        accV1 += xvs * (r.y * inv_d) + linVV * pvv * vj[F + f];
        accV2 += xvs * (r.z * inv_d) + linVV * pvv * vj[2 * F + f];
    }
    sn[a * 2 * F + f] = accS;
    v1[a * F3 + f] = accV0; v1[a * F3 + F + f] = accV1; v1[a * F3 + 2 * F + f] = accV2;
}

void message_fwd(const Launch& L, long long N, int F, int K, float rc, const int* row_ptr, const float4* ej,
                 const float* s, const float* v, const float* phi, const float* Wf, const float* bf, float* sn,
                 float* v1) {
    if (N == 0) return;
    dim3 block(F, 128 / F);
    unsigned grid = (unsigned)((N + block.y - 1) / block.y);
#define MF(KM) k_message_fwd<KM><<<grid, block, 0, L.stream>>>(N, F, K, 1.0f / rc, row_ptr, ej, s, v, phi, Wf, bf, sn, v1)
    if (K <= 16) MF(16); else if (K <= 20) MF(20); else MF(32);
#undef MF
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ a8
__global__ void k_update_mid(long long N, int F, float eps, const float* __restrict__ pq, float* __restrict__ sn) {
    const int F4 = F >> 2;                       // four channels per thread
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F4) return;
    long long a = idx / F4;
    int f = (int)(idx - a * F4) * 4;
    const float* q = pq + a * 6 * F + F + f;
    const float4 q0 = *(const float4*)q, q1 = *(const float4*)(q + 2 * F), q2 = *(const float4*)(q + 4 * F);
    *(float4*)(sn + a * 2 * F + F + f) = make_float4(sqrtf(q0.x * q0.x + q1.x * q1.x + q2.x * q2.x + eps),
                                                     sqrtf(q0.y * q0.y + q1.y * q1.y + q2.y * q2.y + eps),
                                                     sqrtf(q0.z * q0.z + q1.z * q1.z + q2.z * q2.z + eps),
                                                     sqrtf(q0.w * q0.w + q1.w * q1.w + q2.w * q2.w + eps));
}
void update_mid(const Launch& L, long long N, int F, float eps, const float* pq, float* sn) {
    if (N == 0) return;
    k_update_mid<<<(unsigned)((N * (F / 4) + 255) / 256), 256, 0, L.stream>>>(N, F, eps, pq, sn);
    KLAUNCH(L);
}
// v_i[c] <- v'_i[c] + a^vv o p[c] ;  s_i <- s'_i + a^sv o (sum_c p[c] o q[c]) + a^ss      (a = [vv | sv | ss])
__global__ void k_update_out(long long N, int F, const float* __restrict__ sn, const float* __restrict__ v1,
                             const float* __restrict__ pq, const float* __restrict__ a_,
                             float* __restrict__ s_out, float* __restrict__ v_out) {
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F) return;
    long long a = idx / F;
    int f = (int)(idx - a * F);
    const float* p = pq + a * 6 * F + f;
    const float* q = p + F;
    const float avv = a_[a * 3 * F + f], asv = a_[a * 3 * F + F + f], ass = a_[a * 3 * F + 2 * F + f];
    float D = 0.0f;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        float pc = p[c * 2 * F];
        D += pc * q[c * 2 * F];
        v_out[a * 3 * F + c * F + f] = v1[a * 3 * F + c * F + f] + avv * pc;
    }
    s_out[idx] = sn[a * 2 * F + f] + asv * D + ass;
}
void update_out(const Launch& L, long long N, int F, const float* sn, const float* v1, const float* pq,
                const float* a, float* s_out, float* v_out) {
    if (N == 0) return;
    k_update_out<<<(unsigned)((N * F + 255) / 256), 256, 0, L.stream>>>(N, F, sn, v1, pq, a, s_out, v_out);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ a9 (+ a10 seed)
// E_i = wr2 . SiLU(rpre_i) + br2 ; rb_i = [i local] wr2 o SiLU'(rpre_i) ; per-block fp64 partial sums of local E_i
__global__ void __launch_bounds__(256) k_readout(long long N, int R, const float* __restrict__ rpre,
                                                 const float* __restrict__ wr2, const float* __restrict__ br2,
                                                 const float* __restrict__ local_mask, float* __restrict__ rb,
                                                 float* __restrict__ e_atom, double* __restrict__ e_partial) {
    __shared__ double red[256];
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    double mine = 0.0;
    if (a < N) {
        const float m = local_mask[a];
        float e = br2[0];
        for (int r = 0; r < R; r++) {
            float x = rpre[a * R + r];
            e += wr2[r] * siluf_(x);
            rb[a * R + r] = m * wr2[r] * dsiluf_(x);
        }
        e_atom[a] = e;
        mine = m != 0.0f ? (double)e : 0.0;
    }
    red[threadIdx.x] = mine;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) e_partial[blockIdx.x] = red[0];
}
// R in {16, 32, 64}: R / 4 lanes per atom, 16-byte accesses (the thread-per-atom form above walks 32 rows per warp
// instruction: 0.68 ms at 1M atoms for 0.5 GB); block b still owns atoms 256 b .. 256 b + 255 and one fp64 partial
template <int R4>
__global__ void __launch_bounds__(256) k_readout_v(long long N, const float* __restrict__ rpre,
                                                   const float* __restrict__ wr2, const float* __restrict__ br2,
                                                   const float* __restrict__ local_mask, float* __restrict__ rb,
                                                   float* __restrict__ e_atom, double* __restrict__ e_partial) {
    constexpr int R = 4 * R4, APB = 256 / R4;        // atoms per pass of the block
    __shared__ double red[8];
    const int sub = threadIdx.x % R4, slot = threadIdx.x / R4;
    const float4 w = *(const float4*)(wr2 + 4 * sub);
    const float b = br2[0];
    double mine = 0.0;
    for (int pass = 0; pass < 256 / APB; pass++) {
        const long long a = blockIdx.x * 256LL + pass * APB + slot;
        float e = 0.0f, m = 0.0f;
        if (a < N) {
            m = local_mask[a];
            const float4 x = *(const float4*)(rpre + a * R + 4 * sub);
            e = w.x * siluf_(x.x) + w.y * siluf_(x.y) + w.z * siluf_(x.z) + w.w * siluf_(x.w);
            *(float4*)(rb + a * R + 4 * sub) = make_float4(m * w.x * dsiluf_(x.x), m * w.y * dsiluf_(x.y),
                                                           m * w.z * dsiluf_(x.z), m * w.w * dsiluf_(x.w));
        }
#pragma unroll
        for (int o = R4 / 2; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        e += b;
        if (a < N && sub == 0) {
            e_atom[a] = e;
            if (m != 0.0f) mine += (double)e;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mine;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; k++) t += red[k];
        e_partial[blockIdx.x] = t;
    }
}
void readout(const Launch& L, long long N, int R, const float* rpre, const float* wr2, const float* br2,
             const float* local_mask, float* rb, float* e_atom, double* e_partial, int* n_partial) {
    int nb = (int)((N + 255) / 256);
    *n_partial = nb;
    if (N == 0) return;
    if (R == 64) k_readout_v<16><<<nb, 256, 0, L.stream>>>(N, rpre, wr2, br2, local_mask, rb, e_atom, e_partial);
    else if (R == 32) k_readout_v<8><<<nb, 256, 0, L.stream>>>(N, rpre, wr2, br2, local_mask, rb, e_atom, e_partial);
    else if (R == 16) k_readout_v<4><<<nb, 256, 0, L.stream>>>(N, rpre, wr2, br2, local_mask, rb, e_atom, e_partial);
    else k_readout<<<nb, 256, 0, L.stream>>>(N, R, rpre, wr2, br2, local_mask, rb, e_atom, e_partial);
    KLAUNCH(L);
}

// state export in caller order: out[perm[a]] = (s | v_x | v_y | v_z)
__global__ void k_unpermute_state(long long N, int F, const int* __restrict__ perm, const float* __restrict__ s,
                                  const float* __restrict__ v, float* __restrict__ out) {
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * 4 * F) return;
    long long a = idx / (4 * F);
    int k = (int)(idx - a * 4 * F);
    float val = k < F ? s[a * F + k] : v[a * 3 * F + (k - F)];
    out[(size_t)perm[a] * 4 * F + k] = val;
}
void unpermute_state(const Launch& L, long long N, int F, const int* perm, const float* s, const float* v,
                     float* out) {
    if (N == 0) return;
    k_unpermute_state<<<(unsigned)((N * 4 * F + 255) / 256), 256, 0, L.stream>>>(N, F, perm, s, v, out);
    KLAUNCH(L);
}

}  // namespace painn
