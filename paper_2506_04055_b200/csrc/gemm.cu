// gemm.cu -- dense per-atom linear layers:  C[M x N] (+)= A[M x K] . B[N x K]^T + bias   (fp32 row-major)
// (phi-MLP, U/V, update-MLP, readout and their transposed adjoints;
//  weights are fixed, so there are no weight-gradient GEMMs.)
//
// gemm_nt_simt: plain fp32 shared-memory-tiled reference path (kept as the numerical reference of the tcgen05
// path and for shapes the tensor-core kernel does not cover).
#include "common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

constexpr int TM = 64, TN = 64, TK = 16;

// operand-precision emulation (debug knob "gemm_emulate"): 0 fp32, 1 tf32 (RN), 2 bf16 (RN), 3 bf16 hi+lo split
// with the three leading product terms (a_hi b_hi + a_hi b_lo + a_lo b_hi).  Used to size the precision plan of
// the tensor-core path against the parity tolerances before/while it is being written.
int g_gemm_emulate = 0;

__device__ __forceinline__ float rn_tf32(float x) {
    uint32_t u = __float_as_uint(x);
    u += 0xfffu + ((u >> 13) & 1u);
    return __uint_as_float(u & 0xffffe000u);
}
__device__ __forceinline__ float rn_bf16(float x) {
    uint32_t u = __float_as_uint(x);
    u += 0x7fffu + ((u >> 16) & 1u);
    return __uint_as_float(u & 0xffff0000u);
}

__global__ void __launch_bounds__(256) k_gemm_nt_simt(const float* __restrict__ A, int lda,
                                                      const float* __restrict__ B, int ldb, float* __restrict__ C,
                                                      int ldc, long long M, int N, int K,
                                                      const float* __restrict__ bias, int accumulate, int emu) {
    __shared__ float As[TK][TM + 4], Bs[TK][TN + 4], Al[TK][TM + 4], Bh[TK][TN + 4];
    const long long m0 = (long long)blockIdx.x * TM;
    const int n0 = blockIdx.y * TN;
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < K; k0 += TK) {
        for (int idx = threadIdx.x; idx < TM * TK; idx += 256) {
            int r = idx / TK, c = idx % TK;
            long long m = m0 + r;
            float av = (m < M && k0 + c < K) ? A[m * lda + k0 + c] : 0.0f;
            int n = n0 + r;
            float bv = (n < N && k0 + c < K) ? B[(size_t)n * ldb + k0 + c] : 0.0f;
            if (emu == 1) { av = rn_tf32(av); bv = rn_tf32(bv); }
            else if (emu == 2) { av = rn_bf16(av); bv = rn_bf16(bv); }
            else if (emu == 3) {
                float ah = rn_bf16(av), bh = rn_bf16(bv);
                Al[c][r] = rn_bf16(av - ah);
                Bh[c][r] = bh;
                av = ah;
                bv = bh + rn_bf16(bv - bh);
            }
            else if (emu == 4) {   // 3xTF32: hi = truncation to tf32, lo = tf32(a - hi); hi*hi + hi*lo + lo*hi
                float ah = __uint_as_float(__float_as_uint(av) & 0xffffe000u), bh = __uint_as_float(__float_as_uint(bv) & 0xffffe000u);
                Al[c][r] = __uint_as_float(__float_as_uint(av - ah) & 0xffffe000u);
                Bh[c][r] = bh;
                av = ah;
                bv = bh + __uint_as_float(__float_as_uint(bv - bh) & 0xffffe000u);
            }
            As[c][r] = av;
            Bs[c][r] = bv;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < TK; k++) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; i++) { a[i] = As[k][ty * 4 + i]; b[i] = Bs[k][tx * 4 + i]; }
#pragma unroll
            for (int i = 0; i < 4; i++)
#pragma unroll
                for (int j = 0; j < 4; j++) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
            if (emu >= 3) {
#pragma unroll
                for (int i = 0; i < 4; i++) { a[i] = Al[k][ty * 4 + i]; b[i] = Bh[k][tx * 4 + i]; }
#pragma unroll
                for (int i = 0; i < 4; i++)
#pragma unroll
                    for (int j = 0; j < 4; j++) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; i++) {
        long long m = m0 + ty * 4 + i;
        if (m >= M) continue;
#pragma unroll
        for (int j = 0; j < 4; j++) {
            int n = n0 + tx * 4 + j;
            if (n >= N) continue;
            float v = acc[i][j] + (bias ? bias[n] : 0.0f);
            if (accumulate) v += C[m * ldc + n];
            C[m * ldc + n] = v;
        }
    }
}

// weight registry: B pointer -> (hi, lo) TF32 split planes for the tensor-core path (filled at mlp_create)
#include <unordered_map>
static std::unordered_map<const float*, std::pair<const float*, const float*>> g_split;
int g_last_gemm_tc = 0;   // set to 1 by gemm_nt when the tensor-core kernel was used (test hook)
int g_gemm_path = 0;   // 0: tensor cores when the shape is covered, 1: force the SIMT reference path
void gemm_register_split(const float* W, const float* hi, const float* lo) { g_split[W] = {hi, lo}; }
void gemm_unregister_split(const float* W) { g_split.erase(W); }
bool gemm_nt_tc(const Launch& L, const float* A, int lda, const float* Whi, const float* Wlo, int ldw, float* C, int ldc,
                long long M, int N, int K, const float* bias, bool accumulate);

void gemm_nt(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
             int N, int K, const float* bias, bool accumulate) {
    if (M == 0) return;
    if (g_gemm_path == 0 && g_gemm_emulate == 0) {
        auto it = g_split.find(B);
        if (it != g_split.end() &&
            gemm_nt_tc(L, A, lda, it->second.first, it->second.second, ldb, C, ldc, M, N, K, bias, accumulate)) {
            g_last_gemm_tc = 1;
            return;
        }
    }
    dim3 grid((unsigned)((M + TM - 1) / TM), (unsigned)((N + TN - 1) / TN));
    k_gemm_nt_simt<<<grid, 256, 0, L.stream>>>(A, lda, B, ldb, C, ldc, M, N, K, bias, accumulate ? 1 : 0,
                                                   g_gemm_emulate);
    KLAUNCH(L);
}

}  // namespace painn
