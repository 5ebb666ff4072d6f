// gemm.cu -- dense per-atom linear layers:  C[M x N] (+)= A[M x K] . B[N x K]^T + bias   (fp32 row-major)
// (phi-MLP, U/V, update-MLP, readout and their transposed adjoints;
//  weights are fixed, so there are no weight-gradient GEMMs.)
//
// k_gemm_nt_simt: plain fp32 shared-memory-tiled path for the shapes the tensor-core kernels do not cover (F = 32, 64
// models, readout of width 16 / 32).
#include "common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

constexpr int TM = 64, TN = 64, TK = 16;

__global__ void __launch_bounds__(256) k_gemm_nt_simt(const float* __restrict__ A, int lda,
                                                      const float* __restrict__ B, int ldb, float* __restrict__ C,
                                                      int ldc, long long M, int N, int K,
                                                      const float* __restrict__ bias, int accumulate) {
    __shared__ float As[TK][TM + 4], Bs[TK][TN + 4];
    const long long m0 = (long long)blockIdx.x * TM;
    const int n0 = blockIdx.y * TN;
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < K; k0 += TK) {
        for (int idx = threadIdx.x; idx < TM * TK; idx += 256) {
            int r = idx / TK, c = idx % TK;
            long long m = m0 + r;
            As[c][r] = (m < M && k0 + c < K) ? A[m * lda + k0 + c] : 0.0f;
            int n = n0 + r;
            Bs[c][r] = (n < N && k0 + c < K) ? B[(size_t)n * ldb + k0 + c] : 0.0f;
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


// ------------------------------------------------------------------------------------------------
// k_sgemm128: fp32 FFMA path of the FORWARD linear layers (round-to-nearest accumulation; B3).
// 128 x 128 x 8 tiles, 256 threads, 8 x 8 outputs per thread as 2 x 2 strips of 4 (conflict-free LDS.128),
// operands transposed into shared memory ([k][row]), next tile prefetched into registers during the FMAs.
// ACT_A: apply SiLU to A while loading (fuses the activation of the two-layer MLPs into the second GEMM).
__device__ __forceinline__ float silu_g(float x) { return x / (1.0f + __expf(-x)); }

template <bool ACT_A>
__global__ void __launch_bounds__(256, 2) k_sgemm128(const float* __restrict__ A, int lda, const float* __restrict__ B,
                                                      int ldb, float* __restrict__ C, int ldc, long long M, int N, int K,
                                                      const float* __restrict__ bias, int accumulate) {
    constexpr int BMs = 128, BNs = 128, BKs = 8, PAD = 4;
    __shared__ __align__(16) float As[2][BKs][BMs + PAD];
    __shared__ __align__(16) float Bs[2][BKs][BNs + PAD];
    const int tid = threadIdx.x;
    const int n0 = blockIdx.x * BNs;                       // N tiles fastest: CTAs sharing an A tile run together
    const long long m0 = (long long)blockIdx.y * BMs;
    const int lrow = tid >> 1, lk = (tid & 1) * 4;         // loader: one float4 along K per thread per operand
    const int tx = tid & 15, ty = tid >> 4;
    const long long arow = m0 + lrow;
    const bool a_ok = arow < M;
    const float* ap = A + (a_ok ? arow : 0) * lda + lk;
    const float* bp = B + (size_t)(n0 + lrow) * ldb + lk;
    float acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
        for (int j = 0; j < 8; j++) acc[i][j] = 0.0f;
    float4 ra = a_ok ? *(const float4*)ap : make_float4(0.f, 0.f, 0.f, 0.f);
    float4 rb = *(const float4*)bp;
    auto stash = [&](int buf) {
        if (ACT_A) { ra.x = silu_g(ra.x); ra.y = silu_g(ra.y); ra.z = silu_g(ra.z); ra.w = silu_g(ra.w); }
        As[buf][lk + 0][lrow] = ra.x; As[buf][lk + 1][lrow] = ra.y; As[buf][lk + 2][lrow] = ra.z; As[buf][lk + 3][lrow] = ra.w;
        Bs[buf][lk + 0][lrow] = rb.x; Bs[buf][lk + 1][lrow] = rb.y; Bs[buf][lk + 2][lrow] = rb.z; Bs[buf][lk + 3][lrow] = rb.w;
    };
    stash(0);
    __syncthreads();
    const int nk = K / BKs;
    for (int kb = 0; kb < nk; kb++) {
        const int cur = kb & 1;
        if (kb + 1 < nk) {
            ra = a_ok ? *(const float4*)(ap + (kb + 1) * BKs) : make_float4(0.f, 0.f, 0.f, 0.f);
            rb = *(const float4*)(bp + (kb + 1) * BKs);
        }
#pragma unroll
        for (int k = 0; k < BKs; k++) {
            const float4 a0 = *(const float4*)&As[cur][k][ty * 4], a1 = *(const float4*)&As[cur][k][64 + ty * 4];
            const float4 b0 = *(const float4*)&Bs[cur][k][tx * 4], b1 = *(const float4*)&Bs[cur][k][64 + tx * 4];
            const float a[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float b[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
            for (int i = 0; i < 8; i++)
#pragma unroll
                for (int j = 0; j < 8; j++) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        if (kb + 1 < nk) {
            stash(cur ^ 1);
            __syncthreads();
        }
    }
#pragma unroll
    for (int i = 0; i < 8; i++) {
        const long long m = m0 + (i < 4 ? ty * 4 + i : 64 + ty * 4 + (i - 4));
        if (m >= M) continue;
#pragma unroll
        for (int jh = 0; jh < 2; jh++) {
            const int n = n0 + jh * 64 + tx * 4;
            float4 v = make_float4(acc[i][jh * 4], acc[i][jh * 4 + 1], acc[i][jh * 4 + 2], acc[i][jh * 4 + 3]);
            if (bias) { const float4 bb = *(const float4*)(bias + n); v.x += bb.x; v.y += bb.y; v.z += bb.z; v.w += bb.w; }
            float* cp = C + m * ldc + n;
            if (accumulate) { const float4 o = *(const float4*)cp; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
            *(float4*)cp = v;
        }
    }
}

// Weight registry (per model, common.cuh::GemmRegistry): weight pointer -> (hi, lo) TF32 split planes of the 3xTF32
// kernel and -> fp16 integer slices of the exact kernel; filled at mlp_create, read-only afterwards.  Which path a
// call takes comes with the Launch context (gemm_path / fwd_exact), never from process-wide state.
void gemm_register_split(GemmRegistry& reg, const float* W, const float* hi, const float* lo) { reg.split[W] = {hi, lo}; }
bool gemm_nt_tc(const Launch& L, const float* A, int lda, const float* Whi, const float* Wlo, int ldw, float* C, int ldc,
                long long M, int N, int K, const float* bias, bool accumulate, const float* dsilu_pre = nullptr, int ld_pre = 0,
                const float* resid = nullptr);
void mul_dsilu(const Launch& L, long long n, const float* pre, float* g);

static bool split_of(const Launch& L, const float* B, const float** hi, const float** lo) {
    if (!L.reg) return false;
    auto it = L.reg->split.find(B);
    if (it == L.reg->split.end()) return false;
    *hi = it->second.first; *lo = it->second.second;
    return true;
}
static void used_tc(const Launch& L) { if (L.used_tc) *L.used_tc = 1; }

bool gemm_act_supported(int N, int K) { return N % 128 == 0 && K % 8 == 0; }

void gemm_nt(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
             int N, int K, const float* bias, bool accumulate) {
    gemm_nt_act(L, A, lda, B, ldb, C, ldc, M, N, K, bias, accumulate, false);
}

// C = (A . B^T) * SiLU'(pre)   (pre: [M x N] contiguous): adjoint of a SiLU layer; fused into the 3xTF32 epilogue when
// that kernel covers the shape, otherwise GEMM followed by the element-wise kernel
void gemm_nt_dsilu(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
                   int N, int K, const float* pre) {
    if (M == 0) return;
    const float *hi, *lo;
    if (L.gemm_path == 0 && ldc == N && split_of(L, B, &hi, &lo) &&
        gemm_nt_tc(L, A, lda, hi, lo, ldb, C, ldc, M, N, K, nullptr, false, pre, N)) {
        used_tc(L);
        return;
    }
    gemm_nt(L, A, lda, B, ldb, C, ldc, M, N, K, nullptr, false);
    mul_dsilu(L, M * N, pre, C);
}

// C = resid + A . B^T  (resid: [M x N], row stride ldc, may not overlap C): the adjoint GEMMs that add to a term held in
// another buffer read it in the epilogue instead of having it copied into C first
void gemm_nt_resid(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
                   int N, int K, const float* resid) {
    if (M == 0) return;
    const float *hi, *lo;
    if (L.gemm_path == 0 && split_of(L, B, &hi, &lo) &&
        gemm_nt_tc(L, A, lda, hi, lo, ldb, C, ldc, M, N, K, nullptr, false, nullptr, 0, resid)) {
        used_tc(L);
        return;
    }
    cudaMemcpy2DAsync(C, (size_t)ldc * 4, resid, (size_t)ldc * 4, (size_t)N * 4, (size_t)M, cudaMemcpyDeviceToDevice, L.stream);
    gemm_nt(L, A, lda, B, ldb, C, ldc, M, N, K, nullptr, true);
}

// act_a: C = SiLU(A) . B^T + bias  (forward GEMMs only: the exact tensor-core kernel or the fp32 FFMA kernel)
void gemm_nt_act(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
                 int N, int K, const float* bias, bool accumulate, bool act_a) {
    if (M == 0) return;
    const bool fast_ok = N % 128 == 0 && K % 8 == 0 && lda % 4 == 0 && ldb % 4 == 0 &&
                         ldc % 4 == 0 && ((((uintptr_t)A | (uintptr_t)B | (uintptr_t)C | (uintptr_t)bias) & 15) == 0);
    const bool fwd = act_a || L.gemm_path == 1;      // round-to-nearest / exact accumulation wanted (B3)
    if (fwd && L.fwd_exact && gemm_nt_exact(L, A, lda, B, C, ldc, M, N, K, bias, accumulate, act_a)) {
        used_tc(L);
        return;
    }
    if (fwd && fast_ok && M / 128 < 65535) {
        dim3 grid((unsigned)(N / 128), (unsigned)((M + 127) / 128));
        if (act_a) k_sgemm128<true><<<grid, 256, 0, L.stream>>>(A, lda, B, ldb, C, ldc, M, N, K, bias, accumulate ? 1 : 0);
        else k_sgemm128<false><<<grid, 256, 0, L.stream>>>(A, lda, B, ldb, C, ldc, M, N, K, bias, accumulate ? 1 : 0);
        KLAUNCH(L);
        return;
    }
    if (act_a) return;   // shapes neither kernel covers: callers check gemm_act_supported() before asking for act_a
    const float *hi, *lo;
    if (L.gemm_path == 0 && split_of(L, B, &hi, &lo) && gemm_nt_tc(L, A, lda, hi, lo, ldb, C, ldc, M, N, K, bias, accumulate)) {
        used_tc(L);
        return;
    }
    dim3 grid((unsigned)((M + TM - 1) / TM), (unsigned)((N + TN - 1) / TN));
    k_gemm_nt_simt<<<grid, 256, 0, L.stream>>>(A, lda, B, ldb, C, ldc, M, N, K, bias, accumulate ? 1 : 0);
    KLAUNCH(L);
}

}  // namespace painn
