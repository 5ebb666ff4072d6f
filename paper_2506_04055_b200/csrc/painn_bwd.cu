// painn_bwd.cu -- hand-derived adjoint of the PaiNN layers, force assembly, ghost fold, virial
// (north_star item 4; PAPER.md:60-66 force sum rule).
//
// Equations: DESIGN.md section 2 "Adjoint".  xb == dE/dx.  The message adjoint is evaluated in its NO-ATOMICS
// gather form: the filter depends on |r| only and the edge set is symmetric, so everything edge e = (i <- j)
// scatters onto its sender j can be gathered by j walking its OWN CSR row (slot x of row j holds neighbour i and
// r' = r_i - r_j = -r_e):
//   Y_j[c]   = sum_x w^vv o vb'_i[c]           vb_j[c] = vb'_j[c] + phi^vv_j o Y_j[c]
//   phib_j   = [ sum_x w^s o sb'_i | sum_x w^vs o (vb'_i . u_e) | sum_c v_j[c] o Y_j[c] ]
//   g_e      = db_e u_e + (ub_e - (ub_e . u_e) u_e) / d_e ,   stored at slot x  (G[x], accumulated over layers)
// with u_e = -r'/d.  Forces then follow by a second gather through the reverse-edge index:
//   F_j = sum_x ( G[rev[x]] - G[x] ),   W_ab = sum_x r'_x,a G[x]_b .
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include "common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

// ------------------------------------------------------------------------------------------------ a11
// ab = [ sum_c vb[c] o p[c] | sb o D | sb ] ;  Db = sb o a^sv ;  pb[c] = vb[c] o a^vv + Db o q[c] ;  qb[c] = Db o p[c]
__global__ void k_update_bwd1(long long N, int F, const float* __restrict__ sb, const float* __restrict__ vb,
                              const float* __restrict__ pq, const float* __restrict__ a_, float* __restrict__ ab,
                              float* __restrict__ pqb) {
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F) return;
    long long a = idx / F;
    int f = (int)(idx - a * F);
    const float* p = pq + a * 6 * F + f;
    const float* q = p + F;
    const float avv = a_[a * 3 * F + f], asv = a_[a * 3 * F + F + f];
    const float sbi = sb[idx];
    const float Db = sbi * asv;
    float D = 0.0f, vp = 0.0f;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const float pc = p[c * 2 * F], qc = q[c * 2 * F], vbc = vb[a * 3 * F + c * F + f];
        D += pc * qc;
        vp += vbc * pc;
        pqb[a * 6 * F + c * 2 * F + f] = vbc * avv + Db * qc;
        pqb[a * 6 * F + c * 2 * F + F + f] = Db * pc;
    }
    ab[a * 3 * F + f] = vp;
    ab[a * 3 * F + F + f] = sbi * D;
    ab[a * 3 * F + 2 * F + f] = sbi;
}
void update_bwd1(const Launch& L, long long N, int F, const float* sb, const float* vb, const float* pq,
                 const float* a, float* ab, float* pqb) {
    if (N == 0) return;
    k_update_bwd1<<<(unsigned)((N * F + 255) / 256), 256, 0, L.stream>>>(N, F, sb, vb, pq, a, ab, pqb);
    KLAUNCH(L);
}
// qb[c] += nb o q[c] / n ;  sb' = sb + ds ;  vb'[c] = vb[c]  (the U^T pb + V^T qb GEMM accumulates on top)
// four channels per thread (16-byte accesses: the scalar form moved 4.6 TB/s, launch-list of profiles/r01_launches_cfg5.md)
__global__ void k_update_bwd2(long long N, int F, const float* __restrict__ sb, const float* __restrict__ vb,
                              const float* __restrict__ snb, const float* __restrict__ sn,
                              const float* __restrict__ pq, float* __restrict__ pqb, float* __restrict__ s1b,
                              float* __restrict__ v1b) {
    const int F4 = F >> 2;
    long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (idx >= N * F4) return;
    long long a = idx / F4;
    int f = (int)(idx - a * F4) * 4;
    const float4 nb = *(const float4*)(snb + a * 2 * F + F + f), nn = *(const float4*)(sn + a * 2 * F + F + f);
    const float4 r = make_float4(nb.x / nn.x, nb.y / nn.y, nb.z / nn.z, nb.w / nn.w);
    float4 q[3], qb[3];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        q[c] = *(const float4*)(pq + a * 6 * F + c * 2 * F + F + f);
        qb[c] = *(const float4*)(pqb + a * 6 * F + c * 2 * F + F + f);
    }
    const float4 s0 = *(const float4*)(sb + a * F + f), s1 = *(const float4*)(snb + a * 2 * F + f);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        qb[c].x += r.x * q[c].x; qb[c].y += r.y * q[c].y; qb[c].z += r.z * q[c].z; qb[c].w += r.w * q[c].w;
        *(float4*)(pqb + a * 6 * F + c * 2 * F + F + f) = qb[c];
        if (v1b) *(float4*)(v1b + a * 3 * F + c * F + f) = *(const float4*)(vb + a * 3 * F + c * F + f);   // nullptr: the U|V adjoint GEMM reads vb as its residual
    }
    *(float4*)(s1b + a * F + f) = make_float4(s0.x + s1.x, s0.y + s1.y, s0.z + s1.z, s0.w + s1.w);
}
void update_bwd2(const Launch& L, long long N, int F, const float* sb, const float* vb, const float* snb,
                 const float* sn, const float* pq, float* pqb, float* s1b, float* v1b) {
    if (N == 0) return;
    k_update_bwd2<<<(unsigned)((N * (F / 4) + 255) / 256), 256, 0, L.stream>>>(N, F, sb, vb, snb, sn, pq, pqb, s1b, v1b);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ a12
constexpr int BWD_CHUNK = 32;
template <int KMAX>
__global__ void __launch_bounds__(128) k_message_bwd(long long N, int F, int K, float inv_rc,
                                                     const int* __restrict__ row_ptr,
                                                     const float4* __restrict__ ej,
                                                     const float* __restrict__ s1b, const float* __restrict__ v1b,
                                                     const float* __restrict__ phi, const float* __restrict__ v_in,
                                                     const float* __restrict__ Wf, const float* __restrict__ bf,
                                                     float* __restrict__ phib, float* __restrict__ vb_out,
                                                     float4* __restrict__ G, int first) {
    __shared__ float red[4][BWD_CHUNK][4];
    const long long j = blockIdx.x;
    const int f = threadIdx.x;
    const int lane = f & 31, warp = f >> 5, nwarp = (F + 31) >> 5;
    float wS[KMAX], wVS[KMAX], wVV[KMAX];
#pragma unroll
    for (int n = 0; n < KMAX; n++) {
        wS[n] = n < K ? Wf[(size_t)(f)*K + n] : 0.0f;
        wVS[n] = n < K ? Wf[(size_t)(F + f) * K + n] : 0.0f;
        wVV[n] = n < K ? Wf[(size_t)(2 * F + f) * K + n] : 0.0f;
    }
    const float bS = bf[f], bVS = bf[F + f], bVV = bf[2 * F + f];
    const size_t F3 = 3 * (size_t)F;
    const float phiS = phi[j * F3 + f], phiVS = phi[j * F3 + F + f], phiVV = phi[j * F3 + 2 * F + f];
    const float vj0 = v_in[j * F3 + f], vj1 = v_in[j * F3 + F + f], vj2 = v_in[j * F3 + 2 * F + f];
    float pbS = 0.0f, pbVS = 0.0f, Y0 = 0.0f, Y1 = 0.0f, Y2 = 0.0f;
    const float PI_F = 3.14159265358979323846f;
    const int e0 = row_ptr[j], e1 = row_ptr[j + 1];
    for (int c0 = e0; c0 < e1; c0 += BWD_CHUNK) {
        const int cn = min(BWD_CHUNK, e1 - c0);
        for (int k = 0; k < cn; k++) {
            const float4 r = ej[c0 + k];
            const int i_raw = __float_as_int(r.w);
            const bool dummy = i_raw < 0;                 // padding slot: zero weight, gathers its own row
            const int i = dummy ? ~i_raw : i_raw;
            const float d2 = r.x * r.x + r.y * r.y + r.z * r.z;
            const float inv_d = rsqrtf(d2);
            const float d = d2 * inv_d;
            const float ux = -r.x * inv_d, uy = -r.y * inv_d, uz = -r.z * inv_d;   // u_e of edge (i <- j)
            float s1, c1;
            sincospif(d * inv_rc, &s1, &c1);
            float sn_ = s1, cn_ = c1;
            const float a1 = PI_F * inv_rc;
            const float fc = dummy ? 0.0f : 0.5f * (1.0f + c1);
            const float dfc = dummy ? 0.0f : -0.5f * a1 * s1;
            // w = Wf (fc rho) + bf fc ;  w' = Wf (fc' rho + fc rho') + bf fc'   (both as GEMM operands)
            float wS_ = fmaf(bS, fc, 0.f), wVS_ = fmaf(bVS, fc, 0.f), wVV_ = fmaf(bVV, fc, 0.f);
            float dwS = fmaf(bS, dfc, 0.f), dwVS = fmaf(bVS, dfc, 0.f), dwVV = fmaf(bVV, dfc, 0.f);
#pragma unroll
            for (int n = 0; n < KMAX; n++) {
                const float rho = sn_ * inv_d;
                const float drho = ((float)(n + 1) * a1 * cn_ - rho) * inv_d;   // (n pi/rc) cos/d - sin/d^2
                const float r0 = fc * rho, r1 = dfc * rho + fc * drho;
                wS_ = fmaf(wS[n], r0, wS_); wVS_ = fmaf(wVS[n], r0, wVS_); wVV_ = fmaf(wVV[n], r0, wVV_);
                dwS = fmaf(wS[n], r1, dwS); dwVS = fmaf(wVS[n], r1, dwVS); dwVV = fmaf(wVV[n], r1, dwVV);
                const float t = sn_ * c1 + cn_ * s1;
                cn_ = cn_ * c1 - sn_ * s1;
                sn_ = t;
            }
            const float sbi = s1b[(size_t)i * F + f];
            const float vb0 = v1b[(size_t)i * F3 + f], vb1 = v1b[(size_t)i * F3 + F + f],
                        vb2 = v1b[(size_t)i * F3 + 2 * F + f];
            const float X = vb0 * ux + vb1 * uy + vb2 * uz;
            const float Z = vb0 * vj0 + vb1 * vj1 + vb2 * vj2;
            pbS += wS_ * sbi;
            pbVS += wVS_ * X;
            Y0 += wVV_ * vb0; Y1 += wVV_ * vb1; Y2 += wVV_ * vb2;
            float db = phiS * sbi * dwS + phiVS * X * dwVS + phiVV * Z * dwVV;
            const float t = wVS_ * phiVS;
            float ub0 = t * vb0, ub1 = t * vb1, ub2 = t * vb2;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                db += __shfl_xor_sync(0xffffffffu, db, o);
                ub0 += __shfl_xor_sync(0xffffffffu, ub0, o);
                ub1 += __shfl_xor_sync(0xffffffffu, ub1, o);
                ub2 += __shfl_xor_sync(0xffffffffu, ub2, o);
            }
            if (lane == 0) { red[warp][k][0] = db; red[warp][k][1] = ub0; red[warp][k][2] = ub1; red[warp][k][3] = ub2; }
        }
        __syncthreads();
        if (f < cn) {
            float db = 0.0f, ub0 = 0.0f, ub1 = 0.0f, ub2 = 0.0f;
            for (int w = 0; w < nwarp; w++) { db += red[w][f][0]; ub0 += red[w][f][1]; ub1 += red[w][f][2]; ub2 += red[w][f][3]; }
            const float4 r = ej[c0 + f];
            const float d2 = r.x * r.x + r.y * r.y + r.z * r.z;
            const float inv_d = rsqrtf(d2);
            const float ux = -r.x * inv_d, uy = -r.y * inv_d, uz = -r.z * inv_d;
            const float uu = ub0 * ux + ub1 * uy + ub2 * uz;
            float4 g = make_float4(db * ux + (ub0 - uu * ux) * inv_d, db * uy + (ub1 - uu * uy) * inv_d,
                                   db * uz + (ub2 - uu * uz) * inv_d, 0.0f);
            if (!first) { const float4 o = G[c0 + f]; g.x += o.x; g.y += o.y; g.z += o.z; }
            G[c0 + f] = g;
        }
        __syncthreads();
    }
    phib[j * F3 + f] = pbS;
    phib[j * F3 + F + f] = pbVS;
    phib[j * F3 + 2 * F + f] = vj0 * Y0 + vj1 * Y1 + vj2 * Y2;
    vb_out[j * F3 + f] = v1b[j * F3 + f] + phiVV * Y0;
    vb_out[j * F3 + F + f] = v1b[j * F3 + F + f] + phiVV * Y1;
    vb_out[j * F3 + 2 * F + f] = v1b[j * F3 + 2 * F + f] + phiVV * Y2;
}

void message_bwd(const Launch& L, long long N, int F, int K, float rc, const int* row_ptr, const float4* ej,
                 const float* s1b, const float* v1b, const float* phi, const float* v_in, const float* Wf,
                 const float* bf, float* phib, float* vb_out, float4* G, bool first) {
    if (N == 0) return;
    unsigned grid = (unsigned)N;
#define MB(KM) k_message_bwd<KM><<<grid, F, 0, L.stream>>>(N, F, K, 1.0f / rc, row_ptr, ej, s1b, v1b, phi, v_in, Wf, bf, phib, vb_out, G, first ? 1 : 0)
    if (K <= 16) MB(16); else if (K <= 20) MB(20); else MB(32);
#undef MB
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ a13
// One warp per sorted atom a:  F_a = sum_x (G[rev[x]] - G[x]) ; virial partial sum_x r'_x (x) G[x].
// Forces are added (fp64 atomics) onto the caller-order row of the atom itself, or of its owner when a ghost
// owner map is given; `forces` must be zeroed before.
__global__ void __launch_bounds__(256) k_force_final(long long N, long long n_local, const int* __restrict__ row_ptr,
                                                     const float4* __restrict__ ej, const int* __restrict__ rev,
                                                     const float4* __restrict__ G, const int* __restrict__ perm,
                                                     const int* __restrict__ ghost_owner,
                                                     double* __restrict__ forces, double* __restrict__ w_partial) {
    __shared__ double wsum[8][9];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long a = blockIdx.x * 8ll + warp;
    float fx = 0.f, fy = 0.f, fz = 0.f, w[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    if (a < N) {
        for (int x = row_ptr[a] + lane; x < row_ptr[a + 1]; x += 32) {
            const float4 g = G[x], gr = G[rev[x]], r = ej[x];
            fx += gr.x - g.x; fy += gr.y - g.y; fz += gr.z - g.z;
            w[0] += r.x * g.x; w[1] += r.x * g.y; w[2] += r.x * g.z;
            w[3] += r.y * g.x; w[4] += r.y * g.y; w[5] += r.y * g.z;
            w[6] += r.z * g.x; w[7] += r.z * g.y; w[8] += r.z * g.z;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        fx += __shfl_xor_sync(0xffffffffu, fx, o);
        fy += __shfl_xor_sync(0xffffffffu, fy, o);
        fz += __shfl_xor_sync(0xffffffffu, fz, o);
#pragma unroll
        for (int k = 0; k < 9; k++) w[k] += __shfl_xor_sync(0xffffffffu, w[k], o);
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 9; k++) wsum[warp][k] = (double)w[k];
        if (a < N) {
            long long i = perm[a];
            if (ghost_owner != nullptr && i >= n_local) i = ghost_owner[i - n_local];
            atomicAdd(&forces[3 * i + 0], (double)fx);
            atomicAdd(&forces[3 * i + 1], (double)fy);
            atomicAdd(&forces[3 * i + 2], (double)fz);
        }
    }
    __syncthreads();
    if (threadIdx.x < 9) {
        double t = 0.0;
        for (int k = 0; k < 8; k++) t += wsum[k][threadIdx.x];
        w_partial[(size_t)blockIdx.x * 9 + threadIdx.x] = t;
    }
}
void force_final(const Launch& L, long long N, long long n_local, const int* row_ptr, const float4* ej,
                 const int* rev, const float4* G, const int* perm, const int* ghost_owner, double* forces,
                 double* w_partial, int* n_partial) {
    int nb = (int)((N + 7) / 8);
    *n_partial = nb;
    if (N == 0) return;
    k_force_final<<<nb, 256, 0, L.stream>>>(N, n_local, row_ptr, ej, rev, G, perm, ghost_owner, forces, w_partial);
    KLAUNCH(L);
}

// deterministic final sums: energy (n_e partials) and raw 3x3 virial (n_w x 9 partials) -> 6 symmetrised components
__global__ void __launch_bounds__(256) k_reduce_final(const double* __restrict__ e_partial, int n_e,
                                                       const double* __restrict__ w_partial, int n_w,
                                                       double* __restrict__ energy, double* __restrict__ virial) {
    __shared__ double red[10][256];
    double acc[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = threadIdx.x; i < n_e; i += 256) acc[9] += e_partial[i];
    for (int i = threadIdx.x; i < n_w; i += 256)
        for (int k = 0; k < 9; k++) acc[k] += w_partial[(size_t)i * 9 + k];
    for (int k = 0; k < 10; k++) red[k][threadIdx.x] = acc[k];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            for (int k = 0; k < 10; k++) red[k][threadIdx.x] += red[k][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        energy[0] = red[9][0];
        virial[0] = red[0][0]; virial[1] = red[4][0]; virial[2] = red[8][0];
        virial[3] = 0.5 * (red[1][0] + red[3][0]);
        virial[4] = 0.5 * (red[2][0] + red[6][0]);
        virial[5] = 0.5 * (red[5][0] + red[7][0]);
    }
}
// first stage for large systems: block b folds its contiguous share of both partial lists into scratch[b][0..9] (flat,
// coalesced reads of the [n_w][9] list: with 288 = 32 x 9 threads every thread stays on one component)
constexpr int RED_BLOCKS = 128, RED_THREADS = 288;
__global__ void __launch_bounds__(RED_THREADS) k_reduce_stage1(const double* __restrict__ e_partial, int n_e,
                                                               const double* __restrict__ w_partial, int n_w,
                                                               double* __restrict__ scratch) {
    __shared__ double red[RED_THREADS];
    __shared__ double rede[RED_THREADS];
    const int t = threadIdx.x, b = blockIdx.x;
    const long long cw = (n_w + RED_BLOCKS - 1) / RED_BLOCKS, w0 = b * cw * 9, w1 = min((long long)n_w, (b + 1) * cw) * 9;
    double acc = 0.0, ae = 0.0;
    for (long long j = w0 + t; j < w1; j += RED_THREADS) acc += w_partial[j];
    const int ce = (n_e + RED_BLOCKS - 1) / RED_BLOCKS, e1 = min(n_e, (b + 1) * ce);
    for (int j = b * ce + t; j < e1; j += RED_THREADS) ae += e_partial[j];
    red[t] = acc; rede[t] = ae;
    __syncthreads();
    if (t < 9) {
        double x = 0.0;
        for (int i = 0; i < RED_THREADS / 9; i++) x += red[t + 9 * i];
        scratch[b * 9 + t] = x;
    } else if (t == 32) {
        double x = 0.0;
        for (int i = 0; i < RED_THREADS; i++) x += rede[i];
        scratch[RED_BLOCKS * 9 + b] = x;
    }
}
// scratch: RED_BLOCKS x 10 doubles (used when n_w is large; the single-block pass alone took 0.35 ms at 1M atoms)
void reduce_final(const Launch& L, const double* e_partial, int n_e, const double* w_partial, int n_w,
                  double* scratch, double* energy, double* virial) {
    if (scratch && n_w > 8192) {
        k_reduce_stage1<<<RED_BLOCKS, RED_THREADS, 0, L.stream>>>(e_partial, n_e, w_partial, n_w, scratch);
        KLAUNCH(L);
        e_partial = scratch + RED_BLOCKS * 9; n_e = RED_BLOCKS;
        w_partial = scratch; n_w = RED_BLOCKS;
    }
    k_reduce_final<<<1, 256, 0, L.stream>>>(e_partial, n_e, w_partial, n_w, energy, virial);
    KLAUNCH(L);
}

}  // namespace painn
