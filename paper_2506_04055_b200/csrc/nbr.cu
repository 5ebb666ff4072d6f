// nbr.cu -- cell-list neighbour build (north_star item 1).
//
// Replaces the CPU (LAMMPS) neighbour list + per-step cutoff pruning of PAPER.md:58, 68 with a GPU build:
//   bin atoms into cells of side >= rc  ->  counting sort by cell (stable: ties by caller index)  ->
//   per-atom count over the 27-cell stencil  ->  exclusive scan  ->  fill a fixed-capacity CSR
//   (overflow flag, regrow by the host)  ->  reverse-edge index.
// The cutoff predicate is evaluated in fp64 with explicit round-to-nearest mul/add (no FMA contraction) on the
// positions AS GIVEN, so the edge set is bit-identical to the definition (reading A4).
#include "common.cuh"

namespace painn {

#define KLAUNCH(L) (++*(L).counter)

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

// ------------------------------------------------------------------------------------------------ a0 + a1
__global__ void k_bin(const double* __restrict__ pos, const int* __restrict__ types, long long N, int n_species,
                      Grid g, int* __restrict__ cell_id, signed char* __restrict__ wrap,
                      int* __restrict__ cell_count, int* __restrict__ flags, long long n_local,
                      const int* __restrict__ ghost_owner) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int t = types[i];
    int bad = 0;
    if (t < 0 || t >= n_species) bad |= FLAG_TYPE_RANGE;
    if (ghost_owner != nullptr && i >= n_local) {        // the fold adds onto forces[owner]: it must be a local row
        const int o = ghost_owner[i - n_local];
        if (o < 0 || o >= n_local) bad |= FLAG_OWNER_RANGE;
    }
    int c[3];
#pragma unroll
    for (int d = 0; d < 3; d++) {
        double x = pos[3 * i + d];
        if (!isfinite(x)) { bad |= FLAG_NONFINITE; x = 0.0; }
        double w = 0.0, xw;
        if (g.periodic) {
            w = floor(x / g.box[d]);
            xw = x - w * g.box[d];
            if (fabs(w) > 100.0) { bad |= FLAG_NONFINITE; w = 0.0; xw = 0.0; }
        } else {
            xw = x - g.origin[d];
        }
        wrap[3 * i + d] = (signed char)(int)w;
        c[d] = clampi((int)floor(xw * g.inv_side[d]), 0, g.n[d] - 1);
    }
    int cell = cell_encode(g, c[0], c[1], c[2]);
    cell_id[i] = cell;
    atomicAdd(&cell_count[cell], 1);
    if (bad) atomicOr(flags, bad);
}

void nbr_bin(const Launch& L, const double* pos, const int* types, long long N, int n_species, Grid g,
             int* cell_id, signed char* wrap, int* cell_count, int* flags, long long n_local, const int* ghost_owner) {
    if (N == 0) return;
    k_bin<<<(unsigned)((N + 255) / 256), 256, 0, L.stream>>>(pos, types, N, n_species, g, cell_id, wrap,
                                                             cell_count, flags, n_local, ghost_owner);
    KLAUNCH(L);
}

// bounding box (ghost / open mode): bbox6 = {min x,y,z, max x,y,z}; initialised by the kernel's first block
__global__ void k_bbox(const double* __restrict__ pos, long long N, double* __restrict__ part) {
    __shared__ double smin[3][256], smax[3][256];
    double mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x)
        for (int d = 0; d < 3; d++) {
            double x = pos[3 * i + d];
            if (isfinite(x)) { mn[d] = fmin(mn[d], x); mx[d] = fmax(mx[d], x); }
        }
    for (int d = 0; d < 3; d++) { smin[d][threadIdx.x] = mn[d]; smax[d][threadIdx.x] = mx[d]; }
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            for (int d = 0; d < 3; d++) {
                smin[d][threadIdx.x] = fmin(smin[d][threadIdx.x], smin[d][threadIdx.x + s]);
                smax[d][threadIdx.x] = fmax(smax[d][threadIdx.x], smax[d][threadIdx.x + s]);
            }
        __syncthreads();
    }
    if (threadIdx.x < 3) {
        part[6 * blockIdx.x + threadIdx.x] = smin[threadIdx.x][0];
        part[6 * blockIdx.x + 3 + threadIdx.x] = smax[threadIdx.x][0];
    }
}
__global__ void k_bbox_final(const double* __restrict__ part, int nb, double* __restrict__ bbox6) {
    int d = threadIdx.x;
    if (d >= 6) return;
    double v = part[d];
    for (int b = 1; b < nb; b++) v = d < 3 ? fmin(v, part[6 * b + d]) : fmax(v, part[6 * b + d]);
    bbox6[d] = v;
}
// bbox6 must have room for 6 + 6*256 doubles (result first, partials after)
void nbr_bbox(const Launch& L, const double* pos, long long N, double* bbox6) {
    int nb = (int)((N + 255) / 256);
    if (nb > 256) nb = 256;
    if (nb < 1) nb = 1;
    k_bbox<<<nb, 256, 0, L.stream>>>(pos, N, bbox6 + 6);
    KLAUNCH(L);
    k_bbox_final<<<1, 32, 0, L.stream>>>(bbox6 + 6, nb, bbox6);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ scan
constexpr int SCAN_T = 1024, SCAN_I = 4, SCAN_B = SCAN_T * SCAN_I;

__device__ __forceinline__ int block_exclusive_scan(int v, int* total) {   // 1024 threads
    __shared__ int wsum[32];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
        int s = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
        wsum[lane] = s;
    }
    __syncthreads();
    int base = w ? wsum[w - 1] : 0;
    *total = wsum[31];
    return base + x - v;
}

__global__ void __launch_bounds__(SCAN_T) k_scan_block(const int* __restrict__ in, int* __restrict__ out,
                                                       long long n, int* __restrict__ block_tot) {
    long long base = (long long)blockIdx.x * SCAN_B + (long long)threadIdx.x * SCAN_I;
    int v[SCAN_I], s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_I; k++) { v[k] = (base + k < n) ? in[base + k] : 0; s += v[k]; }
    int tot;
    int ex = block_exclusive_scan(s, &tot);
#pragma unroll
    for (int k = 0; k < SCAN_I; k++) { if (base + k < n) out[base + k] = ex; ex += v[k]; }
    if (threadIdx.x == 0) block_tot[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(SCAN_T) k_scan_tops(int* __restrict__ block_tot, long long nb,
                                                      long long* __restrict__ total) {
    __shared__ long long carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (long long b0 = 0; b0 < nb; b0 += SCAN_T) {
        long long b = b0 + threadIdx.x;
        int v = b < nb ? block_tot[b] : 0;
        int tot;
        int ex = block_exclusive_scan(v, &tot);
        long long carry = carry_s;
        if (b < nb) block_tot[b] = (int)(carry + ex);
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = carry_s;
}
__global__ void k_scan_add(int* __restrict__ out, long long n, const int* __restrict__ block_tot,
                           const long long* __restrict__ total) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) out[i] += block_tot[i / SCAN_B];
    if (i == n) out[n] = (int)*total;
}
// out has n+1 entries; block_tmp needs ceil(n / 4096) ints; *total (device) receives the 64-bit sum
void exclusive_scan(const Launch& L, const int* in, int* out, long long n, int* block_tmp, long long* total) {
    long long nb = (n + SCAN_B - 1) / SCAN_B;
    if (nb < 1) nb = 1;
    k_scan_block<<<(unsigned)nb, SCAN_T, 0, L.stream>>>(in, out, n, block_tmp);
    KLAUNCH(L);
    k_scan_tops<<<1, SCAN_T, 0, L.stream>>>(block_tmp, nb, total);
    KLAUNCH(L);
    k_scan_add<<<(unsigned)((n + 1 + 255) / 256), 256, 0, L.stream>>>(out, n, block_tmp, total);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ a2
__global__ void k_place(long long N, const int* __restrict__ cell_id, const int* __restrict__ cell_start,
                        int* __restrict__ cell_fill, int* __restrict__ perm) {
    long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int c = cell_id[i];
    int slot = cell_start[c] + atomicAdd(&cell_fill[c], 1);
    perm[slot] = (int)i;
}
void nbr_place(const Launch& L, long long N, long long ncells, const int* cell_id, const int* cell_start,
               int* cell_fill, int* perm) {
    if (N == 0) return;
    k_place<<<(unsigned)((N + 255) / 256), 256, 0, L.stream>>>(N, cell_id, cell_start, cell_fill, perm);
    KLAUNCH(L);
}
// order inside a cell = ascending caller index (makes the sort stable and the whole build deterministic)
__global__ void k_sort_cells(long long ncells, const int* __restrict__ cell_start, int* __restrict__ perm) {
    long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (c >= ncells) return;
    int b = cell_start[c], e = cell_start[c + 1];
    for (int i = b + 1; i < e; i++) {
        int v = perm[i], k = i - 1;
        while (k >= b && perm[k] > v) { perm[k + 1] = perm[k]; k--; }
        perm[k + 1] = v;
    }
}
void nbr_sort_cells(const Launch& L, long long ncells, const int* cell_start, int* perm) {
    k_sort_cells<<<(unsigned)((ncells + 127) / 128), 128, 0, L.stream>>>(ncells, cell_start, perm);
    KLAUNCH(L);
}
__global__ void k_gather(long long N, long long n_local, const int* __restrict__ perm,
                         const double* __restrict__ pos, const int* __restrict__ types,
                         const signed char* __restrict__ wrap, double* __restrict__ pos_s,
                         int* __restrict__ types_s, signed char* __restrict__ wrap_s, int* __restrict__ inv_perm,
                         float* __restrict__ local_mask, const int* __restrict__ cell_id, int* __restrict__ cell_s) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= N) return;
    int i = perm[a];
    for (int d = 0; d < 3; d++) { pos_s[3 * a + d] = pos[3 * (long long)i + d]; wrap_s[3 * a + d] = wrap[3 * (long long)i + d]; }
    int t = types[i];
    types_s[a] = t;
    inv_perm[i] = (int)a;
    cell_s[a] = cell_id[i];
    local_mask[a] = i < n_local ? 1.0f : 0.0f;
}
void nbr_gather(const Launch& L, long long N, long long n_local, const int* perm, const double* pos,
                const int* types, const signed char* wrap, double* pos_s, int* types_s, signed char* wrap_s,
                int* inv_perm, float* local_mask, const int* cell_id, int* cell_s) {
    if (N == 0) return;
    k_gather<<<(unsigned)((N + 255) / 256), 256, 0, L.stream>>>(N, n_local, perm, pos, types, wrap, pos_s, types_s,
                                                                wrap_s, inv_perm, local_mask, cell_id, cell_s);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ a3
// Visit every candidate (b, shift) of cell-sorted atom a in the fixed stencil order (dz, dy, dx ascending, atoms of a
// cell ascending) and call f(b, code, dx, dy, dz) for those passing  (dx*dx + dy*dy) + dz*dz < cut2  (strict, fp64,
// no contraction);  dx = (x_b + S*L) - x_a with S the image relative to the positions as given.
template <class Fn>
__device__ __forceinline__ void visit_neighbors(long long a, const Grid& g, const NbrSearch& S, Fn f) {
    const double* __restrict__ pos_s = S.pos;
    const signed char* __restrict__ wrap_s = S.wrap;
    const int* __restrict__ cell_start = S.cell_start;
    const double xa = pos_s[3 * a], ya = pos_s[3 * a + 1], za = pos_s[3 * a + 2];
    const int wa0 = wrap_s[3 * a], wa1 = wrap_s[3 * a + 1], wa2 = wrap_s[3 * a + 2];
    int c[3];
    cell_decode(g, S.cell[a], c);
    for (int dz = -1; dz <= 1; dz++) {
        int cz = c[2] + dz, sz = 0;
        if (cz < 0) { if (!g.periodic) continue; cz += g.n[2]; sz = -1; }
        else if (cz >= g.n[2]) { if (!g.periodic) continue; cz -= g.n[2]; sz = 1; }
        for (int dy = -1; dy <= 1; dy++) {
            int cy = c[1] + dy, sy = 0;
            if (cy < 0) { if (!g.periodic) continue; cy += g.n[1]; sy = -1; }
            else if (cy >= g.n[1]) { if (!g.periodic) continue; cy -= g.n[1]; sy = 1; }
            for (int dx = -1; dx <= 1; dx++) {
                int cx = c[0] + dx, sx = 0;
                if (cx < 0) { if (!g.periodic) continue; cx += g.n[0]; sx = -1; }
                else if (cx >= g.n[0]) { if (!g.periodic) continue; cx -= g.n[0]; sx = 1; }
                const int cell = cell_encode(g, cx, cy, cz);
                const int code = (sx + 1) * 9 + (sy + 1) * 3 + (sz + 1);
                const int b0 = cell_start[cell], b1 = cell_start[cell + 1];
                for (int b = b0; b < b1; b++) {
                    if (b == a && code == 13) continue;
                    double Sx = 0.0, Sy = 0.0, Sz = 0.0;
                    if (g.periodic) {
                        Sx = (double)(sx - (int)wrap_s[3 * b] + wa0);
                        Sy = (double)(sy - (int)wrap_s[3 * b + 1] + wa1);
                        Sz = (double)(sz - (int)wrap_s[3 * b + 2] + wa2);
                    }
                    double ex = __dsub_rn(__dadd_rn(pos_s[3 * b], __dmul_rn(Sx, g.box[0])), xa);
                    double ey = __dsub_rn(__dadd_rn(pos_s[3 * b + 1], __dmul_rn(Sy, g.box[1])), ya);
                    double ez = __dsub_rn(__dadd_rn(pos_s[3 * b + 2], __dmul_rn(Sz, g.box[2])), za);
                    double d2 = __dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez));
                    if (d2 < S.cut2) f(b, code, ex, ey, ez);
                }
            }
        }
    }
}
// final row a -> cell-sorted index; cell-sorted neighbour b -> final index (< 0: dropped by the pruning)
__device__ __forceinline__ long long row_old(const NbrSearch& S, long long a) { return S.old_of_new ? S.old_of_new[a] : a; }
__device__ __forceinline__ int idx_new(const NbrSearch& S, int b) { return S.new_of_old ? S.new_of_old[b] : b; }

// x = d / rc as an fp32 pair (x_hi + x_lo, from the fp64 difference the predicate already holds).  The radial basis
// sin(n pi d / rc) turns a relative error eps of d into a phase error n pi x eps: with d computed from the fp32-rounded
// r_e (eps ~ 1e-7) that is 4e-6 at n = 20 -- 60 fp32 ulps, the largest single error of the layer-1 features (DESIGN.md
// B1).  The forward edge kernels take the phase from this pair: sincospi(x_hi), first-order correction with x_lo.
__device__ __forceinline__ float2 phase_pair(double ex, double ey, double ez, double inv_rc) {
    // d = sqrt(d2) without a double-precision square root: fp32 root + one Newton step in fp64 (error ~1e-15 relative)
    const double d2 = ex * ex + ey * ey + ez * ez;
    const float dh = sqrtf((float)d2);
    const double dhd = (double)dh;
    const double d = dhd + fma(-dhd, dhd, d2) * (double)(0.5f / dh);
    const double x = d * inv_rc;
    const float xh = (float)x;
    return make_float2(xh, (float)(x - (double)xh));
}
// one CSR slot (a <- b): fp32 record, image code, search key of the reverse pass, compensated phase
__device__ __forceinline__ void emit_edge(const EdgeOut& o, long long e, int b, int code, double ex, double ey, double ez) {
    o.ej[e] = make_float4((float)ex, (float)ey, (float)ez, __int_as_float(b));
    o.img[e] = (unsigned char)code;
    if (o.key) o.key[e] = (b << 5) | code;        // compact search key of the reverse-edge pass (N < 2^26)
    if (o.xph) o.xph[e] = phase_pair(ex, ey, ez, o.inv_rc);
}
// dummy slots: sender index ~a (negative), |r| = rc; every kernel gives them exactly zero weight
__device__ __forceinline__ void emit_padding(const EdgeOut& o, long long e, long long e1, long long a) {
    for (; e < e1; e++) {
        o.ej[e] = make_float4(o.rc, 0.0f, 0.0f, __int_as_float(~(int)a));
        o.img[e] = 255;
        if (o.key) o.key[e] = -1;
        if (o.xph) o.xph[e] = make_float2(1.0f, 0.0f);
    }
}

// rows: final order; n_rows_p (device, may be null = N): rows >= *n_rows_p are unreached atoms and stay empty
__global__ void __launch_bounds__(128) k_count(long long N, Grid g, NbrSearch S, const int* __restrict__ n_rows_p,
                                               int* __restrict__ row_cnt, unsigned long long* __restrict__ real_total) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    int cnt = 0;
    if (a < N) {
        if (n_rows_p == nullptr || a < *n_rows_p)
            visit_neighbors(row_old(S, a), g, S, [&](int b, int, double, double, double) { cnt += idx_new(S, b) >= 0; });
        // rows are padded to a multiple of 8 slots with zero-weight dummy edges, so that an 8-edge group of the
        // tensor-core edge kernels never straddles two rows (branch-free inner loops)
        row_cnt[a] = (cnt + ROW_PAD - 1) & ~(ROW_PAD - 1);
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(real_total, (unsigned long long)cnt);
}
void nbr_count(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, int* row_cnt,
               unsigned long long* real_total) {
    if (N == 0) return;
    k_count<<<(unsigned)((N + 127) / 128), 128, 0, L.stream>>>(N, g, S, n_rows_p, row_cnt, real_total);
    KLAUNCH(L);
}

__global__ void __launch_bounds__(128) k_fill(long long N, Grid g, NbrSearch S, const int* __restrict__ n_rows_p,
                                              const int* __restrict__ row_ptr, long long cap_edges, EdgeOut o,
                                              int* __restrict__ flags) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= N) return;
    long long e = row_ptr[a];
    if ((long long)row_ptr[a + 1] > cap_edges) { atomicOr(flags, FLAG_EDGE_OVERFLOW); return; }
    if (n_rows_p == nullptr || a < *n_rows_p)
        visit_neighbors(row_old(S, a), g, S, [&](int b, int code, double ex, double ey, double ez) {
            const int bn = idx_new(S, b);
            if (bn < 0) return;
            emit_edge(o, e, bn, code, ex, ey, ez);
            e++;
        });
    emit_padding(o, e, row_ptr[a + 1], a);
}
void nbr_fill(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, const int* row_ptr,
              long long cap_edges, EdgeOut o, int* flags) {
    if (N == 0) return;
    if (N >= (1ll << 26)) o.key = nullptr;
    k_fill<<<(unsigned)((N + 127) / 128), 128, 0, L.stream>>>(N, g, S, n_rows_p, row_ptr, cap_edges, o, flags);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ T-hop pruning
// "T rounds of pseudo-messages from local atoms; atoms never reached are dropped" (Fig. 1e): level 0 = local atoms,
// level t = atoms with a neighbour of level t - 1 (breadth-first over the cutoff graph; with a Verlet skin over the
// list-cutoff graph, a superset, so the levels are lower bounds for every step the list serves).  Cell-sorted indices.
__global__ void k_level_init(long long N, const float* __restrict__ local_mask, unsigned char* __restrict__ level) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a < N) level[a] = local_mask[a] != 0.0f ? 0 : LEVEL_NONE;
}
__global__ void __launch_bounds__(128) k_level_round(long long N, Grid g, NbrSearch S, unsigned char* __restrict__ level, int t) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= N || level[a] != LEVEL_NONE) return;
    bool hit = false;
    // (a level written in this round equals t, never t - 1: reading while others write is harmless)
    visit_neighbors(a, g, S, [&](int b, int, double, double, double) { hit |= level[b] == t - 1; });
    if (hit) level[a] = (unsigned char)t;
}
void nbr_levels(const Launch& L, long long N, Grid g, const NbrSearch& S, const float* local_mask, unsigned char* level, int T) {
    if (N == 0) return;
    k_level_init<<<(unsigned)((N + 255) / 256), 256, 0, L.stream>>>(N, local_mask, level);
    KLAUNCH(L);
    for (int t = 1; t <= T; t++) {
        k_level_round<<<(unsigned)((N + 127) / 128), 128, 0, L.stream>>>(N, g, S, level, t);
        KLAUNCH(L);
    }
}
// Stable partition of the cell-sorted atoms by level (buckets 0..T, then the unreached): final index = atoms of lower
// levels first, cell order kept inside a level.  Every layer's receivers are then a PREFIX of the atom arrays and the
// kernels of the model run unchanged on a shorter N.  Three passes: per-block histogram, bucket-major offsets, placement.
constexpr int LVB = 256;                                // atoms per block
__device__ __forceinline__ int level_bucket(unsigned char lv, int T) { return lv <= T ? lv : T + 1; }
__global__ void __launch_bounds__(LVB) k_level_hist(long long N, const unsigned char* __restrict__ level, int T, int* __restrict__ hist) {
    __shared__ int h[PAINN_MAX_T + 2];
    if (threadIdx.x < T + 2) h[threadIdx.x] = 0;
    __syncthreads();
    long long a = blockIdx.x * (long long)LVB + threadIdx.x;
    if (a < N) atomicAdd(&h[level_bucket(level[a], T)], 1);
    __syncthreads();
    if (threadIdx.x < T + 2) hist[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = h[threadIdx.x];   // bucket-major
}
// exclusive scan over the bucket-major table (one block); prefix[k] = atoms with bucket < k (k = 0..T+2)
__global__ void __launch_bounds__(SCAN_T) k_level_offsets(int* __restrict__ hist, long long n, int nb, int T,
                                                          long long* __restrict__ prefix) {
    __shared__ long long carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (long long b0 = 0; b0 < n; b0 += SCAN_T) {
        long long b = b0 + threadIdx.x;
        int v = b < n ? hist[b] : 0;
        int tot;
        int ex = block_exclusive_scan(v, &tot);
        long long carry = carry_s;
        if (b < n) {
            hist[b] = (int)(carry + ex);
            if (b % nb == 0) prefix[b / nb] = carry + ex;
        }
        __syncthreads();
        if (threadIdx.x == 0) carry_s = carry + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) prefix[T + 2] = carry_s;
}
__global__ void __launch_bounds__(LVB) k_level_place(long long N, const unsigned char* __restrict__ level, int T,
                                                     const int* __restrict__ base, long long n_reach_src_unused,
                                                     const long long* __restrict__ prefix, int* __restrict__ new_of_old,
                                                     int* __restrict__ old_of_new) {
    __shared__ int wcnt[LVB / 32][PAINN_MAX_T + 2];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    long long a = blockIdx.x * (long long)LVB + threadIdx.x;
    const int k = a < N ? level_bucket(level[a], T) : -1;
    for (int i = lane; i < T + 2; i += 32) wcnt[warp][i] = 0;
    __syncwarp();
    const unsigned peers = __match_any_sync(0xffffffffu, k);
    const int rank_in_warp = __popc(peers & ((1u << lane) - 1u));
    if (k >= 0 && rank_in_warp == 0) wcnt[warp][k] = __popc(peers);
    __syncthreads();
    if (k >= 0) {
        int before = 0;
        for (int w = 0; w < warp; w++) before += wcnt[w][k];
        const int idx = base[(size_t)k * gridDim.x + blockIdx.x] + before + rank_in_warp;
        old_of_new[idx] = (int)a;
        new_of_old[a] = k <= T ? idx : -1 - idx;      // unreached atoms keep a slot at the end (outputs stay defined), flagged < 0
    }
    (void)n_reach_src_unused; (void)prefix;
}
// hist: scratch of (T + 2) * ceil(N / 256) ints; prefix: T + 3 long long (device)
void nbr_level_sort(const Launch& L, long long N, const unsigned char* level, int T, int* hist, long long* prefix,
                    int* new_of_old, int* old_of_new) {
    if (N == 0) return;
    const int nb = (int)((N + LVB - 1) / LVB);
    k_level_hist<<<nb, LVB, 0, L.stream>>>(N, level, T, hist);
    KLAUNCH(L);
    k_level_offsets<<<1, SCAN_T, 0, L.stream>>>(hist, (long long)nb * (T + 2), nb, T, prefix);
    KLAUNCH(L);
    k_level_place<<<nb, LVB, 0, L.stream>>>(N, level, T, hist, 0, prefix, new_of_old, old_of_new);
    KLAUNCH(L);
}
// per-atom arrays from the cell-sorted order into the final (level-major) order
__global__ void k_regather(long long N, const int* __restrict__ old_of_new, const double* __restrict__ posC,
                           const int* __restrict__ typesC, const signed char* __restrict__ wrapC, const int* __restrict__ permC,
                           const float* __restrict__ localC, double* __restrict__ pos_s, int* __restrict__ types_s,
                           signed char* __restrict__ wrap_s, int* __restrict__ perm, int* __restrict__ inv_perm,
                           float* __restrict__ local_mask) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= N) return;
    const int o = old_of_new[a];
    for (int d = 0; d < 3; d++) { pos_s[3 * a + d] = posC[3 * (long long)o + d]; wrap_s[3 * a + d] = wrapC[3 * (long long)o + d]; }
    types_s[a] = typesC[o];
    const int i = permC[o];
    perm[a] = i;
    inv_perm[i] = (int)a;
    local_mask[a] = localC[o];
}
void nbr_regather(const Launch& L, long long N, const int* old_of_new, const double* posC, const int* typesC,
                  const signed char* wrapC, const int* permC, const float* localC, double* pos_s, int* types_s,
                  signed char* wrap_s, int* perm, int* inv_perm, float* local_mask) {
    if (N == 0) return;
    k_regather<<<(unsigned)((N + 255) / 256), 256, 0, L.stream>>>(N, old_of_new, posC, typesC, wrapC, permC, localC, pos_s, types_s,
                                                                  wrap_s, perm, inv_perm, local_mask);
    KLAUNCH(L);
}

// ------------------------------------------------------------------------------------------------ Verlet skin
// Superset list at rc + skin, final indices, unpadded rows: sup_j, sup_code.  While no atom has moved by more than
// skin / 2 since it was built, every pair within rc is in it, and a step only re-filters it (the per-step "drop edges
// longer than the cutoff" of PAPER.md:68) instead of binning, sorting and scanning 27 cells.
__global__ void __launch_bounds__(128) k_sup_count(long long N, Grid g, NbrSearch S, const int* __restrict__ n_rows_p,
                                                   int* __restrict__ row_cnt, unsigned long long* __restrict__ padded_total) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    int cnt = 0;
    if (a < N) {
        if (n_rows_p == nullptr || a < *n_rows_p)
            visit_neighbors(row_old(S, a), g, S, [&](int b, int, double, double, double) { cnt += idx_new(S, b) >= 0; });
        row_cnt[a] = cnt;
        cnt = (cnt + ROW_PAD - 1) & ~(ROW_PAD - 1);       // bound of the padded row of any step this list serves
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0 && cnt) atomicAdd(padded_total, (unsigned long long)cnt);
}
__global__ void __launch_bounds__(128) k_sup_fill(long long N, Grid g, NbrSearch S, const int* __restrict__ n_rows_p,
                                                  const int* __restrict__ sup_ptr, int* __restrict__ sup_j,
                                                  unsigned char* __restrict__ sup_code) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= N || (n_rows_p != nullptr && a >= *n_rows_p)) return;
    long long e = sup_ptr[a];
    visit_neighbors(row_old(S, a), g, S, [&](int b, int code, double, double, double) {
        const int bn = idx_new(S, b);
        if (bn < 0) return;
        sup_j[e] = bn;
        sup_code[e] = (unsigned char)code;
        e++;
    });
}
void nbr_sup_count(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, int* row_cnt,
                   unsigned long long* padded_total) {
    if (N == 0) return;
    k_sup_count<<<(unsigned)((N + 127) / 128), 128, 0, L.stream>>>(N, g, S, n_rows_p, row_cnt, padded_total);
    KLAUNCH(L);
}
void nbr_sup_fill(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, const int* sup_ptr, int* sup_j,
                  unsigned char* sup_code) {
    if (N == 0) return;
    k_sup_fill<<<(unsigned)((N + 127) / 128), 128, 0, L.stream>>>(N, g, S, n_rows_p, sup_ptr, sup_j, sup_code);
    KLAUNCH(L);
}
// One warp per row: lanes take the candidates of the superset row 32 at a time (coalesced reads of sup_j / sup_code, the
// position gathers of a batch in flight together) and test them with the SAME fp64 expression as visit_neighbors on the
// current positions as given (pos_s / wrap_s in final order, refreshed by k_reuse_prep): identical edge sets, bit for
// bit.  Kept candidates are compacted in candidate order (ballot + prefix popcount), so count and fill agree.
struct SupCand {
    int b, code;
    double ex, ey, ez;
    bool keep;
};
__device__ __forceinline__ SupCand test_candidate(int x, int x1, long long a, const Grid& g, const double* __restrict__ pos_s,
                                                  const signed char* __restrict__ wrap_s, const int* __restrict__ sup_j,
                                                  const unsigned char* __restrict__ sup_code, double xa, double ya, double za,
                                                  int wa0, int wa1, int wa2) {
    SupCand c;
    c.keep = false;
    c.b = 0; c.code = 13; c.ex = c.ey = c.ez = 0.0;
    if (x >= x1) return c;
    const int b = sup_j[x], code = sup_code[x];
    double Sx = 0.0, Sy = 0.0, Sz = 0.0;
    if (g.periodic) {
        Sx = (double)(code / 9 - 1 - (int)wrap_s[3 * b] + wa0);
        Sy = (double)((code / 3) % 3 - 1 - (int)wrap_s[3 * b + 1] + wa1);
        Sz = (double)(code % 3 - 1 - (int)wrap_s[3 * b + 2] + wa2);
    }
    c.ex = __dsub_rn(__dadd_rn(pos_s[3 * b], __dmul_rn(Sx, g.box[0])), xa);
    c.ey = __dsub_rn(__dadd_rn(pos_s[3 * b + 1], __dmul_rn(Sy, g.box[1])), ya);
    c.ez = __dsub_rn(__dadd_rn(pos_s[3 * b + 2], __dmul_rn(Sz, g.box[2])), za);
    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(c.ex, c.ex), __dmul_rn(c.ey, c.ey)), __dmul_rn(c.ez, c.ez));
    c.keep = d2 < g.rc2;
    c.b = b; c.code = code;
    (void)a;
    return c;
}
__global__ void __launch_bounds__(256) k_refilter_count(long long N, Grid g, const double* __restrict__ pos_s,
                                                        const signed char* __restrict__ wrap_s, const int* __restrict__ sup_ptr,
                                                        const int* __restrict__ sup_j, const unsigned char* __restrict__ sup_code,
                                                        int* __restrict__ row_cnt, unsigned long long* __restrict__ real_total) {
    const long long a = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (a >= N) return;
    const double xa = pos_s[3 * a], ya = pos_s[3 * a + 1], za = pos_s[3 * a + 2];
    const int wa0 = wrap_s[3 * a], wa1 = wrap_s[3 * a + 1], wa2 = wrap_s[3 * a + 2];
    const int x0 = sup_ptr[a], x1 = sup_ptr[a + 1];
    int cnt = 0;
    for (int x = x0; x < x1; x += 32) {
        const SupCand c = test_candidate(x + lane, x1, a, g, pos_s, wrap_s, sup_j, sup_code, xa, ya, za, wa0, wa1, wa2);
        cnt += __popc(__ballot_sync(0xffffffffu, c.keep));
    }
    if (lane == 0) {
        row_cnt[a] = (cnt + ROW_PAD - 1) & ~(ROW_PAD - 1);
        if (cnt) atomicAdd(real_total, (unsigned long long)cnt);
    }
}
__global__ void __launch_bounds__(256) k_refilter_fill(long long N, Grid g, const double* __restrict__ pos_s,
                                                       const signed char* __restrict__ wrap_s, const int* __restrict__ sup_ptr,
                                                       const int* __restrict__ sup_j, const unsigned char* __restrict__ sup_code,
                                                       const int* __restrict__ row_ptr, long long cap_edges, EdgeOut o,
                                                       int* __restrict__ flags) {
    const long long a = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (a >= N) return;
    long long e = row_ptr[a];
    const long long e1 = row_ptr[a + 1];
    if (e1 > cap_edges) { if (lane == 0) atomicOr(flags, FLAG_EDGE_OVERFLOW); return; }   // (cannot happen: bound reserved at build)
    const double xa = pos_s[3 * a], ya = pos_s[3 * a + 1], za = pos_s[3 * a + 2];
    const int wa0 = wrap_s[3 * a], wa1 = wrap_s[3 * a + 1], wa2 = wrap_s[3 * a + 2];
    const int x0 = sup_ptr[a], x1 = sup_ptr[a + 1];
    for (int x = x0; x < x1; x += 32) {
        const SupCand c = test_candidate(x + lane, x1, a, g, pos_s, wrap_s, sup_j, sup_code, xa, ya, za, wa0, wa1, wa2);
        const unsigned m = __ballot_sync(0xffffffffu, c.keep);
        if (c.keep) emit_edge(o, e + __popc(m & ((1u << lane) - 1u)), c.b, c.code, c.ex, c.ey, c.ez);
        e += __popc(m);
    }
    // dummy slots of the padded row
    for (long long k = e + lane; k < e1; k += 32) emit_padding(o, k, k + 1, a);
}
void nbr_refilter_count(const Launch& L, long long N, Grid g, const double* pos_s, const signed char* wrap_s, const int* sup_ptr,
                        const int* sup_j, const unsigned char* sup_code, int* row_cnt, unsigned long long* real_total) {
    if (N == 0) return;
    k_refilter_count<<<(unsigned)((N * 32 + 255) / 256), 256, 0, L.stream>>>(N, g, pos_s, wrap_s, sup_ptr, sup_j, sup_code, row_cnt, real_total);
    KLAUNCH(L);
}
void nbr_refilter_fill(const Launch& L, long long N, Grid g, const double* pos_s, const signed char* wrap_s, const int* sup_ptr,
                       const int* sup_j, const unsigned char* sup_code, const int* row_ptr, long long cap_edges, EdgeOut o, int* flags) {
    if (N == 0) return;
    if (N >= (1ll << 26)) o.key = nullptr;
    k_refilter_fill<<<(unsigned)((N * 32 + 255) / 256), 256, 0, L.stream>>>(N, g, pos_s, wrap_s, sup_ptr, sup_j, sup_code, row_ptr, cap_edges, o, flags);
    KLAUNCH(L);
}
// A step that reuses the list: current positions into the final order, wrap counts continued from the build
// (wrap_now = wrap_build + whole box lengths the as-given coordinate jumped by since), and the validity test: no atom
// further than skin / 2 from where it was at the build (minimum image), same species.  Sets FLAG_REBUILD otherwise.
__global__ void k_reuse_prep(long long N, const int* __restrict__ perm, const double* __restrict__ pos, const int* __restrict__ types,
                             const double* __restrict__ pos_ref_s, const signed char* __restrict__ wrap_ref_s,
                             const int* __restrict__ types_s, Grid g, double half_skin2, double* __restrict__ pos_s,
                             signed char* __restrict__ wrap_s, int* __restrict__ flags) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= N) return;
    const long long i = perm[a];
    int bad = 0;
    double d2 = 0.0;
    for (int d = 0; d < 3; d++) {
        const double x = pos[3 * i + d];
        if (!isfinite(x)) bad |= FLAG_NONFINITE;
        double dx = x - pos_ref_s[3 * a + d], m = 0.0;
        if (g.periodic) { m = rint(dx / g.box[d]); dx -= m * g.box[d]; }
        if (fabs(m) > 100.0) { bad |= FLAG_REBUILD; m = 0.0; }
        d2 += dx * dx;
        pos_s[3 * a + d] = x;
        wrap_s[3 * a + d] = (signed char)((int)wrap_ref_s[3 * a + d] + (int)m);
    }
    if (!(d2 <= half_skin2) || types[i] != types_s[a]) bad |= FLAG_REBUILD;
    if (bad) atomicOr(flags, bad);
}
void nbr_reuse_prep(const Launch& L, long long N, const int* perm, const double* pos, const int* types, const double* pos_ref_s,
                    const signed char* wrap_ref_s, const int* types_s, Grid g, double half_skin2, double* pos_s, signed char* wrap_s,
                    int* flags) {
    if (N == 0) return;
    k_reuse_prep<<<(unsigned)((N + 255) / 256), 256, 0, L.stream>>>(N, perm, pos, types, pos_ref_s, wrap_ref_s, types_s, g, half_skin2,
                                                                    pos_s, wrap_s, flags);
    KLAUNCH(L);
}

// reverse-edge index: for slot e = (a <- b, code) find the slot of (b <- a, 26 - code) in row b
__global__ void k_reverse(long long N, const int* __restrict__ row_ptr, const float4* __restrict__ ej,
                          const unsigned char* __restrict__ img, int* __restrict__ rev, int* __restrict__ miss) {
    // one warp per row a
    long long a = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (a >= N) return;
    for (int e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) {
        int b = __float_as_int(ej[e].w);
        if (b < 0) { rev[e] = e; continue; }          // dummy slot: its own reverse (G[rev] - G = 0)
        int want = 26 - (int)img[e];
        int r = -1;
        for (int x = row_ptr[b]; x < row_ptr[b + 1]; x++)
            if (__float_as_int(ej[x].w) == (int)a && (int)img[x] == want) { r = x; break; }
        if (r < 0) { r = e; atomicAdd(miss, 1); }     // see k_reverse_keys
        rev[e] = r;
    }
}
// The same search on the compact keys (sender << 5 | image code) written by k_fill: rows start at multiples of 8 slots,
// so 8 candidates are two aligned 16-byte loads (the float4 records cost a 32-byte sector per two candidates: 4x the
// L2 traffic, which is what bounds this pass).
// A pair whose d^2 sits within an ulp of rc^2 can pass the fp64 predicate in one direction only when an image shift is
// involved (fl(fl(x_b + S L) - x_a) is not the exact negation of fl(fl(x_a - S L) - x_b)): such a slot has no reverse.
// It maps to itself (G[rev] - G = 0: no force from an edge whose weight fc(rc) is zero anyway) and is counted in *miss.
__global__ void k_reverse_keys(long long N, const int* __restrict__ row_ptr, const int* __restrict__ key,
                               int* __restrict__ rev, int* __restrict__ miss) {
    long long a = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (a >= N) return;
    for (int e = row_ptr[a] + lane; e < row_ptr[a + 1]; e += 32) {
        const int k = key[e];
        if (k < 0) { rev[e] = e; continue; }          // dummy slot: its own reverse (G[rev] - G = 0)
        const int b = k >> 5;
        const int want = ((int)a << 5) | (26 - (k & 31));
        int r = -1;
        const int x1 = row_ptr[b + 1];
        for (int x = row_ptr[b]; x < x1 && r < 0; x += 8) {
            const int4 q0 = *(const int4*)(key + x), q1 = *(const int4*)(key + x + 4);
            if (q0.x == want) r = x;
            else if (q0.y == want) r = x + 1;
            else if (q0.z == want) r = x + 2;
            else if (q0.w == want) r = x + 3;
            else if (q1.x == want) r = x + 4;
            else if (q1.y == want) r = x + 5;
            else if (q1.z == want) r = x + 6;
            else if (q1.w == want) r = x + 7;
        }
        if (r < 0) { r = e; atomicAdd(miss, 1); }
        rev[e] = r;
    }
}
// key: the array nbr_fill wrote (nullptr, or N >= 2^26: search the float4 records)
void nbr_reverse(const Launch& L, long long N, const int* row_ptr, const float4* ej, const unsigned char* img,
                 const int* key, int* rev, int* miss) {
    if (N == 0) return;
    if (key && N < (1ll << 26)) {
        k_reverse_keys<<<(unsigned)((N * 32 + 255) / 256), 256, 0, L.stream>>>(N, row_ptr, key, rev, miss);
        KLAUNCH(L);
        return;
    }
    k_reverse<<<(unsigned)((N * 32 + 255) / 256), 256, 0, L.stream>>>(N, row_ptr, ej, img, rev, miss);
    KLAUNCH(L);
}

// export in caller indices with images relative to the positions as given
__global__ void k_export(long long N, const int* __restrict__ row_ptr, const float4* __restrict__ ej,
                         const unsigned char* __restrict__ img, const int* __restrict__ perm,
                         const signed char* __restrict__ wrap_s, int* __restrict__ out_i, int* __restrict__ out_j,
                         signed char* __restrict__ out_img) {
    long long a = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (a >= N) return;
    for (int e = row_ptr[a]; e < row_ptr[a + 1]; e++) {
        int b = __float_as_int(ej[e].w);
        if (b < 0) { out_i[e] = -1; out_j[e] = -1; continue; }   // dummy slot (compacted away by the host)
        int code = img[e];
        int s[3] = {code / 9 - 1, (code / 3) % 3 - 1, code % 3 - 1};
        out_i[e] = perm[a];
        out_j[e] = perm[b];
        for (int d = 0; d < 3; d++)
            out_img[3 * (long long)e + d] = (signed char)(s[d] - (int)wrap_s[3 * (long long)b + d] + (int)wrap_s[3 * a + d]);
    }
}
void nbr_export(const Launch& L, long long N, const int* row_ptr, const float4* ej, const unsigned char* img,
                const int* perm, const signed char* wrap_s, int* out_i, int* out_j, signed char* out_img) {
    if (N == 0) return;
    k_export<<<(unsigned)((N + 127) / 128), 128, 0, L.stream>>>(N, row_ptr, ej, img, perm, wrap_s, out_i, out_j,
                                                                out_img);
    KLAUNCH(L);
}

}  // namespace painn
