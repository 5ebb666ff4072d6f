// common.cuh -- shared declarations of the PaiNN hot-path kernels (internal to the CUDA path).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <unordered_map>
#include <utility>
#include <vector>

#define PAINN_MAX_T 8
#define PAINN_MAX_K 32
#define ROW_PAD 8          // CSR rows are padded to a multiple of ROW_PAD slots (dummy edges: sender index < 0)

namespace painn {

// Cell grid of one call (host-computed, passed by value to the neighbour kernels).
struct Grid {
    double origin[3];   // ghost mode: bounding-box min; periodic mode: 0
    double box[3];      // periodic box lengths (periodic mode)
    double inv_side[3]; // 1 / cell side
    int n[3];           // cells per dimension
    int periodic;       // 1: periodic (n_ghost == 0), 0: open boundaries
    double rc2;         // cutoff^2
    int strip;          // cell order: y is cut into strips of this many cells; inside a strip z, y, x (x fastest).
                        // strip >= n[1] is the plain (z, y, x) order.  DESIGN.md section 6 (L2 working set of the gathers)
};

// Linear index of cell (cx, cy, cz) and its inverse.  With strips of B cells in y the atoms of three consecutive z planes of
// a strip are 3 n[0] B cells apart instead of 3 n[0] n[1]: the rows the edge kernels gather stay L2-resident between planes.
__host__ __device__ __forceinline__ int cell_encode(const Grid& g, int cx, int cy, int cz) {
    const int B = g.strip, sy = cy / B, y0 = sy * B;
    const int w = g.n[1] - y0 < B ? g.n[1] - y0 : B;
    return (y0 * g.n[2] + cz * w + (cy - y0)) * g.n[0] + cx;
}
__host__ __device__ __forceinline__ void cell_decode(const Grid& g, int cell, int (&c)[3]) {
    const int B = g.strip, per_strip = B * g.n[2] * g.n[0];
    const int sy = cell / per_strip, y0 = sy * B;
    const int w = g.n[1] - y0 < B ? g.n[1] - y0 : B;
    int rem = cell - sy * per_strip;
    c[0] = rem % g.n[0]; rem /= g.n[0];
    c[1] = y0 + rem % w;
    c[2] = rem / w;
}

// error flags written by the device (bit mask in flags[0])
enum { FLAG_TYPE_RANGE = 1, FLAG_NONFINITE = 2, FLAG_EDGE_OVERFLOW = 4, FLAG_OWNER_RANGE = 8, FLAG_REBUILD = 16 };
#define LEVEL_NONE 255     // hop level of an atom no local atom reaches within T hops

// Cell-sorted search structure of one neighbour build and the optional relabelling into the final atom order.
struct NbrSearch {
    const double* pos;          // [N][3] positions as given, cell-sorted
    const signed char* wrap;    // [N][3] wrap counts
    const int* cell;            // [N] cell of each atom
    const int* cell_start;      // [n_cells + 1]
    const int* new_of_old;      // final index of cell-sorted atom b (< 0: dropped), or nullptr = identity
    const int* old_of_new;      // cell-sorted index of final row a, or nullptr = identity
    double cut2;                // (list cutoff)^2: rc^2, or (rc + skin)^2 for the superset list
};
// Where a CSR slot is written (nbr.cu::emit_edge)
struct EdgeOut {
    float4* ej;                 // (r_e fp32, sender index bits)
    unsigned char* img;         // image code, 255 = padding slot
    int* key;                   // (sender << 5 | code) search key of the reverse pass, or nullptr
    float2* xph;                // compensated phase d / rc as (hi, lo), or nullptr
    double inv_rc;
    float rc;
};

struct LayerW {
    const float *Wm1, *bm1, *Wm2, *bm2, *Wf, *bf, *UV, *Wu1, *bu1, *Wu2, *bu2;   // [out x in] row-major
    const float *Wm1T, *Wm2T, *UVT, *Wu1T, *Wu2T;                                // transposes [in x out]
};

// Tensor-core operands of the GEMM weights, cut once at mlp_create and owned by the model (gemm.cu / gemm_tc.cu).
struct ExactW {
    int N, K;
    void* planes;          // device [K / 128][3][N][128] integer-valued fp16 slices
    float* cs;             // device [K / 128][N] column scales
};
struct GemmRegistry {
    std::unordered_map<const float*, std::pair<const float*, const float*>> split;   // W -> (hi, lo) TF32 planes
    std::unordered_map<const float*, ExactW> exact;                                   // W -> exact slices
};

struct Launch {            // per-call launch context: everything a kernel launcher may depend on besides its arguments
    cudaStream_t stream;
    long long* counter;    // kernels launched
    const GemmRegistry* reg = nullptr;
    int gemm_path = 0;     // 0: adjoint GEMMs (tcgen05 3xTF32 when the shape is covered), 1: forward GEMMs (exact accumulation)
    int fwd_exact = 1;     // forward GEMMs: 1 exact integer-slice tcgen05 kernel when covered, 0 fp32 FFMA kernel
    int* used_tc = nullptr;   // set to 1 when a tensor-core GEMM kernel ran (test hook of mlp_debug_gemm)
    int apu_fwd = 12, apu_bwd = 16;   // consecutive cell-sorted atoms per work unit of the tensor-core edge kernels (1..31)
};

// ---- neighbour build (nbr.cu) ----
void nbr_bin(const Launch& L, const double* pos, const int* types, long long N, int n_species, Grid g,
             int* cell_id, signed char* wrap, int* cell_count, int* flags, long long n_local, const int* ghost_owner);
void nbr_bbox(const Launch& L, const double* pos, long long N, double* bbox6);
void exclusive_scan(const Launch& L, const int* in, int* out, long long n, int* block_tmp, long long* total);
void nbr_place(const Launch& L, long long N, long long ncells, const int* cell_id, const int* cell_start,
               int* cell_fill, int* perm);
void nbr_sort_cells(const Launch& L, long long ncells, const int* cell_start, int* perm);
void nbr_gather(const Launch& L, long long N, long long n_local, const int* perm, const double* pos,
                const int* types, const signed char* wrap, double* pos_s, int* types_s, signed char* wrap_s,
                int* inv_perm, float* local_mask, const int* cell_id, int* cell_s);
void nbr_count(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, int* row_cnt,
               unsigned long long* real_total);
void nbr_fill(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, const int* row_ptr,
              long long cap_edges, EdgeOut o, int* flags);
void nbr_levels(const Launch& L, long long N, Grid g, const NbrSearch& S, const float* local_mask, unsigned char* level, int T);
void nbr_level_sort(const Launch& L, long long N, const unsigned char* level, int T, int* hist, long long* prefix,
                    int* new_of_old, int* old_of_new);
void nbr_regather(const Launch& L, long long N, const int* old_of_new, const double* posC, const int* typesC,
                  const signed char* wrapC, const int* permC, const float* localC, double* pos_s, int* types_s,
                  signed char* wrap_s, int* perm, int* inv_perm, float* local_mask);
void nbr_sup_count(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, int* row_cnt,
                   unsigned long long* padded_total);
void nbr_sup_fill(const Launch& L, long long N, Grid g, const NbrSearch& S, const int* n_rows_p, const int* sup_ptr, int* sup_j,
                  unsigned char* sup_code);
void nbr_refilter_count(const Launch& L, long long N, Grid g, const double* pos_s, const signed char* wrap_s, const int* sup_ptr,
                        const int* sup_j, const unsigned char* sup_code, int* row_cnt, unsigned long long* real_total);
void nbr_refilter_fill(const Launch& L, long long N, Grid g, const double* pos_s, const signed char* wrap_s, const int* sup_ptr,
                       const int* sup_j, const unsigned char* sup_code, const int* row_ptr, long long cap_edges, EdgeOut o, int* flags);
void nbr_reuse_prep(const Launch& L, long long N, const int* perm, const double* pos, const int* types, const double* pos_ref_s,
                    const signed char* wrap_ref_s, const int* types_s, Grid g, double half_skin2, double* pos_s, signed char* wrap_s,
                    int* flags);
void nbr_reverse(const Launch& L, long long N, const int* row_ptr, const float4* ej, const unsigned char* img,
                 const int* key, int* rev, int* miss);
void nbr_export(const Launch& L, long long N, const int* row_ptr, const float4* ej, const unsigned char* img,
                const int* perm, const signed char* wrap_s, int* out_i, int* out_j, signed char* out_img);

void gemm_register_split(GemmRegistry& reg, const float* W, const float* hi, const float* lo);
// exact integer-slice tensor-core path of the forward GEMMs (gemm_tc.cu): slices of W [N x K] are cut at create
void gemm_register_exact(GemmRegistry& reg, const float* Wdev, const float* Whost, int N, int K);
void gemm_registry_free(GemmRegistry& reg);
bool gemm_nt_exact(const Launch& L, const float* A, int lda, const float* W, float* C, int ldc, long long M, int N, int K,
                   const float* bias, bool accumulate, bool act_a);
// ---- dense node GEMM (gemm.cu):  C[M x N] (+)= A[M x K] . B[N x K]^T + bias ----
void gemm_nt(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
             int N, int K, const float* bias, bool accumulate);

void gemm_nt_act(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
                 int N, int K, const float* bias, bool accumulate, bool act_a);
void gemm_nt_resid(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
                   int N, int K, const float* resid);
bool gemm_act_supported(int N, int K);
void gemm_nt_dsilu(const Launch& L, const float* A, int lda, const float* B, int ldb, float* C, int ldc, long long M,
                   int N, int K, const float* pre);

// ---- model kernels (painn_fwd.cu / painn_bwd.cu) ----
void embed(const Launch& L, long long N, int F, const int* types_s, const float* Emb, float* s0, float* v0);
void silu_fwd(const Launch& L, long long n, const float* x, float* y);
void mul_dsilu(const Launch& L, long long n, const float* pre, float* g);   // g *= SiLU'(pre)
void message_fwd(const Launch& L, long long N, int F, int K, float rc, const int* row_ptr, const float4* ej,
                 const float* s, const float* v, const float* phi, const float* Wf, const float* bf, float* sn,
                 float* v1);
void update_mid(const Launch& L, long long N, int F, float eps, const float* pq, float* sn);
void update_out(const Launch& L, long long N, int F, const float* sn, const float* v1, const float* pq,
                const float* a, float* s_out, float* v_out);
void readout(const Launch& L, long long N, int R, const float* rpre, const float* wr2, const float* br2,
             const float* local_mask, float* rb, float* e_atom, double* e_partial, int* n_partial);
void update_bwd1(const Launch& L, long long N, int F, const float* sb, const float* vb, const float* pq,
                 const float* a, float* ab, float* pqb);
void update_bwd2(const Launch& L, long long N, int F, const float* sb, const float* vb, const float* snb,
                 const float* sn, const float* pq, float* pqb, float* s1b, float* v1b);
void message_bwd(const Launch& L, long long N, int F, int K, float rc, const int* row_ptr, const float4* ej,
                 const float* s1b, const float* v1b, const float* phi, const float* v_in, const float* Wf,
                 const float* bf, float* phib, float* vb_out, float4* G, bool first);
void force_final(const Launch& L, long long N, long long n_local, const int* row_ptr, const float4* ej,
                 const int* rev, const float4* G, const int* perm, const int* ghost_owner, double* forces,
                 double* w_partial, int* n_partial);
void reduce_final(const Launch& L, const double* e_partial, int n_e, const double* w_partial, int n_w,
                  double* scratch, double* energy, double* virial);
void unpermute_state(const Launch& L, long long N, int F, const int* perm, const float* s, const float* v,
                     float* out);

// ---- tensor-core edge kernels (edge_v3.cu), F = 128: per-edge filter on tcgen05, software-pipelined gathers ----
void make_gather_rows(const Launch& L, long long N, const float* phi, const float* v, float* Q4, float* Q1, bool has_v);
void make_gather_rows_bwd(const Launch& L, long long N, const float* s1b, const float* v1b, float* Gb);
bool message_fwd_v3(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* s,
                    const float* v, const float* Q4, const float* Q1, const void* A_rows, float* sn, float* v1,
                    bool has_v, const int* types_s, const float* tab, int n_tab, const float2* xph);
bool message_bwd_v3(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* Gb,
                    const float* phi, const float* v_in, const float* v1b, const void* A_rows, float* phib,
                    float* vb_out, float4* G, bool first, bool layer0);

void edge_build_filter_rows(const float* Wf, const float* bf, int K, std::vector<unsigned short>& img);
bool message_bwd0_v3(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej, const float* Gb,
                     const int* types_s, const float* tab, int n_tab, const int* rev, const void* A_img, float4* G, bool first);
// ---- layer 0 with the channels contracted outside the edge loop (edge_l0.cu) ----
bool message_fwd0_collapsed_accum(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej,
                                  const int* types_s, int n_species, const float* s_in, int F, float* sn, int ldsn, float* As,
                                  float* Av, int NP, const float2* xph);
bool message_bwd0_collapsed(const Launch& L, long long N, int K, float rc, const int* row_ptr, const float4* ej,
                            const int* types_s, int n_species, const int* rev, const float* Bv, const float* Cs, int NP,
                            float4* G, bool first);

}  // namespace painn
