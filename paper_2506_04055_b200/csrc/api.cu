// api.cu -- the C ABI of include/mlp.h: weight blob parsing, buffer management (fixed capacity, grow on
// overflow: PAPER.md:84-86) and the per-timestep orchestration of the hot path.
#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>      // header-only; ranges are no-ops unless a profiler injects its library

#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/mlp.h"
#include "common.cuh"

using namespace painn;

namespace {

struct Buf {
    void* p = nullptr;
    size_t bytes = 0;
};

enum Stage { ST_NBR = 0, ST_FWD_NODE, ST_FWD_EDGE, ST_BWD_NODE, ST_BWD_EDGE, ST_FORCE, ST_L0, ST_COUNT };
// "layer0": both collapsed layer-0 message passes with their GEMMs (edge_l0.cu); fwd_edge / bwd_edge then hold layers >= 1
const char* kStageNames[ST_COUNT] = {"nbr_build", "fwd_node", "fwd_edge", "bwd_node", "bwd_edge", "force_virial", "layer0"};

struct LayerBuf {
    float *hpre, *phi, *sn, *v1, *pq, *zpre, *a;
};

}  // namespace

struct mlp_model {
    int n_species = 0, F = 0, K = 0, T = 0, R = 0;
    double rc = 0, eps = 0;
    // weights (device, fp32)
    std::vector<Buf> wbufs;
    std::vector<const float*> gemm_weights;
    float* Emb = nullptr;
    LayerW lw[PAINN_MAX_T];
    float *Wr1 = nullptr, *br1 = nullptr, *wr2 = nullptr, *br2 = nullptr, *Wr1T = nullptr;
    GemmRegistry reg;                   // tensor-core operands of the GEMM weights (split planes, exact slices)
    void* filt_rows[PAINN_MAX_T] = {};  // tcgen05 A operand (bf | Wf) of the edge kernels: three fp16 product-term planes, rows [3][F][80]
    int cell_strip = 6;                 // y-strip width of the cell order in cells (0: plain z, y, x order)
    int edge_path = 0;                  // 0: tensor-core edge kernels when F == 128, 1: plain fp32 kernels
    int apu_fwd = 12, apu_bwd = 16;     // atoms per work unit of the tensor-core edge kernels (option atoms_per_unit)
    int gemm_fwd_exact = 1;             // forward GEMMs: 1 exact integer-slice tcgen05 kernel, 0 fp32 FFMA kernel
    int phase_comp = 1;                 // forward edge kernels take the radial phase d / rc as an fp32 pair from the fp64 build
    float* tab0 = nullptr;              // [n_species][F] float2 (phi^s, phi^vs) of layer 0: s^0 = Emb[z] depends on the species only
    float *Wl0s = nullptr, *Wl0v = nullptr;   // [np0][F]: layer-0 adjoint with the channels contracted first (edge_l0.cu)
    float *Wl0sT = nullptr, *Wl0vT = nullptr; // [F][np0]: their transposes, the forward counterpart
    int np0 = 0;                        // columns of those GEMMs: n_species (K + 1) rounded up to 128
    int l0_collapse = 1;                // option: use them (0: k_msg_bwd0)
    // neighbour-list options: Verlet skin in Angstrom (0: every call rebuilds the list), T-hop pruning of
    // ghost-mode graphs, CUDA-graph replay of the steps that reuse the list
    double skin = 1.0;
    int prune = 1, use_graph = 1;
    // capacities
    long long cap_atoms = 0, cap_edges = 0, cap_cells = 0, cap_sup = 0;
    std::vector<Buf*> all;
    // atom-sized
    Buf b_cell_id, b_wrap, b_perm, b_inv_perm, b_pos_s, b_types_s, b_wrap_s, b_cell_s, b_local, b_row_cnt, b_row_ptr,
        b_scan_tmp;
    // cell-sized
    Buf b_cell_count, b_cell_start, b_cell_fill;
    // cell-sorted copies + relabelling of the pruned (level-major) atom order; reference state of the skin list
    Buf b_posC, b_typesC, b_wrapC, b_permC, b_localC, b_level, b_new_of_old, b_old_of_new, b_lvl_hist, b_pos_ref, b_wrap_ref,
        b_sup_ptr;
    // edge-sized
    Buf b_ej, b_img, b_rev, b_G, b_xph;   // b_xph: compensated phase (x_hi, x_lo) per edge slot
    Buf b_sup_j, b_sup_code;              // superset list at rc + skin (final indices, image codes)
    // node feature buffers
    Buf b_S[PAINN_MAX_T + 1], b_V[PAINN_MAX_T + 1];
    Buf b_hpre[PAINN_MAX_T], b_phi[PAINN_MAX_T], b_sn[PAINN_MAX_T], b_v1[PAINN_MAX_T], b_pq[PAINN_MAX_T],
        b_zpre[PAINN_MAX_T], b_a[PAINN_MAX_T];
    Buf b_h, b_rpre, b_rb, b_eatom, b_sb, b_s1b, b_vb, b_v1b, b_ab, b_pqb, b_gb, b_snb, b_phib, b_hb;
    Buf b_epart, b_wpart, b_red;        // b_red: 128 x 10 doubles, first stage of the final reduction
    Buf b_Q4, b_Q1;   // gather rows of the tensor-core edge kernels
    // small
    Buf b_misc;            // device: [0..7] flags (int), then long long totals, then bbox doubles
    void* h_misc = nullptr;   // pinned mirror
    // host staging for mlp_compute_host
    Buf d_pos, d_types, d_owner, d_out;   // d_out: energy[1] virial[6] forces[3N]
    Buf b_gout, b_gowner;                 // outputs / owner map of the captured step (same layout as d_out)
    cudaStream_t own_stream = nullptr;
    cudaStream_t side_stream = nullptr;            // reverse-edge index is built beside the forward pass
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_gin = nullptr, ev_gout = nullptr;
    // last call
    long long N_last = 0, n_local_last = 0, E_last = 0 /* padded slots */, E_real_last = 0;
    Grid grid_last{};
    // state of the list kept between calls (skin > 0)
    struct ListState {
        bool valid = false;
        long long N = 0, n_local = 0, n_ghost = 0;
        double box[3] = {0, 0, 0};
        Grid g{};
        bool pruned = false;
        long long prefix[PAINN_MAX_T + 3] = {};    // atoms with hop level < k (pruned lists)
        long long n_rebuild = 0, n_reuse = 0;
    } ls;
    void* h_misc2 = nullptr;              // pinned: totals of a step whose host read is deferred (list reuse / graph replay)
    bool stats_pending = false;
    cudaStream_t stats_stream = nullptr;
    // captured reuse step
    cudaGraphExec_t graph_exec = nullptr;
    bool graph_has_owner = false;         // what the captured step was built for
    void *graph_out = nullptr, *graph_owner = nullptr;
    long long graph_launches = 0;         // kernels inside the captured step
    mlp_stats stats{};
    std::string err;
    // stage timing
    bool timing = false;
    bool nvtx_open = false;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<std::pair<int, cudaEvent_t>> marks;
    long long forced_edge_cap = 0;
    bool fwd_tc = false;   // run the forward GEMMs on tensor cores too (faster, biased energy)
    bool bwd_exact = false;   // adjoint GEMMs through the exact integer-slice kernel instead of 3xTF32
};

namespace {

const char* kNoModel = "mlp: NULL model";

int fail(mlp_model* m, int code, const std::string& msg) {
    if (m) m->err = msg;
    return code;
}
#define CU(m, call)                                                                                   \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return fail(m, e_ == cudaErrorMemoryAllocation ? MLP_ERR_NOMEM : MLP_ERR_CUDA,            \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                          \
    } while (0)

int ensure(mlp_model* m, Buf& b, size_t bytes, bool count_regrow = true) {
    if (bytes <= b.bytes) return MLP_OK;
    // contents are never carried over, so the old buffer goes first (peak memory = the larger of the two, not the sum)
    if (b.p) {
        cudaFree(b.p);
        m->stats.device_bytes -= (long long)b.bytes;
        b.p = nullptr;
        b.bytes = 0;
    }
    CU(m, cudaMalloc(&b.p, bytes));
    b.bytes = bytes;
    m->stats.device_bytes += (long long)bytes;
    (void)count_regrow;
    return MLP_OK;
}
#define ENS(m, b, bytes)                             \
    do {                                             \
        int r_ = ensure(m, b, (size_t)(bytes));      \
        if (r_ != MLP_OK) return r_;                 \
    } while (0)

template <class T>
T* P(const Buf& b) { return reinterpret_cast<T*>(b.p); }

void free_buf(Buf& b, mlp_model* m);
struct TmpBuf : Buf {             // scratch of the debug exports: released on every return path
    mlp_model* m;
    explicit TmpBuf(mlp_model* m_) : m(m_) {}
    ~TmpBuf() { free_buf(*this, m); }
};

int upload(mlp_model* m, const std::vector<float>& h, float** out) {
    Buf b;
    ENS(m, b, h.size() * sizeof(float));
    CU(m, cudaMemcpy(b.p, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice));
    m->wbufs.push_back(b);
    *out = (float*)b.p;
    return MLP_OK;
}
float rn_tf32_host(float x) {
    uint32_t u;
    memcpy(&u, &x, 4);
    u += 0xfffu + ((u >> 13) & 1u);
    u &= 0xffffe000u;
    memcpy(&x, &u, 4);
    return x;
}
// GEMM weight: fp32 matrix plus its (hi, lo) TF32 split planes for the 3xTF32 tensor-core path
int upload_gemm_weight(mlp_model* m, const std::vector<float>& w, float** out) {
    int r = upload(m, w, out);
    if (r != MLP_OK) return r;
    std::vector<float> hi(w.size()), lo(w.size());
    for (size_t i = 0; i < w.size(); i++) { hi[i] = rn_tf32_host(w[i]); lo[i] = rn_tf32_host(w[i] - hi[i]); }
    float *dh, *dl;
    if ((r = upload(m, hi, &dh)) != MLP_OK) return r;
    if ((r = upload(m, lo, &dl)) != MLP_OK) return r;
    painn::gemm_register_split(m->reg, *out, dh, dl);
    m->gemm_weights.push_back(*out);
    return MLP_OK;
}
std::vector<float> to_f32(const double* p, size_t n) {
    std::vector<float> v(n);
    for (size_t i = 0; i < n; i++) v[i] = (float)p[i];
    return v;
}
std::vector<float> transpose(const std::vector<float>& w, int rows, int cols) {   // [rows x cols] -> [cols x rows]
    std::vector<float> t((size_t)rows * cols);
    for (int r = 0; r < rows; r++)
        for (int c = 0; c < cols; c++) t[(size_t)c * rows + r] = w[(size_t)r * cols + c];
    return t;
}

// The three alloc_* functions zero their capacity first and set it only when every buffer is in place: a failed
// cudaMalloc half-way leaves capacity 0, so the next call reallocates instead of running kernels on freed pointers.
int alloc_atoms(mlp_model* m, long long cap) {
    const size_t F = m->F, R = m->R, n = (size_t)cap;
    m->cap_atoms = 0;
    ENS(m, m->b_cell_id, n * 4); ENS(m, m->b_wrap, n * 3); ENS(m, m->b_perm, n * 4); ENS(m, m->b_inv_perm, n * 4);
    ENS(m, m->b_pos_s, n * 24); ENS(m, m->b_types_s, n * 4); ENS(m, m->b_wrap_s, n * 3); ENS(m, m->b_cell_s, n * 4);
    ENS(m, m->b_local, n * 4); ENS(m, m->b_row_cnt, n * 4); ENS(m, m->b_row_ptr, (n + 1) * 4);
    ENS(m, m->b_scan_tmp, (std::max<size_t>(n, (size_t)m->cap_cells) / 4096 + 2) * 4);   // exclusive_scan over atoms and over cells
    for (int t = 0; t <= m->T; t++) { ENS(m, m->b_S[t], n * F * 4); ENS(m, m->b_V[t], n * 3 * F * 4); }
    for (int t = 0; t < m->T; t++) {
        ENS(m, m->b_hpre[t], n * F * 4); ENS(m, m->b_phi[t], n * 3 * F * 4); ENS(m, m->b_sn[t], n * 2 * F * 4);
        ENS(m, m->b_v1[t], n * 3 * F * 4); ENS(m, m->b_pq[t], n * 6 * F * 4); ENS(m, m->b_zpre[t], n * F * 4);
        ENS(m, m->b_a[t], n * 3 * F * 4);
    }
    ENS(m, m->b_h, n * F * 4); ENS(m, m->b_rpre, n * R * 4); ENS(m, m->b_rb, n * R * 4); ENS(m, m->b_eatom, n * 4);
    ENS(m, m->b_sb, n * F * 4); ENS(m, m->b_s1b, n * F * 4); ENS(m, m->b_vb, n * 3 * F * 4);
    ENS(m, m->b_v1b, n * 3 * F * 4); ENS(m, m->b_ab, n * 3 * F * 4); ENS(m, m->b_pqb, n * 6 * F * 4);
    ENS(m, m->b_gb, n * F * 4); ENS(m, m->b_snb, n * 2 * F * 4); ENS(m, m->b_phib, n * 3 * F * 4);
    ENS(m, m->b_hb, n * F * 4);
    if (m->F == 128) { ENS(m, m->b_Q4, n * F * 16); ENS(m, m->b_Q1, n * F * 4); }
    ENS(m, m->b_epart, (n / 256 + 2) * 8); ENS(m, m->b_wpart, (n / 8 + 2) * 9 * 8);
    ENS(m, m->b_red, 128 * 10 * 8);
    m->cap_atoms = cap;
    return MLP_OK;
}
int alloc_edges(mlp_model* m, long long cap) {
    const size_t n = (size_t)cap;
    m->cap_edges = 0;
    ENS(m, m->b_ej, n * 16); ENS(m, m->b_img, n); ENS(m, m->b_rev, n * 4); ENS(m, m->b_G, n * 16); ENS(m, m->b_xph, n * 8);
    m->cap_edges = cap;
    return MLP_OK;
}
int alloc_cells(mlp_model* m, long long cap) {
    const size_t n = (size_t)cap;
    m->cap_cells = 0;
    ENS(m, m->b_cell_count, (n + 1) * 4); ENS(m, m->b_cell_start, (n + 2) * 4); ENS(m, m->b_cell_fill, (n + 1) * 4);
    ENS(m, m->b_scan_tmp, (std::max<size_t>(n, (size_t)m->cap_atoms) / 4096 + 2) * 4);   // the cell scan uses it too
    m->cap_cells = cap;
    return MLP_OK;
}

void free_buf(Buf& b, mlp_model* m) {
    if (b.p) cudaFree(b.p);
    if (m) m->stats.device_bytes -= (long long)b.bytes;
    b.p = nullptr;
    b.bytes = 0;
}

// layout of b_misc / h_misc
struct Misc {
    int flags[8];                         // [0] FLAG_* bits, [1] reverse-edge misses
    long long cell_total;
    long long edge_total;                 // padded CSR slots (rows padded to ROW_PAD)
    unsigned long long real_edges;        // edges with d < rc
    long long sup_total;                  // entries of the superset list
    unsigned long long sup_padded;        // bound of the padded CSR of any step the superset list serves
    long long prefix[PAINN_MAX_T + 3];    // pruned lists: atoms with hop level < k; [T + 1] = reached atoms (kept across calls)
    double bbox[6 + 6 * 256];
};
constexpr size_t MISC_HEAD = offsetof(Misc, bbox);        // what the host reads
constexpr size_t MISC_CLEAR = offsetof(Misc, prefix);     // what every call zeroes

// Stage boundary: an NVTX range per stage (host-side, around the launches of the stage; visible in nsys / ncu --nvtx) and,
// with stage timing enabled, a CUDA event on the stream.  stage < 0 closes the last range of the call.
void mark(mlp_model* m, cudaStream_t st, int stage) {
    if (m->nvtx_open) { nvtxRangePop(); m->nvtx_open = false; }
    if (stage >= 0 && stage < ST_COUNT) { nvtxRangePushA(kStageNames[stage]); m->nvtx_open = true; }
    if (!m->timing) return;
    size_t k = m->marks.size();
    if (k >= m->ev_pool.size()) {
        cudaEvent_t e;
        cudaEventCreate(&e);
        m->ev_pool.push_back(e);
    }
    cudaEventRecord(m->ev_pool[k], st);
    m->marks.push_back({stage, m->ev_pool[k]});
}

void drop_graph(mlp_model* m) {
    if (m->graph_exec) { cudaGraphExecDestroy(m->graph_exec); m->graph_exec = nullptr; }
}

// everything one mlp_compute call hands to the stages below
struct StepCtx {
    mlp_model* m;
    Launch& L;
    cudaStream_t st;
    const double* pos;
    const int* types;
    const double* box;
    long long n_local, n_ghost;
    const int* ghost_owner;
    double *energy, *forces, *virial;
    long long N;
    bool periodic;
};

// totals of a step whose host read was deferred (list reuse): wait for that step and take them over
int settle_stats(mlp_model* m) {
    if (!m->stats_pending) return MLP_OK;
    CU(m, cudaStreamSynchronize(m->stats_stream));
    const Misc* h2 = (const Misc*)m->h_misc2;
    m->E_last = h2->edge_total;
    m->E_real_last = (long long)h2->real_edges;
    m->stats.n_edges = m->E_real_last;
    m->stats_pending = false;
    return MLP_OK;
}

int run_model(StepCtx& cx);

EdgeOut edge_out(mlp_model* m) {
    return EdgeOut{P<float4>(m->b_ej), P<unsigned char>(m->b_img), P<int>(m->b_G), m->phase_comp ? P<float2>(m->b_xph) : nullptr,
                   1.0 / m->rc, (float)m->rc};
}

int regrow_edges(mlp_model* m, long long need) {
    // enlarge: x1.5, at least the counted need plus head-room ("overflown and nearly filled")
    long long nc = std::max((long long)(1.5 * m->cap_edges), need + need / 8);
    free_buf(m->b_ej, m); free_buf(m->b_img, m); free_buf(m->b_rev, m); free_buf(m->b_G, m); free_buf(m->b_xph, m);
    int r = alloc_edges(m, nc);
    if (r != MLP_OK) return r;
    m->stats.n_regrow++;
    return MLP_OK;
}

// a0-a3 from scratch: cell grid, binning, counting sort, [T-hop pruning + level-major relabelling], then either the CSR
// at rc (skin == 0) or the superset list at rc + skin (the CSR of the step is then filtered from it by step_from_list).
// Two host reads at most: the bounding box (ghost mode) and flags + totals (the overflow check of PAPER.md:84).
int build_list(StepCtx& cx, bool use_skin) {
    mlp_model* m = cx.m;
    Launch& L = cx.L;
    cudaStream_t st = cx.st;
    const long long N = cx.N, n_local = cx.n_local;
    const double* box = cx.box;
    const bool periodic = cx.periodic;
    const int T = m->T;
    Misc* dm = P<Misc>(m->b_misc);
    Misc* hm = (Misc*)m->h_misc;
    const double rlist = m->rc + (use_skin ? m->skin : 0.0);

    // ---- cell grid (cells of side >= list cutoff) ----
    Grid g{};
    g.periodic = periodic ? 1 : 0;
    g.rc2 = m->rc * m->rc;
    double lo[3] = {0, 0, 0}, ext[3] = {box[0], box[1], box[2]};
    if (!periodic) {
        nbr_bbox(L, cx.pos, N, dm->bbox);
        CU(m, cudaMemcpyAsync(hm->bbox, dm->bbox, 6 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(m, cudaStreamSynchronize(st));
        for (int d = 0; d < 3; d++) {
            if (!(hm->bbox[d] <= hm->bbox[3 + d])) return fail(m, MLP_ERR_NONFINITE, "no finite positions");
            lo[d] = hm->bbox[d];
            ext[d] = hm->bbox[3 + d] - hm->bbox[d];
        }
    }
    const double min_side = rlist * (1.0 + 1e-9);
    long long ncells = 1;
    for (int d = 0; d < 3; d++) {
        long long n = (long long)std::floor(ext[d] / min_side);
        if (n < 1) n = 1;
        if (!periodic) n += 1;   // open mode: side = rlist (1+1e-9) exactly, last cell partially filled
        g.n[d] = (int)n;
        g.origin[d] = lo[d];
        g.box[d] = box[d];
        g.inv_side[d] = periodic ? (double)n / ext[d] : 1.0 / min_side;
        ncells *= n;
    }
    // a periodic dimension with fewer than 3 cells would visit the same cell twice with the same shift: with the skin the
    // 27-cell stencil needs box >= 3 cells only when images could coincide; n = 1, 2 are handled by distinct shifts
    // cap the grid (sparse / huge bounding boxes): coarser cells are still correct, only slower
    const long long max_cells = std::max<long long>(4 * N + 4096, 32768);
    while (ncells > max_cells) {
        int dmax = 0;
        for (int d = 1; d < 3; d++) if (g.n[d] > g.n[dmax]) dmax = d;
        int nn = (g.n[dmax] + 1) / 2;
        if (periodic) g.inv_side[dmax] = (double)nn / ext[dmax];
        else { g.inv_side[dmax] *= 0.5; }
        g.n[dmax] = nn;
        ncells = (long long)g.n[0] * g.n[1] * g.n[2];
    }
    if (ncells > m->cap_cells) {
        int r = alloc_cells(m, ncells + ncells / 2);
        if (r != MLP_OK) return r;
    }
    g.strip = m->cell_strip > 0 && m->cell_strip < g.n[1] ? m->cell_strip : std::max(g.n[1], 1);
    m->grid_last = g;
    int* cell_count = P<int>(m->b_cell_count);
    int* cell_start = P<int>(m->b_cell_start);
    int* cell_fill = P<int>(m->b_cell_fill);
    CU(m, cudaMemsetAsync(cell_count, 0, (size_t)(ncells + 1) * 4, st));
    CU(m, cudaMemsetAsync(cell_fill, 0, (size_t)(ncells + 1) * 4, st));

    // ---- a0-a2: bin, counting sort, gather into cell-sorted order ----
    const bool prune = m->prune && !periodic && N > 0;
    if (prune) {
        const size_t n = (size_t)m->cap_atoms;
        ENS(m, m->b_posC, n * 24); ENS(m, m->b_typesC, n * 4); ENS(m, m->b_wrapC, n * 3); ENS(m, m->b_permC, n * 4);
        ENS(m, m->b_localC, n * 4); ENS(m, m->b_level, n); ENS(m, m->b_new_of_old, n * 4); ENS(m, m->b_old_of_new, n * 4);
        ENS(m, m->b_lvl_hist, (size_t)(PAINN_MAX_T + 2) * (n / 256 + 2) * 4);
    }
    double* posC = prune ? P<double>(m->b_posC) : P<double>(m->b_pos_s);
    int* typesC = prune ? P<int>(m->b_typesC) : P<int>(m->b_types_s);
    signed char* wrapC = prune ? P<signed char>(m->b_wrapC) : P<signed char>(m->b_wrap_s);
    int* permC = prune ? P<int>(m->b_permC) : P<int>(m->b_perm);
    float* localC = prune ? P<float>(m->b_localC) : P<float>(m->b_local);
    nbr_bin(L, cx.pos, cx.types, N, m->n_species, g, P<int>(m->b_cell_id), P<signed char>(m->b_wrap), cell_count, dm->flags, n_local,
            cx.ghost_owner);
    exclusive_scan(L, cell_count, cell_start, ncells, P<int>(m->b_scan_tmp), &dm->cell_total);
    nbr_place(L, N, ncells, P<int>(m->b_cell_id), cell_start, cell_fill, permC);
    nbr_sort_cells(L, ncells, cell_start, permC);
    nbr_gather(L, N, n_local, permC, cx.pos, cx.types, P<signed char>(m->b_wrap), posC, typesC, wrapC, P<int>(m->b_inv_perm),
               localC, P<int>(m->b_cell_id), P<int>(m->b_cell_s));
    NbrSearch S{posC, wrapC, P<int>(m->b_cell_s), cell_start, nullptr, nullptr, rlist * rlist};
    const int* n_rows_p = nullptr;

    // ---- T-hop pruning (ghost mode): hop levels from the local atoms, level-major final order ----
    if (prune) {
        nbr_levels(L, N, g, S, localC, P<unsigned char>(m->b_level), T);
        nbr_level_sort(L, N, P<unsigned char>(m->b_level), T, P<int>(m->b_lvl_hist), dm->prefix, P<int>(m->b_new_of_old),
                       P<int>(m->b_old_of_new));
        nbr_regather(L, N, P<int>(m->b_old_of_new), posC, typesC, wrapC, permC, localC, P<double>(m->b_pos_s), P<int>(m->b_types_s),
                     P<signed char>(m->b_wrap_s), P<int>(m->b_perm), P<int>(m->b_inv_perm), P<float>(m->b_local));
        S.new_of_old = P<int>(m->b_new_of_old);
        S.old_of_new = P<int>(m->b_old_of_new);
        n_rows_p = (const int*)&dm->prefix[T + 1];        // low word of the count of reached atoms (N < 2^31, little endian)
    }

    // ---- a3: count -> scan -> (host read: flags, totals, overflow check) -> fill ----
    if (use_skin) {
        ENS(m, m->b_sup_ptr, (size_t)(m->cap_atoms + 1) * 4);
        ENS(m, m->b_pos_ref, (size_t)m->cap_atoms * 24); ENS(m, m->b_wrap_ref, (size_t)m->cap_atoms * 3);
        nbr_sup_count(L, N, g, S, n_rows_p, P<int>(m->b_row_cnt), &dm->sup_padded);
        exclusive_scan(L, P<int>(m->b_row_cnt), P<int>(m->b_sup_ptr), N, P<int>(m->b_scan_tmp), &dm->sup_total);
    } else {
        nbr_count(L, N, g, S, n_rows_p, P<int>(m->b_row_cnt), &dm->real_edges);
        exclusive_scan(L, P<int>(m->b_row_cnt), P<int>(m->b_row_ptr), N, P<int>(m->b_scan_tmp), &dm->edge_total);
    }
    CU(m, cudaMemcpyAsync(hm, dm, MISC_HEAD, cudaMemcpyDeviceToHost, st));
    CU(m, cudaStreamSynchronize(st));
    if (hm->flags[0] & FLAG_NONFINITE) return fail(m, MLP_ERR_NONFINITE, "non-finite (or absurdly far) position");
    if (hm->flags[0] & FLAG_TYPE_RANGE) return fail(m, MLP_ERR_TYPE_RANGE, "atom type outside 0..n_species-1");
    if (hm->flags[0] & FLAG_OWNER_RANGE) return fail(m, MLP_ERR_ARG, "ghost_owner entry outside 0..n_local-1");
    const long long E = use_skin ? (long long)hm->sup_padded : hm->edge_total;
    if (E >= (1ll << 31) - 64 || hm->sup_total >= (1ll << 31) - 64) return fail(m, MLP_ERR_NOMEM, "more than 2^31 edges");
    if (E > m->cap_edges) {
        int r = regrow_edges(m, E);
        if (r != MLP_OK) return r;
    }
    mlp_model::ListState& ls = m->ls;
    ls.pruned = prune;
    for (int k = 0; k <= T + 2; k++) ls.prefix[k] = prune ? hm->prefix[k] : 0;
    ls.g = g;
    if (use_skin) {
        if (hm->sup_total > m->cap_sup) {
            const long long nc = hm->sup_total + hm->sup_total / 8;
            m->cap_sup = 0;
            ENS(m, m->b_sup_j, (size_t)nc * 4); ENS(m, m->b_sup_code, (size_t)nc);
            m->cap_sup = nc;
        }
        nbr_sup_fill(L, N, g, S, n_rows_p, P<int>(m->b_sup_ptr), P<int>(m->b_sup_j), P<unsigned char>(m->b_sup_code));
        CU(m, cudaMemcpyAsync(m->b_pos_ref.p, m->b_pos_s.p, (size_t)N * 24, cudaMemcpyDeviceToDevice, st));
        CU(m, cudaMemcpyAsync(m->b_wrap_ref.p, m->b_wrap_s.p, (size_t)N * 3, cudaMemcpyDeviceToDevice, st));
        ls.valid = true;
        ls.N = N; ls.n_local = n_local; ls.n_ghost = cx.n_ghost;
        for (int d = 0; d < 3; d++) ls.box[d] = box[d];
    } else {
        nbr_fill(L, N, g, S, n_rows_p, P<int>(m->b_row_ptr), m->cap_edges, edge_out(m), dm->flags);
        m->E_last = E;
        m->E_real_last = (long long)hm->real_edges;
        m->stats.n_edges = m->E_real_last;
    }
    return MLP_OK;
}

// A step served by the kept superset list: the CSR at rc is filtered from it with the fp64 predicate on the current
// positions (the per-step cutoff pruning of PAPER.md:68), then the model runs.  No host read: the padded CSR of any such
// step fits the edge buffers by construction (sup_padded was reserved at the build), totals are read back lazily.
int step_from_list(StepCtx& cx) {
    mlp_model* m = cx.m;
    Launch& L = cx.L;
    const long long N = cx.N;
    Misc* dm = P<Misc>(m->b_misc);
    const Grid& g = m->ls.g;
    nbr_refilter_count(L, N, g, P<double>(m->b_pos_s), P<signed char>(m->b_wrap_s), P<int>(m->b_sup_ptr), P<int>(m->b_sup_j),
                       P<unsigned char>(m->b_sup_code), P<int>(m->b_row_cnt), &dm->real_edges);
    exclusive_scan(L, P<int>(m->b_row_cnt), P<int>(m->b_row_ptr), N, P<int>(m->b_scan_tmp), &dm->edge_total);
    nbr_refilter_fill(L, N, g, P<double>(m->b_pos_s), P<signed char>(m->b_wrap_s), P<int>(m->b_sup_ptr), P<int>(m->b_sup_j),
                      P<unsigned char>(m->b_sup_code), P<int>(m->b_row_ptr), m->cap_edges, edge_out(m), dm->flags);
    int r = run_model(cx);
    if (r != MLP_OK) return r;
    CU(m, cudaMemcpyAsync(m->h_misc2, dm, MISC_HEAD, cudaMemcpyDeviceToHost, cx.st));
    m->stats_pending = true;
    m->stats_stream = cx.st;
    return MLP_OK;
}

// a4-a13 on the CSR in the edge buffers.  With a pruned list the atoms are in level-major order and layer t only
// updates the rows within T - 1 - t hops of a local atom (a prefix): Fig. 1e.
int run_model(StepCtx& cx) {
    mlp_model* m = cx.m;
    Launch& L = cx.L;
    cudaStream_t st = cx.st;
    const long long N = cx.N, n_local = cx.n_local;
    const int* ghost_owner = cx.ghost_owner;
    double *energy = cx.energy, *forces = cx.forces, *virial = cx.virial;
    const int F = m->F, K = m->K, T = m->T, R = m->R;
    const float rcf = (float)m->rc;
    Misc* dm = P<Misc>(m->b_misc);
    float4* ej = P<float4>(m->b_ej);
    const int* row_ptr = P<int>(m->b_row_ptr);
    const float2* xph = m->phase_comp ? P<float2>(m->b_xph) : nullptr;
    long long& launches = *L.counter;
    // rows that layer t updates (receivers) and rows whose layer-t input state exists (senders)
    long long Nrecv[PAINN_MAX_T], Nsend[PAINN_MAX_T];
    const bool pruned = m->ls.pruned;
    for (int t = 0; t < T; t++) {
        Nrecv[t] = pruned ? m->ls.prefix[T - t] : N;            // hop level <= T - 1 - t
        Nsend[t] = pruned ? m->ls.prefix[T - t + 1] : N;        // hop level <= T - t
    }
    const long long Nreach = pruned ? m->ls.prefix[T + 1] : N;

    // the reverse-edge index is needed by the layer-0 adjoint and the force assembly only: build it on a side stream,
    // overlapped with the forward pass (its warps fit beside the GEMM / element-wise kernels).  Its compact search
    // keys live in the G buffer, which nothing touches before the adjoint pass (joined below before it starts)
    {
        Launch Ls = L;
        Ls.stream = m->side_stream;
        CU(m, cudaEventRecord(m->ev_fork, st));
        CU(m, cudaStreamWaitEvent(m->side_stream, m->ev_fork, 0));
        nbr_reverse(Ls, N, row_ptr, ej, P<unsigned char>(m->b_img), P<int>(m->b_G), P<int>(m->b_rev), &dm->flags[1]);
        CU(m, cudaEventRecord(m->ev_join, m->side_stream));
    }

    // ---- forward ----
    // Tensor-core accumulation truncates toward zero after every MMA (measured, B3): a relative bias of
    // ~ -0.4 ulp per chained MMA that the energy (an absolute 1e-4/atom tolerance on E/atom ~ 40-160) cannot absorb,
    // while forces (relative tolerance) can.  Forward GEMMs (launch context Lf) therefore run the exact integer-slice
    // tcgen05 kernel (fp32 FFMA kernel where it does not cover the shape), the adjoint GEMMs (Lb) tcgen05 3xTF32.
    Launch Lf = L, Lb = L;
    Lf.gemm_path = m->fwd_tc ? 0 : 1;
    // debug: gemm_fwd_exact is a bit mask over the forward GEMM types (2 phi-MLP in, 4 phi-MLP out, 8 U|V, 16 gate-MLP in,
    // 32 gate-MLP out, 64 readout and layer-0 sums); 1 = all
    auto LfT = [&](int type) { Launch x = Lf; x.fwd_exact = m->gemm_fwd_exact == 1 ? 1 : ((m->gemm_fwd_exact >> (type + 1)) & 1); return x; };
    Lb.gemm_path = m->bwd_exact ? 1 : 0;
    const bool tc_edges = m->edge_path == 0 && F == 128 && K <= 23 && m->filt_rows[0] != nullptr;
    mark(m, st, ST_FWD_NODE);
    embed(L, Nreach, F, P<int>(m->b_types_s), m->Emb, P<float>(m->b_S[0]), P<float>(m->b_V[0]));
    float* h = P<float>(m->b_h);
    for (int t = 0; t < T; t++) {
        const LayerW& l = m->lw[t];
        const long long Nr = Nrecv[t], Ns = Nsend[t];       // rows updated by this layer / rows that send into it
        float *S = P<float>(m->b_S[t]), *V = P<float>(m->b_V[t]);
        float *hpre = P<float>(m->b_hpre[t]), *phi = P<float>(m->b_phi[t]), *sn = P<float>(m->b_sn[t]),
              *v1 = P<float>(m->b_v1[t]), *pq = P<float>(m->b_pq[t]), *zpre = P<float>(m->b_zpre[t]),
              *a = P<float>(m->b_a[t]);
        // layer 0: s^0 = Emb[z], so phi(s^0) is a per-species table (built at create); no per-atom phi-MLP, no gather rows
        const bool l0_table = t == 0 && tc_edges && m->tab0;
        const bool fuse_act = !m->fwd_tc && gemm_act_supported(3 * F, F);   // SiLU applied while loading A
        if (!l0_table) {
            gemm_nt(LfT(0), S, F, l.Wm1, F, hpre, F, Ns, F, F, l.bm1, false);
            if (fuse_act) gemm_nt_act(LfT(1), hpre, F, l.Wm2, F, phi, 3 * F, Ns, 3 * F, F, l.bm2, false, true);
            else {
                silu_fwd(L, Ns * F, hpre, h);
                gemm_nt(Lf, h, F, l.Wm2, F, phi, 3 * F, Ns, 3 * F, F, l.bm2, false);
            }
        }
        mark(m, st, ST_FWD_EDGE);
        bool done = false;
        if (l0_table && m->l0_collapse && m->Wl0sT && m->np0 == 128) {
            // layer 0: per-(receiver, species) radial sums (O(K) per edge), then two GEMMs (edge_l0.cu).  The sums live in
            // the gather-row buffers, which layer 0 does not use: Q1 [N][128], Q4 [3N][128] floats
            float *As = P<float>(m->b_Q1), *Av = P<float>(m->b_Q4);
            mark(m, st, ST_L0);
            if (message_fwd0_collapsed_accum(L, Nr, K, rcf, row_ptr, ej, P<int>(m->b_types_s), m->n_species, S, F, sn, 2 * F, As, Av,
                                             m->np0, xph)) {
                gemm_nt(LfT(5), As, m->np0, m->Wl0sT, m->np0, sn, 2 * F, Nr, F, m->np0, nullptr, true);
                gemm_nt(LfT(5), Av, m->np0, m->Wl0vT, m->np0, v1, F, 3 * Nr, F, m->np0, nullptr, false);
                done = true;
            }
        }
        if (!done && tc_edges && (t > 0 || l0_table)) {
            if (!l0_table) make_gather_rows(L, Ns, phi, V, P<float>(m->b_Q4), P<float>(m->b_Q1), t > 0);
            done = message_fwd_v3(L, Nr, K, rcf, row_ptr, ej, S, V, P<float>(m->b_Q4), P<float>(m->b_Q1), m->filt_rows[t], sn, v1, t > 0, P<int>(m->b_types_s), m->tab0, m->n_species, xph);
        }
        if (!done) {
            if (l0_table) return fail(m, MLP_ERR_CUDA, "layer-0 table path unavailable");   // (phi was not computed)
            message_fwd(L, Nr, F, K, rcf, row_ptr, ej, S, V, phi, l.Wf, l.bf, sn, v1);
        }
        mark(m, st, ST_FWD_NODE);
        gemm_nt(LfT(2), v1, F, l.UV, F, pq, 2 * F, 3 * Nr, 2 * F, F, nullptr, false);
        update_mid(L, Nr, F, (float)m->eps, pq, sn);
        gemm_nt(LfT(3), sn, 2 * F, l.Wu1, 2 * F, zpre, F, Nr, F, 2 * F, l.bu1, false);
        if (fuse_act) gemm_nt_act(LfT(4), zpre, F, l.Wu2, F, a, 3 * F, Nr, 3 * F, F, l.bu2, false, true);
        else {
            silu_fwd(L, Nr * F, zpre, h);
            gemm_nt(Lf, h, F, l.Wu2, F, a, 3 * F, Nr, 3 * F, F, l.bu2, false);
        }
        update_out(L, Nr, F, sn, v1, pq, a, P<float>(m->b_S[t + 1]), P<float>(m->b_V[t + 1]));
    }
    int n_epart = 0, n_wpart = 0;
    const long long Nout = Nrecv[T - 1];                    // rows that carry s^T: with a pruned list exactly the local atoms
    gemm_nt(LfT(5), P<float>(m->b_S[T]), F, m->Wr1, F, P<float>(m->b_rpre), R, Nout, R, F, m->br1, false);
    readout(L, Nout, R, P<float>(m->b_rpre), m->wr2, m->br2, P<float>(m->b_local), P<float>(m->b_rb),
            P<float>(m->b_eatom), P<double>(m->b_epart), &n_epart);

    // ---- backward ----
    CU(m, cudaStreamWaitEvent(st, m->ev_join, 0));          // reverse-edge index ready
    mark(m, st, ST_BWD_NODE);
    float *sb = P<float>(m->b_sb), *s1b = P<float>(m->b_s1b), *vb = P<float>(m->b_vb), *v1b = P<float>(m->b_v1b);
    gemm_nt(Lb, P<float>(m->b_rb), R, m->Wr1T, R, sb, F, Nout, F, R, nullptr, false);
    if (Nout > 0) CU(m, cudaMemsetAsync(vb, 0, (size_t)Nout * 3 * F * 4, st));
    // pruned list: the edge kernels of a layer only visit a prefix of the rows, so G cannot rely on the first layer's
    // overwrite: start from zero and accumulate everywhere
    if (pruned && m->b_G.p) CU(m, cudaMemsetAsync(m->b_G.p, 0, m->b_G.bytes, st));
    for (int t = T - 1; t >= 0; t--) {
        const LayerW& l = m->lw[t];
        const long long Nr = Nrecv[t], Ns = Nsend[t];
        const bool first = t == T - 1 && !pruned;              // first adjoint edge pass overwrites G
        float *ab = P<float>(m->b_ab), *pqb = P<float>(m->b_pqb), *gb = P<float>(m->b_gb), *snb = P<float>(m->b_snb),
              *phib = P<float>(m->b_phib), *hb = P<float>(m->b_hb);
        update_bwd1(L, Nr, F, sb, vb, P<float>(m->b_pq[t]), P<float>(m->b_a[t]), ab, pqb);
        gemm_nt_dsilu(Lb, ab, 3 * F, l.Wu2T, 3 * F, gb, F, Nr, F, 3 * F, P<float>(m->b_zpre[t]));
        gemm_nt(Lb, gb, F, l.Wu1T, F, snb, 2 * F, Nr, 2 * F, F, nullptr, false);
        // vb'_1 = vb + (U^T pb + V^T qb): the GEMM takes vb as the residual of its epilogue (no copy into v1b first)
        update_bwd2(L, Nr, F, sb, vb, snb, P<float>(m->b_sn[t]), P<float>(m->b_pq[t]), pqb, s1b, nullptr);
        gemm_nt_resid(Lb, pqb, 2 * F, l.UVT, 2 * F, v1b, F, 3 * Nr, F, 2 * F, vb);
        // rows this layer does not update carry a zero (s', v') adjoint: the senders' own rows (Nr .. Ns) and every row a
        // sender may gather from (its neighbours: up to one hop further out)
        const long long Nz = pruned ? Nreach : Nr;
        if (Nz > Nr) {
            CU(m, cudaMemsetAsync(s1b + Nr * F, 0, (size_t)(Nz - Nr) * F * 4, st));
            CU(m, cudaMemsetAsync(v1b + Nr * 3 * F, 0, (size_t)(Nz - Nr) * 3 * F * 4, st));
        }
        mark(m, st, ST_BWD_EDGE);
        bool done = false;
        const bool l0_table = t == 0 && tc_edges && m->tab0;
        if (l0_table && m->l0_collapse && m->Wl0s && m->np0 == 128) {
            // layer 0: contract the channels per (receiver, sender species) with two GEMMs, then O(K) work per edge.
            // B -> the gather-row buffer ([3N][128] floats of its [N][128] float4), C -> the (unused at layer 0) phib buffer
            float *Bv = P<float>(m->b_Q4), *Cs = phib;
            mark(m, st, ST_L0);
            gemm_nt(Lb, v1b, F, m->Wl0v, F, Bv, m->np0, 3 * Nr, m->np0, F, nullptr, false);
            gemm_nt(Lb, s1b, F, m->Wl0s, F, Cs, m->np0, Nr, m->np0, F, nullptr, false);
            done = message_bwd0_collapsed(L, Nr, K, rcf, row_ptr, ej, P<int>(m->b_types_s), m->n_species, P<int>(m->b_rev), Bv,
                                          Cs, m->np0, P<float4>(m->b_G), first);
        }
        if (!done && tc_edges) {
            make_gather_rows_bwd(L, Nz, s1b, v1b, P<float>(m->b_Q4));     // (rows Nr .. Nz are zero)
            if (l0_table)
                done = message_bwd0_v3(L, Nr, K, rcf, row_ptr, ej, P<float>(m->b_Q4), P<int>(m->b_types_s), m->tab0, m->n_species,
                                       P<int>(m->b_rev), m->filt_rows[0], P<float4>(m->b_G), first);
            if (!done)
                done = message_bwd_v3(L, Ns, K, rcf, row_ptr, ej, P<float>(m->b_Q4), P<float>(m->b_phi[t]),
                                      P<float>(m->b_V[t]), v1b, m->filt_rows[t], phib, vb, P<float4>(m->b_G), first, t == 0);
        }
        if (!done) {
            if (l0_table) return fail(m, MLP_ERR_CUDA, "layer-0 table path unavailable");
            message_bwd(L, Ns, F, K, rcf, row_ptr, ej, s1b, v1b, P<float>(m->b_phi[t]), P<float>(m->b_V[t]), l.Wf, l.bf,
                        phib, vb, P<float4>(m->b_G), first);
        }
        mark(m, st, ST_BWD_NODE);
        if (t == 0) break;      // s^0 is the (constant) embedding: its adjoint is never used
        gemm_nt_dsilu(Lb, phib, 3 * F, l.Wm2T, 3 * F, hb, F, Ns, F, 3 * F, P<float>(m->b_hpre[t]));
        gemm_nt(Lb, hb, F, l.Wm1T, F, s1b, F, Ns, F, F, nullptr, true);
        std::swap(sb, s1b);
    }

    // ---- forces, ghost fold, virial, energy ----
    mark(m, st, ST_FORCE);
    if (N > 0) CU(m, cudaMemsetAsync(forces, 0, (size_t)N * 3 * 8, st));
    force_final(L, N, n_local, row_ptr, ej, P<int>(m->b_rev), P<float4>(m->b_G), P<int>(m->b_perm), ghost_owner,
                forces, P<double>(m->b_wpart), &n_wpart);
    reduce_final(L, P<double>(m->b_epart), n_epart, P<double>(m->b_wpart), n_wpart, P<double>(m->b_red), energy, virial);
    (void)launches;
    return MLP_OK;
}

}  // namespace

extern "C" {

__attribute__((visibility("default"))) const char* mlp_version(void) { return "painn-b200 0.1.0 sm_100a"; }

__attribute__((visibility("default"))) const char* mlp_last_error(mlp_model* m) { return m ? m->err.c_str() : kNoModel; }

__attribute__((visibility("default"))) int mlp_create(const void* weights, size_t nbytes, int n_species, double cutoff, long long capacity,
               mlp_model** out) {
    if (!out) return MLP_ERR_ARG;
    *out = nullptr;
    if (!weights || capacity <= 0) return MLP_ERR_ARG;
    const unsigned char* b = (const unsigned char*)weights;
    if (nbytes < 48 || memcmp(b, "PNN1", 4) != 0) return MLP_ERR_WEIGHTS;
    uint32_t h[7];
    memcpy(h, b + 4, sizeof h);
    double rc, eps;
    memcpy(&rc, b + 32, 8);
    memcpy(&eps, b + 40, 8);
    if (h[0] != 1) return MLP_ERR_WEIGHTS;
    const int ns = (int)h[1], F = (int)h[2], K = (int)h[3], T = (int)h[4], R = (int)h[5];
    if (ns != n_species || rc != cutoff || !(rc > 0)) return MLP_ERR_WEIGHTS;
    if (!(F == 32 || F == 64 || F == 128) || K < 1 || K > PAINN_MAX_K || T < 1 || T > PAINN_MAX_T || R != F / 2 ||
        ns < 1)
        return MLP_ERR_WEIGHTS;
    size_t per_layer = (size_t)F * F + F + 3 * F * F + 3 * F + 3 * F * K + 3 * F + 2 * (size_t)F * F + 2 * F * F + F +
                       3 * F * F + 3 * F;
    size_t n_dbl = (size_t)ns * F + T * per_layer + (size_t)R * F + R + R + 1;
    if (nbytes != 48 + 8 * n_dbl) return MLP_ERR_WEIGHTS;

    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) return MLP_ERR_CUDA;

    mlp_model* m = new (std::nothrow) mlp_model();
    if (!m) return MLP_ERR_NOMEM;
    m->n_species = ns; m->F = F; m->K = K; m->T = T; m->R = R; m->rc = rc; m->eps = eps;
    std::vector<double> w(n_dbl);
    memcpy(w.data(), b + 48, 8 * n_dbl);
    const double* p = w.data();
    int rcode = MLP_OK;
    auto up = [&](size_t n, float** dst, std::vector<float>* keep = nullptr) {
        if (rcode != MLP_OK) { p += n; return; }
        std::vector<float> v = to_f32(p, n);
        p += n;
        rcode = keep ? upload_gemm_weight(m, v, dst) : upload(m, v, dst);   // keep != nullptr <=> GEMM matrix
        if (keep) *keep = v;
    };
    auto upT = [&](const std::vector<float>& v, int rows, int cols, float** dst) {
        if (rcode != MLP_OK) return;
        const std::vector<float> t = transpose(v, rows, cols);          // [cols x rows]
        rcode = upload_gemm_weight(m, t, dst);
        if (rcode == MLP_OK) painn::gemm_register_exact(m->reg, *dst, t.data(), cols, rows);
    };
    up((size_t)ns * F, &m->Emb);
    std::vector<float> Wf0_h, bf0_h;          // layer-0 filter weights (for the collapsed layer-0 adjoint)
    for (int t = 0; t < T; t++) {
        LayerW& l = m->lw[t];
        std::vector<float> Wm1, Wm2, U, V, Wu1, Wu2;
        float* tmp;
        up((size_t)F * F, (float**)&l.Wm1, &Wm1); up(F, (float**)&l.bm1);
        up((size_t)3 * F * F, (float**)&l.Wm2, &Wm2); up(3 * F, (float**)&l.bm2);
        {
            std::vector<float> Wf_h = to_f32(p, (size_t)3 * F * K), bf_h = to_f32(p + (size_t)3 * F * K, (size_t)3 * F);
            if (t == 0) { Wf0_h = Wf_h; bf0_h = bf_h; }
            if (F == 128 && K <= 23 && rcode == MLP_OK) {
                std::vector<unsigned short> img;
                edge_build_filter_rows(Wf_h.data(), bf_h.data(), K, img);
                Buf b3;
                rcode = ensure(m, b3, img.size() * 2);
                if (rcode == MLP_OK && cudaMemcpy(b3.p, img.data(), img.size() * 2, cudaMemcpyHostToDevice) != cudaSuccess) rcode = MLP_ERR_CUDA;
                m->wbufs.push_back(b3);
                m->filt_rows[t] = b3.p;
            }
        }
        up((size_t)3 * F * K, (float**)&l.Wf); up(3 * F, (float**)&l.bf);
        // U and V are consecutive in the blob -> stacked [2F x F] matrix UV = [U ; V]
        std::vector<float> UV = to_f32(p, (size_t)2 * F * F);
        p += (size_t)2 * F * F;
        if (rcode == MLP_OK) rcode = upload_gemm_weight(m, UV, &tmp);
        l.UV = tmp;
        up((size_t)F * 2 * F, (float**)&l.Wu1, &Wu1); up(F, (float**)&l.bu1);
        up((size_t)3 * F * F, (float**)&l.Wu2, &Wu2); up(3 * F, (float**)&l.bu2);
        if (rcode == MLP_OK) {      // integer slices for the exact tensor-core path of the forward GEMMs
            painn::gemm_register_exact(m->reg, l.Wm1, Wm1.data(), F, F);
            painn::gemm_register_exact(m->reg, l.Wm2, Wm2.data(), 3 * F, F);
            painn::gemm_register_exact(m->reg, l.UV, UV.data(), 2 * F, F);
            painn::gemm_register_exact(m->reg, l.Wu1, Wu1.data(), F, 2 * F);
            painn::gemm_register_exact(m->reg, l.Wu2, Wu2.data(), 3 * F, F);
        }
        upT(Wm1, F, F, (float**)&l.Wm1T);
        upT(Wm2, 3 * F, F, (float**)&l.Wm2T);
        upT(UV, 2 * F, F, (float**)&l.UVT);
        upT(Wu1, F, 2 * F, (float**)&l.Wu1T);
        upT(Wu2, 3 * F, F, (float**)&l.Wu2T);
    }
    std::vector<float> Wr1;
    up((size_t)R * F, &m->Wr1, &Wr1); up(R, &m->br1); up(R, &m->wr2); up(1, &m->br2);
    if (rcode == MLP_OK) painn::gemm_register_exact(m->reg, m->Wr1, Wr1.data(), R, F);
    upT(Wr1, R, F, &m->Wr1T);
    if (rcode == MLP_OK && F == 128 && m->filt_rows[0] && ns <= 16) {
        // layer-0 sender rows per species: phi(Emb[z]) through the same forward GEMM path as the per-atom rows
        Buf bh, bp;
        rcode = ensure(m, bh, (size_t)ns * F * 4);
        if (rcode == MLP_OK) rcode = ensure(m, bp, (size_t)ns * 3 * F * 4);
        if (rcode == MLP_OK) {
            long long cnt = 0;
            Launch L{nullptr, &cnt};
            L.reg = &m->reg;
            L.gemm_path = 1;                  // the same forward GEMM kernels as the per-atom rows of the other layers
            gemm_nt(L, m->Emb, F, m->lw[0].Wm1, F, P<float>(bh), F, ns, F, F, m->lw[0].bm1, false);
            silu_fwd(L, (long long)ns * F, P<float>(bh), P<float>(bh));
            gemm_nt(L, P<float>(bh), F, m->lw[0].Wm2, F, P<float>(bp), 3 * F, ns, 3 * F, F, m->lw[0].bm2, false);
            std::vector<float> ph((size_t)ns * 3 * F), tab((size_t)ns * F * 2);
            if (cudaDeviceSynchronize() != cudaSuccess ||
                cudaMemcpy(ph.data(), bp.p, ph.size() * 4, cudaMemcpyDeviceToHost) != cudaSuccess)
                rcode = MLP_ERR_CUDA;
            for (int z = 0; z < ns; z++)
                for (int f = 0; f < F; f++) {
                    tab[((size_t)z * F + f) * 2] = ph[(size_t)z * 3 * F + f];
                    tab[((size_t)z * F + f) * 2 + 1] = ph[(size_t)z * 3 * F + F + f];
                }
            if (rcode == MLP_OK) rcode = upload(m, tab, &m->tab0);
            // layer-0 adjoint, channels contracted first (edge_l0.cu): rows n = z (K + 1) + k,
            //   Wl0s[n][c] = Wf^s[c][k] phi^s_z[c],  Wl0v[n][c] = Wf^vs[c][k] phi^vs_z[c]   (k = 0: the bias bf)
            const int KP1 = K + 1, np0 = ((ns * KP1 + 127) / 128) * 128;
            if (rcode == MLP_OK && K <= 23 && !Wf0_h.empty()) {
                std::vector<float> ws((size_t)np0 * F, 0.f), wv((size_t)np0 * F, 0.f);
                for (int z = 0; z < ns; z++)
                    for (int k = 0; k < KP1; k++)
                        for (int c = 0; c < F; c++) {
                            const float fs = k == 0 ? bf0_h[c] : Wf0_h[(size_t)c * K + (k - 1)];
                            const float fv = k == 0 ? bf0_h[F + c] : Wf0_h[(size_t)(F + c) * K + (k - 1)];
                            ws[((size_t)z * KP1 + k) * F + c] = fs * tab[((size_t)z * F + c) * 2];
                            wv[((size_t)z * KP1 + k) * F + c] = fv * tab[((size_t)z * F + c) * 2 + 1];
                        }
                rcode = upload_gemm_weight(m, ws, &m->Wl0s);
                if (rcode == MLP_OK) rcode = upload_gemm_weight(m, wv, &m->Wl0v);
                const std::vector<float> wsT = transpose(ws, np0, F), wvT = transpose(wv, np0, F);
                if (rcode == MLP_OK) rcode = upload_gemm_weight(m, wsT, &m->Wl0sT);
                if (rcode == MLP_OK) painn::gemm_register_exact(m->reg, m->Wl0sT, wsT.data(), F, np0);
                if (rcode == MLP_OK) rcode = upload_gemm_weight(m, wvT, &m->Wl0vT);
                if (rcode == MLP_OK) painn::gemm_register_exact(m->reg, m->Wl0vT, wvT.data(), F, np0);
                if (rcode == MLP_OK) m->np0 = np0;
            }
        }
        free_buf(bh, m);
        free_buf(bp, m);
    }
    if (rcode == MLP_OK) rcode = ensure(m, m->b_misc, sizeof(Misc));
    if (rcode == MLP_OK && (cudaMallocHost(&m->h_misc, sizeof(Misc)) != cudaSuccess || cudaMallocHost(&m->h_misc2, sizeof(Misc)) != cudaSuccess))
        rcode = MLP_ERR_NOMEM;
    if (rcode == MLP_OK && (cudaStreamCreateWithFlags(&m->own_stream, cudaStreamNonBlocking) != cudaSuccess ||
                            cudaStreamCreateWithFlags(&m->side_stream, cudaStreamNonBlocking) != cudaSuccess ||
                            cudaEventCreateWithFlags(&m->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                            cudaEventCreateWithFlags(&m->ev_join, cudaEventDisableTiming) != cudaSuccess ||
                            cudaEventCreateWithFlags(&m->ev_gin, cudaEventDisableTiming) != cudaSuccess ||
                            cudaEventCreateWithFlags(&m->ev_gout, cudaEventDisableTiming) != cudaSuccess))
        rcode = MLP_ERR_CUDA;
    if (rcode == MLP_OK) rcode = alloc_atoms(m, capacity);
    if (rcode == MLP_OK) rcode = alloc_edges(m, 64 * capacity);
    if (rcode == MLP_OK) rcode = alloc_cells(m, capacity + 1024);
    if (rcode != MLP_OK) {
        mlp_destroy(m);
        return rcode;
    }
    m->stats.atom_capacity = m->cap_atoms;
    m->stats.edge_capacity = m->cap_edges;
    *out = m;
    return MLP_OK;
}

__attribute__((visibility("default"))) void mlp_destroy(mlp_model* m) {
    if (!m) return;
    painn::gemm_registry_free(m->reg);
    for (Buf& b : m->wbufs) free_buf(b, nullptr);
    Buf* bs[] = {&m->b_cell_id, &m->b_wrap, &m->b_perm, &m->b_inv_perm, &m->b_pos_s, &m->b_types_s, &m->b_wrap_s,
                 &m->b_cell_s, &m->b_local, &m->b_row_cnt, &m->b_row_ptr, &m->b_scan_tmp, &m->b_cell_count,
                 &m->b_cell_start, &m->b_cell_fill, &m->b_ej, &m->b_img, &m->b_rev, &m->b_G, &m->b_xph, &m->b_sup_j, &m->b_sup_code,
                 &m->b_posC, &m->b_typesC, &m->b_wrapC, &m->b_permC, &m->b_localC, &m->b_level, &m->b_new_of_old, &m->b_old_of_new,
                 &m->b_lvl_hist, &m->b_pos_ref, &m->b_wrap_ref, &m->b_sup_ptr, &m->b_h, &m->b_rpre,
                 &m->b_rb, &m->b_eatom, &m->b_sb, &m->b_s1b, &m->b_vb, &m->b_v1b, &m->b_ab, &m->b_pqb, &m->b_gb,
                 &m->b_snb, &m->b_phib, &m->b_hb, &m->b_Q4, &m->b_Q1, &m->b_epart, &m->b_wpart, &m->b_red, &m->b_misc, &m->d_pos, &m->d_types,
                 &m->d_owner, &m->d_out, &m->b_gout, &m->b_gowner};
    for (Buf* b : bs) free_buf(*b, nullptr);
    for (int t = 0; t <= PAINN_MAX_T; t++) { free_buf(m->b_S[t], nullptr); free_buf(m->b_V[t], nullptr); }
    for (int t = 0; t < PAINN_MAX_T; t++) {
        free_buf(m->b_hpre[t], nullptr); free_buf(m->b_phi[t], nullptr); free_buf(m->b_sn[t], nullptr); free_buf(m->b_v1[t], nullptr);
        free_buf(m->b_pq[t], nullptr); free_buf(m->b_zpre[t], nullptr); free_buf(m->b_a[t], nullptr);
    }
    if (m->graph_exec) cudaGraphExecDestroy(m->graph_exec);
    if (m->h_misc) cudaFreeHost(m->h_misc);
    if (m->h_misc2) cudaFreeHost(m->h_misc2);
    if (m->own_stream) cudaStreamDestroy(m->own_stream);
    if (m->side_stream) cudaStreamDestroy(m->side_stream);
    if (m->ev_fork) cudaEventDestroy(m->ev_fork);
    if (m->ev_join) cudaEventDestroy(m->ev_join);
    if (m->ev_gin) cudaEventDestroy(m->ev_gin);
    if (m->ev_gout) cudaEventDestroy(m->ev_gout);
    for (cudaEvent_t e : m->ev_pool) cudaEventDestroy(e);
    delete m;
}

__attribute__((visibility("default"))) int mlp_set_option(mlp_model* m, const char* name, long long value) {
    if (!m || !name) return MLP_ERR_ARG;
    // every option may change what a captured step would launch: drop the graph and the kept list
    if (m->graph_exec) { cudaGraphExecDestroy(m->graph_exec); m->graph_exec = nullptr; }
    m->ls.valid = false;
    if (!strcmp(name, "stage_timing")) { m->timing = value != 0; return MLP_OK; }
    if (!strcmp(name, "skin_mA")) {
        if (value < 0 || value > 20000) return fail(m, MLP_ERR_ARG, "skin_mA must be 0 .. 20000 (1e-3 Angstrom)");
        m->skin = 1e-3 * (double)value;
        return MLP_OK;
    }
    if (!strcmp(name, "prune")) { m->prune = value != 0; return MLP_OK; }
    if (!strcmp(name, "use_graph")) { m->use_graph = value != 0; return MLP_OK; }
    if (!strcmp(name, "edge_path")) { m->edge_path = (int)value; return MLP_OK; }
    if (!strcmp(name, "cell_strip")) {
        if (value < 0) return fail(m, MLP_ERR_ARG, "cell_strip must be >= 0");
        m->cell_strip = (int)value;
        return MLP_OK;
    }
    if (!strcmp(name, "l0_collapse")) { m->l0_collapse = (int)value; return MLP_OK; }
    if (!strcmp(name, "gemm_fwd_tc")) { m->fwd_tc = value != 0; return MLP_OK; }
    if (!strcmp(name, "gemm_bwd_exact")) { m->bwd_exact = value != 0; return MLP_OK; }
    if (!strcmp(name, "gemm_fwd_exact")) { m->gemm_fwd_exact = (int)value; return MLP_OK; }
    if (!strcmp(name, "phase_comp")) { m->phase_comp = value != 0; return MLP_OK; }
    if (!strcmp(name, "atoms_per_unit")) {
        if (value < 0 || value > 31) return fail(m, MLP_ERR_ARG, "atoms_per_unit must be 1..31 (one row pointer per lane) or 0");
        m->apu_bwd = value ? (int)value : 16;
        m->apu_fwd = value ? (int)value : 12;
        return MLP_OK;
    }
    if (!strcmp(name, "edge_capacity")) {
        if (value <= 0) return fail(m, MLP_ERR_ARG, "edge_capacity must be > 0");
        // shrink-or-set (test hook): drop the edge buffers and reallocate at the requested size
        free_buf(m->b_ej, m); free_buf(m->b_img, m); free_buf(m->b_rev, m); free_buf(m->b_G, m); free_buf(m->b_xph, m);
        int r = alloc_edges(m, value);
        m->stats.edge_capacity = m->cap_edges;
        return r;
    }
    return fail(m, MLP_ERR_ARG, std::string("unknown option ") + name);
}

__attribute__((visibility("default"))) int mlp_get_stats(mlp_model* m, mlp_stats* out) {
    if (!m || !out) return MLP_ERR_ARG;
    int r = settle_stats(m);
    if (r != MLP_OK) return r;
    *out = m->stats;
    return MLP_OK;
}

__attribute__((visibility("default"))) int mlp_get_stage_ms(mlp_model* m, int max_stages, const char** names, float* ms) {
    if (!m || !names || !ms || max_stages < 0) return -MLP_ERR_ARG;
    float acc[ST_COUNT] = {0};
    if (m->marks.size() >= 2) {
        if (cudaEventSynchronize(m->marks.back().second) != cudaSuccess) return -MLP_ERR_CUDA;
        for (size_t k = 0; k + 1 < m->marks.size(); k++) {
            float t = 0;
            cudaEventElapsedTime(&t, m->marks[k].second, m->marks[k + 1].second);
            int s = m->marks[k].first;
            if (s >= 0 && s < ST_COUNT) acc[s] += t;
        }
    }
    int n = max_stages < ST_COUNT ? max_stages : ST_COUNT;
    for (int k = 0; k < n; k++) { names[k] = kStageNames[k]; ms[k] = acc[k]; }
    return n;
}

__attribute__((visibility("default"))) int mlp_compute(mlp_model* m, const double* pos, const int* types, const double* box, long long n_local,
                long long n_ghost, const int* ghost_owner, double* energy, double* forces, double* virial,
                void* cuda_stream) {
    if (!m) return MLP_ERR_ARG;
    if (!box || n_local < 0 || n_ghost < 0 || !energy || !virial) return fail(m, MLP_ERR_ARG, "bad argument");
    const long long N = n_local + n_ghost;
    if (N > 0 && (!pos || !types || !forces)) return fail(m, MLP_ERR_ARG, "NULL atom array");
    if (N >= (1ll << 31)) return fail(m, MLP_ERR_ARG, "too many atoms");
    for (int d = 0; d < 3; d++)
        if (!std::isfinite(box[d]) || !(box[d] > 0)) return fail(m, MLP_ERR_NONFINITE, "box length not finite/positive");
    const bool periodic = n_ghost == 0;
    if (periodic)
        for (int d = 0; d < 3; d++)
            if (box[d] < 2.0 * m->rc) return fail(m, MLP_ERR_BOX_TOO_SMALL, "periodic box length < 2 * cutoff");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    long long launches = 0;
    Launch L{st, &launches};
    L.reg = &m->reg;
    L.fwd_exact = m->gemm_fwd_exact;
    L.apu_fwd = m->apu_fwd;
    L.apu_bwd = m->apu_bwd;
    m->marks.clear();
    m->stats.n_calls++;
    const int T = m->T;

    // ---- capacity (atoms): buffers only grow ----
    if (N > m->cap_atoms) {
        long long nc = std::max(N, (long long)(1.5 * m->cap_atoms));
        drop_graph(m);
        m->ls.valid = false;
        int r = alloc_atoms(m, nc);
        if (r != MLP_OK) return r;
        m->stats.n_regrow++;
    }
    Misc* dm = P<Misc>(m->b_misc);
    Misc* hm = (Misc*)m->h_misc;
    CU(m, cudaMemsetAsync(dm, 0, MISC_CLEAR, st));
    mark(m, st, ST_NBR);
    const bool use_skin = m->skin > 0.0 && N > 0;
    StepCtx cx{m, L, st, pos, types, box, n_local, n_ghost, ghost_owner, energy, forces, virial, N, periodic};

    // ---- a step that reuses the kept list: refresh positions, test the displacement, replay ----
    mlp_model::ListState& ls = m->ls;
    bool reuse = false;
    if (use_skin && ls.valid && ls.N == N && ls.n_local == n_local && ls.n_ghost == n_ghost && ls.box[0] == box[0] &&
        ls.box[1] == box[1] && ls.box[2] == box[2]) {
        nbr_reuse_prep(L, N, P<int>(m->b_perm), pos, types, P<double>(m->b_pos_ref), P<signed char>(m->b_wrap_ref),
                       P<int>(m->b_types_s), ls.g, 0.25 * m->skin * m->skin, P<double>(m->b_pos_s), P<signed char>(m->b_wrap_s),
                       dm->flags);
        CU(m, cudaMemcpyAsync(hm, dm, sizeof(int) * 8, cudaMemcpyDeviceToHost, st));
        CU(m, cudaStreamSynchronize(st));
        if (hm->flags[0] & FLAG_NONFINITE) return fail(m, MLP_ERR_NONFINITE, "non-finite (or absurdly far) position");
        reuse = !(hm->flags[0] & FLAG_REBUILD);
        if (!reuse) CU(m, cudaMemsetAsync(dm, 0, MISC_CLEAR, st));
    }
    if (reuse) {
        ls.n_reuse++;
        int r = MLP_OK;
        const bool want_graph = m->use_graph && !m->timing;
        // The captured step lives on the model's own stream (the caller's may be the legacy default stream, which cannot be
        // captured), ordered after / before the caller's stream with two events, and touches NO caller buffer: it reads the
        // model's copy of the owner map and writes E, W, F into the model's staging buffer, both copied outside the graph.
        // So one capture serves every later reuse step, whatever buffers the caller passes.
        cudaStream_t gs = m->own_stream;
        const bool has_owner = ghost_owner != nullptr && n_ghost > 0;
        double* gout = nullptr;
        int* gowner = nullptr;
        if (want_graph) {
            ENS(m, m->b_gout, (size_t)(7 + 3 * N) * 8);
            if (has_owner) ENS(m, m->b_gowner, (size_t)n_ghost * 4);
            gout = P<double>(m->b_gout);
            gowner = has_owner ? P<int>(m->b_gowner) : nullptr;
        }
        if (want_graph && !(m->graph_exec && m->graph_has_owner == has_owner && m->graph_out == (void*)gout && m->graph_owner == (void*)gowner)) {
            // capture this step once; later steps replay it (no launch overhead, no host read)
            drop_graph(m);
            cudaGraph_t graph = nullptr;
            const long long l0 = launches;
            if (cudaStreamBeginCapture(gs, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                Launch Lg = L;
                Lg.stream = gs;
                StepCtx cgx{m, Lg, gs, pos, types, box, n_local, n_ghost, gowner, gout, gout + 7, gout + 1, N, periodic};
                r = step_from_list(cgx);
                cudaError_t ce = cudaStreamEndCapture(gs, &graph);
                if (r == MLP_OK && ce == cudaSuccess && graph &&
                    cudaGraphInstantiate(&m->graph_exec, graph, nullptr, nullptr, 0) == cudaSuccess) {
                    m->graph_has_owner = has_owner;
                    m->graph_out = gout;
                    m->graph_owner = gowner;
                    m->graph_launches = launches - l0;
                } else
                    m->graph_exec = nullptr;
                if (graph) cudaGraphDestroy(graph);
            }
            launches = l0;
            if (!m->graph_exec) {
                cudaGetLastError();
                m->use_graph = 0;                                   // capture is not available here: launch directly from now on
                r = MLP_OK;
            }
        }
        if (want_graph && m->graph_exec) {
            CU(m, cudaEventRecord(m->ev_gin, st));
            CU(m, cudaStreamWaitEvent(gs, m->ev_gin, 0));
            if (has_owner) CU(m, cudaMemcpyAsync(gowner, ghost_owner, (size_t)n_ghost * 4, cudaMemcpyDeviceToDevice, gs));
            CU(m, cudaGraphLaunch(m->graph_exec, gs));
            CU(m, cudaMemcpyAsync(energy, gout, 8, cudaMemcpyDeviceToDevice, gs));
            CU(m, cudaMemcpyAsync(virial, gout + 1, 48, cudaMemcpyDeviceToDevice, gs));
            if (N > 0) CU(m, cudaMemcpyAsync(forces, gout + 7, (size_t)N * 24, cudaMemcpyDeviceToDevice, gs));
            CU(m, cudaEventRecord(m->ev_gout, gs));
            CU(m, cudaStreamWaitEvent(st, m->ev_gout, 0));
            launches += m->graph_launches;
            m->stats.n_graph_replays++;
            m->stats_pending = true;
            m->stats_stream = gs;
        } else
            r = step_from_list(cx);
        if (r != MLP_OK) return r;
    } else {
        drop_graph(m);
        ls.valid = false;
        int r = build_list(cx, use_skin);
        if (r != MLP_OK) return r;
        ls.n_rebuild++;
        r = use_skin ? step_from_list(cx) : run_model(cx);
        if (r != MLP_OK) return r;
    }
    mark(m, st, -1);
    CU(m, cudaGetLastError());

    m->N_last = N; m->n_local_last = n_local;
    m->stats.n_atoms = N; m->stats.atom_capacity = m->cap_atoms; m->stats.edge_capacity = m->cap_edges;
    for (int d = 0; d < 3; d++) m->stats.n_cells[d] = m->grid_last.n[d];
    m->stats.n_launches = launches;
    m->stats.n_list_rebuilds = ls.n_rebuild; m->stats.n_list_reuses = ls.n_reuse;
    m->stats.n_reached = ls.pruned ? ls.prefix[T + 1] : N;
    return MLP_OK;
}

__attribute__((visibility("default"))) int mlp_compute_host(mlp_model* m, const double* pos, const int* types, const double* box, long long n_local,
                     long long n_ghost, const int* ghost_owner, double* energy, double* forces, double* virial) {
    if (!m) return MLP_ERR_ARG;
    if (n_local < 0 || n_ghost < 0 || !energy || !virial) return fail(m, MLP_ERR_ARG, "bad argument");
    const long long N = n_local + n_ghost;
    if (N > 0 && (!pos || !types || !forces)) return fail(m, MLP_ERR_ARG, "NULL atom array");
    cudaStream_t st = m->own_stream;
    ENS(m, m->d_pos, (size_t)N * 24 + 8); ENS(m, m->d_types, (size_t)N * 4 + 8);
    ENS(m, m->d_out, (size_t)(7 + 3 * N) * 8);
    if (ghost_owner) ENS(m, m->d_owner, (size_t)n_ghost * 4 + 8);
    if (N > 0) {
        CU(m, cudaMemcpyAsync(m->d_pos.p, pos, (size_t)N * 24, cudaMemcpyHostToDevice, st));
        CU(m, cudaMemcpyAsync(m->d_types.p, types, (size_t)N * 4, cudaMemcpyHostToDevice, st));
    }
    if (ghost_owner && n_ghost > 0)
        CU(m, cudaMemcpyAsync(m->d_owner.p, ghost_owner, (size_t)n_ghost * 4, cudaMemcpyHostToDevice, st));
    double* dout = P<double>(m->d_out);
    int r = mlp_compute(m, P<double>(m->d_pos), P<int>(m->d_types), box, n_local, n_ghost,
                        ghost_owner ? P<int>(m->d_owner) : nullptr, dout, dout + 7, dout + 1, st);
    if (r != MLP_OK) return r;
    CU(m, cudaMemcpyAsync(energy, dout, 8, cudaMemcpyDeviceToHost, st));
    CU(m, cudaMemcpyAsync(virial, dout + 1, 48, cudaMemcpyDeviceToHost, st));
    if (N > 0) CU(m, cudaMemcpyAsync(forces, dout + 7, (size_t)N * 24, cudaMemcpyDeviceToHost, st));
    CU(m, cudaStreamSynchronize(st));
    return MLP_OK;
}

__attribute__((visibility("default"))) int mlp_get_neighbors(mlp_model* m, long long* n_edges, int* i, int* j, signed char* image3) {
    if (!m || !n_edges) return MLP_ERR_ARG;
    { int r = settle_stats(m); if (r != MLP_OK) return r; }
    *n_edges = m->E_real_last;
    if (!i) return MLP_OK;
    if (!j || !image3) return fail(m, MLP_ERR_ARG, "NULL output");
    const long long E = m->E_last, N = m->N_last;
    if (E == 0) return MLP_OK;
    TmpBuf bi(m), bj(m), bm(m);
    ENS(m, bi, E * 4); ENS(m, bj, E * 4); ENS(m, bm, E * 3);
    long long launches = 0;
    Launch L{m->own_stream, &launches};
    CU(m, cudaDeviceSynchronize());
    nbr_export(L, N, P<int>(m->b_row_ptr), P<float4>(m->b_ej), P<unsigned char>(m->b_img), P<int>(m->b_perm),
               P<signed char>(m->b_wrap_s), P<int>(bi), P<int>(bj), P<signed char>(bm));
    std::vector<int> hi(E), hj(E);
    std::vector<signed char> him(3 * (size_t)E);
    CU(m, cudaMemcpyAsync(hi.data(), bi.p, E * 4, cudaMemcpyDeviceToHost, m->own_stream));
    CU(m, cudaMemcpyAsync(hj.data(), bj.p, E * 4, cudaMemcpyDeviceToHost, m->own_stream));
    CU(m, cudaMemcpyAsync(him.data(), bm.p, E * 3, cudaMemcpyDeviceToHost, m->own_stream));
    CU(m, cudaStreamSynchronize(m->own_stream));
    long long k = 0;                                        // drop the padding slots
    for (long long e = 0; e < E; e++)
        if (hi[e] >= 0) {
            i[k] = hi[e]; j[k] = hj[e];
            image3[3 * k] = him[3 * e]; image3[3 * k + 1] = him[3 * e + 1]; image3[3 * k + 2] = him[3 * e + 2];
            k++;
        }
    return MLP_OK;
}

__attribute__((visibility("default"))) int mlp_debug_gemm(const float* A, const float* W, const float* bias,
                                                           float* C, long long M, int N, int K, int accumulate,
                                                           int path, int* used_tc) {
    if (!A || !W || !C || M < 0 || N <= 0 || K <= 0) return MLP_ERR_ARG;
    mlp_model tmp;
    mlp_model* m = &tmp;
    std::vector<float> w(W, W + (size_t)N * K);
    float *dW = nullptr, *dB = nullptr;
    int r = upload_gemm_weight(m, w, &dW);
    if (r == MLP_OK && bias) r = upload(m, std::vector<float>(bias, bias + N), &dB);
    if (r == MLP_OK) {
        long long launches = 0;
        int used = 0;
        Launch L{nullptr, &launches};
        L.reg = &m->reg;
        L.used_tc = &used;
        L.gemm_path = path == 0 ? 0 : 1;             // 0: 3xTF32 (adjoint path), 1: fp32 FFMA, 2: exact integer slices
        L.fwd_exact = path == 2 ? 1 : 0;
        if (path == 2) {
            painn::gemm_register_exact(m->reg, dW, w.data(), N, K);
            if (!painn::gemm_nt_exact(L, A, K, dW, C, N, M, N, K, dB, accumulate != 0, false)) r = MLP_ERR_ARG;
            else used = 1;
        } else
            gemm_nt(L, A, K, dW, K, C, N, M, N, K, dB, accumulate != 0);
        if (used_tc) *used_tc = used;
        cudaError_t e = cudaDeviceSynchronize();
        if (e != cudaSuccess) r = MLP_ERR_CUDA;
    }
    painn::gemm_registry_free(m->reg);
    for (Buf& b : m->wbufs) free_buf(b, nullptr);
    return r;
}

__attribute__((visibility("default"))) int mlp_get_layer_state(mlp_model* m, int t, float* out) {
    if (!m || !out || t < 0 || t > m->T) return MLP_ERR_ARG;
    const long long N = m->N_last;
    if (N == 0) return MLP_OK;
    TmpBuf b(m);
    ENS(m, b, (size_t)N * 4 * m->F * 4);
    long long launches = 0;
    Launch L{m->own_stream, &launches};
    CU(m, cudaDeviceSynchronize());
    unpermute_state(L, N, m->F, P<int>(m->b_perm), P<float>(m->b_S[t]), P<float>(m->b_V[t]), P<float>(b));
    CU(m, cudaMemcpyAsync(out, b.p, (size_t)N * 4 * m->F * 4, cudaMemcpyDeviceToHost, m->own_stream));
    CU(m, cudaStreamSynchronize(m->own_stream));
    return MLP_OK;
}

}  // extern "C"
