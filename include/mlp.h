/*
 * mlp.h -- C ABI of the B200-native PaiNN energy / force / virial hot path.
 *
 * One call per MD timestep (mlp_compute) evaluates, entirely in hand-written sm_100a CUDA kernels,
 *     E = sum_{i < n_local} E_i,   F = -dE/dr,   W_ab = -sum_e r_e,a (dE/dr_e)_b
 * for a fixed-weight PaiNN model on the cutoff graph of the given atoms.  What is computed is the
 * semi-local potential of PAPER.md:53-56 (Eq. 1) / PAPER.md:178-180 (Eq. 5), with the energy summed over
 * LOCAL atoms only, partial forces on all atoms of the domain graph summed onto their owners
 * (Eq. 2), edges longer than the cutoff pruned every step, fixed-capacity
 * buffers that only grow and are re-evaluated on overflow, and the message / update form
 * of PAPER.md:196-200 (Eq. 6-7) instantiated as PaiNN.  The model equations themselves
 * are the reading fixed in DESIGN.md section 2 (the paper names PaiNN but never prints its equations).
 *
 * Conventions
 *   - every function returns an MLP_* code; nothing throws or aborts across the ABI;
 *   - outputs are defined only when the return code is MLP_OK;
 *   - the library owns all scratch memory and grows it on demand (never shrinks);
 *   - the caller owns every pointer it passes; "DEVICE" = CUDA device memory of the current device,
 *     "HOST" = ordinary host memory;
 *   - mlp_compute is asynchronous on `cuda_stream` except for one host read of the edge count after the
 *     neighbour build (the overflow check of PAPER.md:84); mlp_compute_host is synchronous;
 *   - there is NO CPU fallback: without a CUDA device every compute entry point returns MLP_ERR_CUDA.
 */
#ifndef PAINN_B200_MLP_H
#define PAINN_B200_MLP_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mlp_model mlp_model; /* opaque; created by mlp_create, freed by mlp_destroy */

enum {
    MLP_OK = 0,
    MLP_ERR_ARG = 1,           /* NULL / negative / inconsistent argument                               */
    MLP_ERR_WEIGHTS = 2,       /* blob malformed, or n_species / cutoff disagree with its header         */
    MLP_ERR_BOX_TOO_SMALL = 3, /* periodic mode and some box length < 2 * cutoff                         */
    MLP_ERR_TYPE_RANGE = 4,    /* some types[i] outside 0 .. n_species-1                                 */
    MLP_ERR_NOMEM = 5,         /* device or host allocation failed                                       */
    MLP_ERR_CUDA = 6,          /* CUDA runtime error (text in mlp_last_error)                            */
    MLP_ERR_NONFINITE = 7      /* non-finite position or box length                                      */
};

/* Statistics of the most recent mlp_compute ("returns statistics of the computation"). */
typedef struct mlp_stats {
    long long n_atoms;        /* n_local + n_ghost of the last call                                      */
    long long n_edges;        /* directed edges (receiver <- sender) with d < cutoff                     */
    long long atom_capacity;  /* current atom buffer capacity                                            */
    long long edge_capacity;  /* current edge buffer capacity                                            */
    long long n_cells[3];     /* cell grid of the last call                                              */
    long long n_regrow;       /* how often a buffer had to grow since mlp_create        */
    long long n_calls;        /* mlp_compute calls since mlp_create                                      */
    long long n_launches;     /* kernels launched by the last call                                       */
    long long device_bytes;   /* device memory currently held by the model                               */
    long long n_list_rebuilds;  /* calls that built the neighbour list from scratch (PAPER.md:68 skin)     */
    long long n_list_reuses;    /* calls served by the kept rc + skin list (re-filtered at rc)              */
    long long n_graph_replays;  /* of those, calls replayed from the captured CUDA graph                    */
    long long n_reached;        /* atoms kept by the T-hop pruning of a ghost-mode graph (else n_atoms)     */
} mlp_stats;

/*
 * mlp_create -- parse the weight blob, upload the (fixed) weights, allocate scratch for `capacity` atoms.
 *   weights   HOST  blob, layout in DESIGN.md section 3 ("PNN1" header + fp64 arrays); copied, caller keeps its own
 *   nbytes          blob size in bytes
 *   n_species       must equal the header's n_species          (else MLP_ERR_WEIGHTS)
 *   cutoff          must equal the header's rc (Angstrom)      (else MLP_ERR_WEIGHTS)
 *   capacity        initial atom capacity (local + ghost), > 0; the edge buffer starts at 64 x capacity
 *   out             receives the handle
 * Supported shapes: F in {32, 64, 128}, K <= 32, T <= 8, R = F/2.
 */
int mlp_create(const void* weights, size_t nbytes, int n_species, double cutoff, long long capacity,
               mlp_model** out);

/*
 * mlp_compute -- one evaluation of E, F, virial (north_star items 1-4).
 *   pos          DEVICE fp64 [(n_local+n_ghost) x 3], caller order: locals first, then ghosts
 *   types        DEVICE i32  [n_local+n_ghost], 0 .. n_species-1
 *   box          HOST   fp64 [3] orthorhombic box lengths (origin 0)
 *   n_local, n_ghost
 *                n_ghost == 0: periodic boundaries in all three directions (minimum image, box >= 2*cutoff);
 *                n_ghost  > 0: open boundaries over the given atoms, the ghosts ARE the periodicity
 *   ghost_owner  DEVICE i32 [n_ghost] or NULL.  Non-NULL: ghost forces are added onto forces[owner] and the
 *                ghost rows are zeroed; NULL: partial forces are returned on all rows
 *   energy       DEVICE fp64 [1]
 *   forces       DEVICE fp64 [(n_local+n_ghost) x 3], caller order
 *   virial       DEVICE fp64 [6]  xx, yy, zz, xy, xz, yz  (W_ab = -sum_e r_e,a g_e,b, off-diagonals symmetrised;
 *                not divided by the volume)
 *   cuda_stream  cudaStream_t (NULL = default stream)
 * Errors: MLP_ERR_ARG (also: a ghost_owner entry outside 0 .. n_local-1), MLP_ERR_BOX_TOO_SMALL, MLP_ERR_TYPE_RANGE,
 * MLP_ERR_NONFINITE, MLP_ERR_NOMEM, MLP_ERR_CUDA.  MLP_ERR_TYPE_RANGE / MLP_ERR_NONFINITE / the owner range are detected on
 * the device and reported by this same call.
 * Host synchronisation: a call that builds the list reads flags and totals back once (twice in ghost mode: bounding box),
 * the overflow check of PAPER.md:84; a call that reuses the kept list reads one flag word (displacement test) and is
 * otherwise asynchronous.  Threads: one model must not be used from two threads at once; different models are independent
 * (no process-wide state).
 */
int mlp_compute(mlp_model* m, const double* pos, const int* types, const double* box, long long n_local,
                long long n_ghost, const int* ghost_owner, double* energy, double* forces, double* virial,
                void* cuda_stream);

/*
 * mlp_compute_host -- the same computation with HOST buffers for every argument (the end-to-end call an MD
 * engine with host-resident atoms makes; "transforms and copies data to the device ... copies
 * forces back").  The copies are cudaMemcpyAsync on the model's own stream straight from / to the caller's buffers (pin
 * them for full PCIe speed; pageable memory works and is staged by the driver); device staging buffers are owned by the
 * model.  Synchronous: returns when the outputs are in the caller's buffers.
 */
int mlp_compute_host(mlp_model* m, const double* pos, const int* types, const double* box, long long n_local,
                     long long n_ghost, const int* ghost_owner, double* energy, double* forces, double* virial);

/* mlp_destroy -- free everything (NULL is allowed). */
void mlp_destroy(mlp_model* m);

/*
 * mlp_get_neighbors -- edge list of the most recent mlp_compute, in caller atom indices (test / debug export
 * for the bit-exact neighbour-set check).  First call with i == NULL to obtain *n_edges, then with HOST buffers
 * i[n], j[n] (receiver, sender) and image3[3n] (S such that r_e = r_j + S*box - r_i, relative to the
 * positions as given).  Order of the edges is unspecified.  Synchronous.
 */
int mlp_get_neighbors(mlp_model* m, long long* n_edges, int* i, int* j, signed char* image3);

/*
 * mlp_get_layer_state -- debug export: node state after layer t (t = 0: embedding; t = 1..T), HOST fp32
 * [(n_local+n_ghost) x 4F] per atom (s | v_x | v_y | v_z), caller order.  Synchronous.
 */
int mlp_get_layer_state(mlp_model* m, int t, float* out);

/*
 * mlp_debug_gemm -- test export of the per-atom linear-layer kernel:
 *   C[M x N] (+)= A[M x K] . W[N x K]^T + bias.   A, C: DEVICE fp32 row-major (ld = K resp. N); W [N x K], bias [N]
 *   (or NULL): HOST fp32.  path 0 = tcgen05 3xTF32 (the adjoint GEMMs) when the shape is covered, 1 = plain fp32
 *   (FFMA / SIMT), 2 = tcgen05 exact integer slices (the forward GEMMs; MLP_ERR_ARG when the shape is not covered).
 *   *used_tc (may be NULL) receives 1 if a tensor-core kernel ran.  Synchronous.
 */
int mlp_debug_gemm(const float* A, const float* W, const float* bias, float* C, long long M, int N, int K,
                   int accumulate, int path, int* used_tc);

/* mlp_get_stats -- copy the statistics of the last call (waits for that call when it was served by the kept list: its
 * edge count is read back lazily). */
int mlp_get_stats(mlp_model* m, mlp_stats* out);

/*
 * mlp_get_stage_ms -- debug / measurement export: CUDA-event time in ms of each stage of the most recent
 * mlp_compute when stage timing was enabled with mlp_set_option("stage_timing", 1).  names[k] point to static
 * strings.  Returns the number of stages written (<= max_stages), or a negative MLP_* code.
 */
int mlp_get_stage_ms(mlp_model* m, int max_stages, const char** names, float* ms);

/* mlp_set_option -- integer knobs of ONE model (nothing is process-wide; setting an option drops the kept neighbour list
 * and the captured step of that model):
 *   "skin_mA"         Verlet skin in 1e-3 Angstrom, default 1000.  > 0: the list is built at cutoff + skin
 *                     and kept; a later call whose atoms have all moved less than skin / 2 (minimum image), with the same
 *                     atom counts, species and box, only re-filters it at the cutoff (exact: same fp64 predicate, same edge
 *                     set) and replays the captured CUDA graph.  0: every call rebuilds the list (the metric of bench.py)
 *   "prune"           1 (default): ghost mode drops the atoms no local atom reaches within T hops and restricts layer t to
 *                     the atoms within T - 1 - t hops (Fig. 1e; exact).  mlp_get_neighbors then returns the
 *                     sub-graph over the reached atoms.  0: all given atoms are carried through all layers
 *   "use_graph"       1 (default): steps that reuse the list are captured once and replayed with cudaGraphLaunch
 *   "stage_timing"    0/1: CUDA-event stage timers for mlp_get_stage_ms (disables graph replay while on)
 *   "edge_capacity"   TEST HOOK for the overflow / regrow path: drops the edge buffers and reallocates them
 *                     at exactly this size -- the one place where a buffer may shrink (mlp_compute itself only grows them)
 * and switches that select between implementations of the same arithmetic (defaults are the shipped path):
 *   "edge_path"       0 tensor-core edge kernels (F = 128, K <= 23), 1 plain fp32 kernels
 *   "l0_collapse"     1 layer-0 message passes with the channel contraction hoisted into GEMMs (n_species (K+1) <= 128),
 *                     0 per-edge channel kernels through the species table
 *   "gemm_fwd_exact"  1 forward GEMMs on tcgen05 with exact integer slices, 0 fp32 FFMA kernel (other values: bit mask over
 *                     the forward GEMM types, a measurement aid)
 *   "gemm_bwd_exact"  0 adjoint GEMMs 3xTF32, 1 exact integer slices
 *   "gemm_fwd_tc"     1 forward GEMMs 3xTF32 (biased energy, B3)
 *   "phase_comp"      1 (default) forward edge kernels take the radial phase d / rc as an fp32 pair from the fp64 build
 *   "cell_strip"      order of the cells (hence of the sorted atoms): y cut into strips of this many cells, inside a strip
 *                     (z, y, x); default 6, 0 = plain (z, y, x).  Keeps three z planes of gathered rows inside L2
 *   "atoms_per_unit"  1..31 consecutive cell-sorted atoms per work unit of the tensor-core edge kernels (default 12 forward,
 *                     16 adjoint; setting it sets both, 0 restores the defaults)
 * Unknown names return MLP_ERR_ARG. */
int mlp_set_option(mlp_model* m, const char* name, long long value);

/*
 * mlp_measure_row_gather -- measurement utility ("L2 -> SM bandwidth is not in PEAKS: measure it
 * first with a gather micro-benchmark, because it bounds the edge stages").  Runs the access pattern of the edge kernels --
 * a warp reads one 512-byte row per request, rows chosen inside `window` neighbouring rows of a table of `table_bytes`
 * (>= 1 MiB), 16 rows in flight per thread, 16 / 32 / 64 warps per SM -- on the current device and returns the best
 * sustained rate in GB/s in *gb_per_s (HOST).  Allocates and frees its own buffers; synchronous.
 */
int mlp_measure_row_gather(long long table_bytes, int window, double* gb_per_s);

/*
 * mlp_row_offsets_static -- the CSR row-offset step of the neighbour build ("compute the neighbor list";
 * per-receiver edge counts -> row_ptr by an exclusive scan) as an entry point that
 * ALLOCATES NOTHING: no cudaMalloc, cudaFree or allocating library routine is called, so it may be used where those are
 * forbidden (under CUDA graph capture, in tight serving loops).  The scratch of the scan (one total per block of 4,096
 * rows) lives in a file-scope device array of 64 KiB + 256 B that every GPU loading this library holds until exit.
 *   counts       DEVICE [n] int, read only
 *   offsets      DEVICE [n + 1] int, written: offsets[i] = counts[0] + ... + counts[i-1]; offsets[n] = the total (low 32 bits)
 *   n            0 <= n <= MLP_ROW_OFFSETS_STATIC_MAX, else MLP_ERR_ARG (nothing is launched)
 *   total        DEVICE long long, receives the 64-bit total; may be NULL
 *   cuda_stream  cudaStream_t (NULL = default stream); asynchronous, three kernel launches
 * Every call on a device shares the one array, which keeps the last call's contents (the call clears the one word that
 * must start at zero itself).  Calls that overlap on the GPU -- different streams, or host threads with no ordering
 * between their launches -- race on it: order them on one stream or with events.
 */
#define MLP_ROW_OFFSETS_STATIC_MAX 67108864LL
int mlp_row_offsets_static(const int* counts, int* offsets, long long n, long long* total, void* cuda_stream);

/*
 * mlp_debug_row_offsets -- the same step through the EXISTING path: the scan kernels mlp_compute launches (nbr.cu), with
 * a block buffer from cudaMalloc, on caller buffers.  Same arguments (total must not be NULL); synchronous.  Test hook.
 */
int mlp_debug_row_offsets(const int* counts, int* offsets, long long n, long long* total, void* cuda_stream);

/* mlp_last_error -- text of the last error on this model (static string when m == NULL). */
const char* mlp_last_error(mlp_model* m);

/* mlp_version -- static string "painn-b200 <semver> sm_100a". */
const char* mlp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PAINN_B200_MLP_H */
