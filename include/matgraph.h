/*
 * matgraph.h — C ABI of the B200-native periodic crystal-graph library (libmatgraph.so).
 *
 * What it computes (arxiv 2307.05380; line numbers refer to the paper text, PAPER.md):
 *   Def. 1  a material M = (rho, x, z): lattice rho in GL_3(R), fractional coordinates x.
 *   Def. 3  Gamma_1 = { (i, j, tau) in Gamma_0 x Gamma_0 x Z^3 : ||rho (x_j - x_i + tau)|| < c_i }
 *                     (the printed "x_i x_i" is read as x_j - x_i, R1).  A constant c_i is
 *                     the CUTOFF graph; c_i = distance of the k-th neighbour is the KNN graph.
 *   Alg. 1-2 the paper's expanding search + ordered stack: KNN keeps the k shortest
 *                     edges per source.  Here: exactly k per source, ties ordered by
 *                     (distance, dst, tau_x, tau_y, tau_z) (R2, R8).
 *   Batches of independent structures are processed together; the graph can be
 *   regenerated on the GPU after the model moved the atoms -> mg_update_graph.
 *
 * Conventions (R3, R5, R6, R9, R16):
 *   lattice   float32 [n_struct,3,3] row-major, ROWS are the lattice vectors a_1,a_2,a_3;
 *             cartesian = f . lattice[s].
 *   pos       float32 [n_atoms,3] FRACTIONAL coordinates; values outside [0,1) are legal, cell
 *             offsets are relative to the coordinates as given.
 *   struct_ptr int32 [n_struct+1], struct_ptr[0] = 0, struct_ptr[n_struct] = n_atoms; atoms of
 *             structure s are struct_ptr[s] .. struct_ptr[s+1]-1.  Empty structures are legal.
 *   edge (i, j, tau): src = i, dst = j are GLOBAL 0-based atom indices of the same structure,
 *             offset = tau (int8 x 3), vec = (pos[j] + tau - pos[i]) . lattice[s]  (Angstrom, float32,
 *             evaluated in FP64 and rounded once), dist = |vec|.  (i, i, 0) is never emitted;
 *             periodic self images (i, i, tau != 0) are.
 *   Output is CSR by source atom: row_ptr[i] .. row_ptr[i+1]-1 are the edges of source i.
 *             Cutoff rows: order inside a row unspecified.  KNN rows: exactly k entries, sorted by
 *             (distance, dst, tau lexicographic); row_ptr[i] = k*i.
 *
 * Pointers: every pointer argument named in an mg_edges or as pos / lattice / struct_ptr of a
 * non-_host call is a DEVICE pointer owned by the CALLER (e.g. a torch tensor); the library never
 * frees or keeps them past the call (mg_graph keeps struct_ptr, which must outlive the graph).
 * Calls are asynchronous on `cuda_stream` (a cudaStream_t, NULL = legacy default stream) and never
 * synchronise, except where stated.  Arguments are validated synchronously (MG_ERR_INVALID_ARG);
 * data-dependent failures (singular / non-finite lattice, |tau| > 127, more edges than
 * `capacity`, structure too large) are recorded in a device status word and returned by mg_check.
 * A structure with an invalid lattice emits no edges.  On capacity overflow row_ptr and *n_edges
 * still receive the full required count and only edges with index < capacity are written.
 * There is no CPU fallback: without a CUDA device every call fails with MG_ERR_CUDA.
 */
#ifndef MATGRAPH_H
#define MATGRAPH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_ctx mg_ctx;       /* opaque: device scratch workspace + status word        */
typedef struct mg_graph mg_graph;   /* opaque: a fixed (kind, r_c | k, struct_ptr) to update */

typedef enum {
    MG_OK = 0,
    MG_ERR_INVALID_ARG = 1,
    MG_ERR_CUDA = 2,
    MG_ERR_SINGULAR_LATTICE = 3,
    MG_ERR_NONFINITE = 4,
    MG_ERR_OFFSET_RANGE = 5,   /* a search box needs |tau| > 127 (int8 offsets)            */
    MG_ERR_CAPACITY = 6,       /* more edges than mg_edges.capacity (or than 2^31-1)       */
    MG_ERR_UNSUPPORTED = 7,    /* k or structure size outside what this build handles      */
    MG_ERR_TOO_LARGE = 8       /* mg_symmetrize_static: sizes beyond its static scratch    */
} mg_status;

enum { MG_KIND_CUTOFF = 0, MG_KIND_KNN = 1 };

typedef struct {
    int32_t *row_ptr;   /* [n_atoms+1]  CSR by source atom                                  */
    int32_t *src;       /* [capacity]   global source index                                 */
    int32_t *dst;       /* [capacity]   global target index                                 */
    int8_t  *offset;    /* [capacity,3] integer cell tau of the target image                */
    float   *vec;       /* [capacity,3] displacement rho (x_dst + tau - x_src), Angstrom    */
    float   *dist;      /* [capacity] or NULL                                               */
    int64_t  capacity;  /* edges the arrays can hold                                        */
    int64_t *n_edges;   /* one int64, written by the call                                   */
} mg_edges;

/* Context.  `device` is a CUDA ordinal.  mg_reserve grows the scratch workspace for batches of up
 * to (n_struct, n_atoms) outside the hot path; the graph calls grow it themselves when needed
 * (which allocates, hence is not capturable in a CUDA graph the first time).
 * Environment read by mg_create (diagnostics only; results do not depend on them):
 *   MATGRAPH_NO_PDL      launch the kernels without programmatic dependent launch;
 *   MATGRAPH_MASK_WORDS  words (0..4096) of the per-warp hit-mask scratch the cutoff count launch
 *                        may use (chunks of the code pool of the one-launch path); beyond it the masks are
 *                        evaluated / the rows listed a second time (tests);
 *   MATGRAPH_FUSED, MATGRAPH_LEGACY  force the one-launch / the two-launch cutoff kernels for every batch;
 *   MATGRAPH_WRITE_KERNEL  one-launch path: the edge arrays are written by a launch of their own (A/B variant);
 *   MATGRAPH_NO_COOP     one-launch path: plain instead of cooperative launch (its grid is sized to be resident);
 *   MG_DEBUG             print the CUDA error behind an MG_ERR_CUDA to stderr. */
mg_status mg_create(mg_ctx **ctx, int device);
void      mg_destroy(mg_ctx *ctx);
mg_status mg_reserve(mg_ctx *ctx, int32_t n_struct, int32_t n_atoms);

/* Cutoff graph, Def. 3 with constant c_i = r_c, strict '<'.  Stream-ordered, no host
 * synchronisation: a search-bounds launch (per structure n_a = ceil(r_c / h_a), h_a = V / |a_b x a_c|, the
 * per-pair sub-box inside that box, a cost prefix that cuts the batch into equal ranges), then image
 * enumeration with an FP32 distance filter (FP64 decision inside the rounding window, so that the edge SET
 * is Def. 3's in FP64) and K4's count -> device-wide scan -> emit, as one of two kernel sets chosen per
 * call: a count launch + an emit launch (batches of small cells), or one cooperative launch that finds,
 * scans across its resident CTAs and writes (batches of large structures; also mg_cutoff_graph_radii). */
mg_status mg_cutoff_graph(mg_ctx *ctx, const float *pos, const float *lattice,
                          const int32_t *struct_ptr, int32_t n_struct, int32_t n_atoms,
                          float r_c, const mg_edges *out, void *cuda_stream);

/* Def. 3 with one cutoff per SOURCE atom ("c_i > 0 for 1 <= i <= n"; e.g. covalent radii):
 * edge (i, j, tau) iff ||rho (x_j - x_i + tau)|| < radii[i], strict.  radii: device float32 [n_atoms].  Such a
 * graph is not symmetric in general.  A structure with a radius that is not a positive finite number emits
 * no edges and MG_ERR_UNSUPPORTED surfaces from mg_check.  Otherwise like mg_cutoff_graph. */
mg_status mg_cutoff_graph_radii(mg_ctx *ctx, const float *pos, const float *lattice,
                                const int32_t *struct_ptr, int32_t n_struct, int32_t n_atoms,
                                const float *radii, const mg_edges *out, void *cuda_stream);

/* Two-phase helper: number of edges mg_cutoff_graph would emit.  SYNCHRONISES the stream and
 * writes the count to HOST memory. */
mg_status mg_cutoff_count(mg_ctx *ctx, const float *pos, const float *lattice,
                          const int32_t *struct_ptr, int32_t n_struct, int32_t n_atoms,
                          float r_c, int64_t *n_edges_host, void *cuda_stream);

/* KNN graph (Alg. 1-2): exactly k edges per atom, periodic self images included,
 * rows sorted by (distance, dst, tau).  Needs out->capacity >= k * n_atoms.  1 <= k <= MG_MAX_K. */
#define MG_MAX_K 64
mg_status mg_knn_graph(mg_ctx *ctx, const float *pos, const float *lattice,
                       const int32_t *struct_ptr, int32_t n_struct, int32_t n_atoms,
                       int32_t k, const mg_edges *out, void *cuda_stream);

/* Dynamic geometry (R17).  mg_graph_create fixes kind, r_c or k and
 * struct_ptr (device pointer, kept), sizes the workspace and may synchronise.  mg_update_graph
 * regenerates the graph for new pos / lattice: no allocation, no host synchronisation, CUDA-graph
 * capturable; the result equals a fresh mg_cutoff_graph / mg_knn_graph on the same inputs
 * (state kept from the previous step only changes speed). */
mg_status mg_graph_create(mg_ctx *ctx, int kind, float r_c, int32_t k, const int32_t *struct_ptr,
                          int32_t n_struct, int32_t n_atoms, mg_graph **graph);
void      mg_graph_destroy(mg_graph *graph);
mg_status mg_update_graph(mg_ctx *ctx, mg_graph *graph, const float *pos, const float *lattice,
                          const mg_edges *out, void *cuda_stream);

/* HOST-buffer entry points: every pointer (inputs and the mg_edges arrays, n_edges included) is
 * HOST memory.  Copies the inputs to the device, runs the graph call, copies row_ptr, n_edges and
 * the first min(n_edges, capacity) edges back, and SYNCHRONISES.  Returns the device status. */
mg_status mg_cutoff_graph_host(mg_ctx *ctx, const float *pos, const float *lattice,
                               const int32_t *struct_ptr, int32_t n_struct, int32_t n_atoms,
                               float r_c, const mg_edges *out_host);
mg_status mg_knn_graph_host(mg_ctx *ctx, const float *pos, const float *lattice,
                            const int32_t *struct_ptr, int32_t n_struct, int32_t n_atoms,
                            int32_t k, const mg_edges *out_host);

/* Symmetric graph (section 3 "Symmetric graph"): the KNN graph is directed; `out` receives the
 * edges of `in` plus, for every edge (i, j, tau) whose reverse (j, i, -tau) is not in `in`, that reverse
 * edge (vec negated, same dist), CSR by source, every edge once.  The rows of `in` keep their order; the
 * added edges follow them in no particular order.  `in` is any graph this library produced (device
 * arrays, in->n_edges a device scalar; in->capacity bounds the edges read).  out->capacity must hold the
 * result (at most twice the edges of `in`), else MG_ERR_CAPACITY surfaces from mg_check with the required
 * count in *out->n_edges.  out->dist needs in->dist.  May grow the workspace on the first call.  An `in` whose
 * own call overflowed (*in->n_edges above in->capacity) is read up to in->capacity and reported as
 * MG_ERR_CAPACITY by mg_check. */
mg_status mg_symmetrize(mg_ctx *ctx, const mg_edges *in, int32_t n_atoms, const mg_edges *out, void *cuda_stream);

/* mg_symmetrize for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same operation on the same kernels, same arguments and results as mg_symmetrize, but it
 * needs no mg_ctx and calls no cudaMalloc / cudaFree / allocating library routine.  Its scratch (one flag
 * byte per input edge, two counters per atom, a status word) lives in ONE file-scope static device array
 * of about 4.5 MB that every GPU holds from the moment it loads the library until the process exits.
 *   limits   n_atoms <= MG_STATIC_MAX_ATOMS and in->capacity <= MG_STATIC_MAX_EDGES, else MG_ERR_TOO_LARGE
 *            (nothing is launched); out->capacity is the caller's and is not limited.
 *   device   the CUDA device the arrays live on; the call makes it current.  The first call on a device
 *            looks the array's address up (cudaGetSymbolAddress) and reads the SM count: make that call
 *            outside a stream capture.
 *   errors   no status word is reported: *out->n_edges always receives the required edge count, and a
 *            value above out->capacity means the result was cut off at the capacity (mg_check does not see
 *            this call).  An incomplete `in` (*in->n_edges above in->capacity) is read up to in->capacity.
 *   sharing  every call on a device uses the same array, which keeps the last call's contents; the call
 *            clears what must start at zero on `cuda_stream`.  Two calls that overlap on the GPU (different
 *            streams without an ordering between them, or a captured graph replayed concurrently with
 *            another call) race on it and give wrong graphs: order them. */
#define MG_STATIC_MAX_ATOMS 65536
#define MG_STATIC_MAX_EDGES 4194304
mg_status mg_symmetrize_static(int32_t device, const mg_edges *in, int32_t n_atoms, const mg_edges *out,
                               void *cuda_stream);

/* Triplets Gamma_2 (Def. 3; "Triplets generation"): the ordered pairs (a, b), a != b, of
 * edges that share their source.  For source i with edges row_ptr[i] .. row_ptr[i+1]-1 (degree d) the
 * d (d - 1) pairs are edge_a[t], edge_b[t] (edge indices) for tri_ptr[i] <= t < tri_ptr[i+1], ordered by
 * (a, b).  All pointers are device pointers; *n_triplets receives tri_ptr[n_atoms] (also when it exceeds
 * `capacity`: MG_ERR_CAPACITY from mg_check, only triplets below the capacity are written).  Keeps one
 * partial sum per 8192 atoms in the context: may grow the workspace on the first call (mg_reserve covers it). */
typedef struct {
    int64_t *tri_ptr;      /* [n_atoms+1]                                        */
    int32_t *edge_a;       /* [capacity] first edge of the pair                  */
    int32_t *edge_b;       /* [capacity] second edge                             */
    int64_t  capacity;
    int64_t *n_triplets;   /* one int64, written by the call                     */
} mg_triplets;
mg_status mg_triplets_graph(mg_ctx *ctx, const int32_t *row_ptr, int32_t n_atoms, const mg_triplets *out,
                            void *cuda_stream);

/* SYNCHRONISES the stream, returns the first data-dependent error recorded since the last
 * mg_check (MG_OK if none) and clears the device status word. */
mg_status mg_check(mg_ctx *ctx, void *cuda_stream);

/* Number of kernels this library launched on behalf of ctx since mg_create (bench bookkeeping). */
int64_t mg_launch_count(const mg_ctx *ctx);

/* Profiling aid.  mg_set_profile(ctx, 1): every following mg_cutoff_graph / mg_knn_graph /
 * mg_update_graph call brackets its kernels with CUDA events on the caller's stream (a few event
 * records per call; off by default).  mg_profile_read SYNCHRONISES on the last recorded event and
 * returns the mean duration in milliseconds of [0] the search-bounds kernel (K1), [1] the cutoff
 * count kernel, [2] the cutoff emit kernel, [3] the KNN kernel over the calls made since
 * mg_set_profile, and how many calls each mean covers (count4 may be NULL). */
mg_status mg_set_profile(mg_ctx *ctx, int on);
mg_status mg_profile_read(mg_ctx *ctx, double *mean_ms4, int64_t *count4);

const char *mg_status_string(mg_status status);

#ifdef __cplusplus
}
#endif
#endif /* MATGRAPH_H */
