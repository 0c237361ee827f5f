// matgraph.cu — C ABI of libmatgraph (include/matgraph.h): argument checks, workspace, launches.
// No torch types, no CPU fallback: every graph is produced by the sm_100a kernels in this
// directory.
#include "../../include/matgraph.h"

#include <cuda_runtime.h>
#include <math.h>
#include <mutex>
#include <new>
#include <stdlib.h>
#include <string.h>

#include "common.cuh"
#include "prep.cuh"
#include "cut_prep.cuh"
#include "cutoff_pairs.cuh"
#include "cut_scan.cuh"
#include "knn_small.cuh"
#include "knn_pairs.cuh"
#include "graph_ops.cuh"

// the pair-lane KNN kernel for k > 16 is a module of its own (knn_large.cu)
cudaError_t mg_knn_large_setup(int *occ);
cudaError_t mg_knn_large_launch(const void *args, size_t args_bytes, int grid, cudaStream_t st, int pdl);
// ... and so is the KNN kernel for batches of large structures (knn_bins.cu)
#include "knn_bins_args.cuh"
cudaError_t mg_knn_bins_setup(int *occ);
cudaError_t mg_knn_bins_launch(const KnnBinsArgs *a, int grid, cudaStream_t st, int pdl);

struct mg_ctx {
    int device = 0;
    int sm_count = 0;
    unsigned *d_ctl = nullptr;            // [0..1] cutoff ticket/done, [2..3] knn ticket/done, [4] status,
                                          // [5] knn prep blocks done, [6] number of cutoff tasks, [7] cut-prep block ticket, [8..9] cutoff emit ticket/done
    StructRec *d_rec = nullptr;           // per-structure records (prep.cuh)
    size_t rec_cap = 0;
    int32_t *d_atom_struct = nullptr;     // [n_atoms]
    size_t atom_cap = 0;
    unsigned *d_wtotal = nullptr;         // [n_warps + 1] cutoff edges per warp / their exclusive scan, [64] group totals
    int2 *d_wstart = nullptr;             // [n_warps] first (structure, pair) of each warp's range
    unsigned *d_wclock = nullptr;         // [2, n_warps] per-warp cycles of the last cutoff call
    int mask_words = 0;                   // usable words of a range's mask scratch (MATGRAPH_MASK_WORDS)
    unsigned *d_wmask = nullptr;          // [n_warps, MG_MASK_WORDS] hit masks kept from count to emit
    int cut_warps = 0, last_cut_warps = 0;
    int fused_occ = 0, fused_coop = 0;    // fused cutoff kernel: CTAs per SM, cooperative launch accepted
    int force_scan = 0, force_legacy = 0; // MATGRAPH_FUSED=1 / MATGRAPH_LEGACY=1: one cutoff path for every batch
    int write_kernel = 0;                 // MATGRAPH_WRITE_KERNEL=1: edges written by a launch of their own
    unsigned long long *d_slots = nullptr;// [sm_count * fused_occ] per-CTA edge totals tagged with the call's epoch
    uint2 *d_pool = nullptr;              // [pool_chunks, MGS_CHUNK] codes before their final place is known
    size_t pool_chunks = 0;
    // products of the scan kernel for the write kernel (cut_scan.cuh)
    uint2 *d_codes = nullptr;             // [code_cap] (dst, tau) of every edge, in output order
    int4 *d_slice_row = nullptr;          // [code_cap / MGS_SLICE + 2]
    size_t code_cap = 0;
    float4 *d_xw4 = nullptr;              // [atom64_cap] wrapped coordinates (cut_prep.cuh)
    float4 *d_xs4 = nullptr;              // [atom64_cap] ... in bin order (cut_bins.cuh)
    int *d_binstart = nullptr;            // [bin_cap] first entry of each bin
    int *d_binlist = nullptr;             // [crec_cap] structures with a cell list (written by the prep kernel)
    size_t bin_cap = 0;
    double *d_pos64 = nullptr;            // [atom64_cap, 4]
    size_t atom64_cap = 0;
    double *d_lat64 = nullptr;            // [lat64_cap, 9]
    size_t lat64_cap = 0;
    int write_occ = 0;
    // scratch of mg_symmetrize (graph_ops.cuh)
    unsigned char *d_symflag = nullptr;   // [symflag_cap]
    size_t symflag_cap = 0;
    int *d_symcnt = nullptr;              // [2, symcnt_cap] missing reverse edges per row, append cursors
    size_t symcnt_cap = 0;
    long long *d_scanpart = nullptr;      // [scanpart_cap] chunk totals of the scans of graph_ops.cuh
    size_t scanpart_cap = 0;
    CutRec *d_crec = nullptr;             // per-structure records of the cutoff path (cut_prep.cuh)
    unsigned long long *d_bpre = nullptr; // cost prefix over the prep blocks
    size_t crec_cap = 0;
    int32_t *d_rowptr_tmp = nullptr;      // for mg_cutoff_count
    size_t rowptr_cap = 0;
    long long *d_count = nullptr;
    int cutoff_occ = 0, count_occ = 0, knn_occ[2] = {0, 0}, knnp_occ = 0, knnb_occ = 0;
    int64_t launches = 0;
    int pdl = 1;                          // programmatic dependent launch (MATGRAPH_NO_PDL=1 turns it off)
    int profile = 0;                      // mg_set_profile: events around the kernels of the next calls
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    double prof_ms[4] = {0, 0, 0, 0};     // accumulated: prep, count, emit, knn
    int64_t prof_n[4] = {0, 0, 0, 0};
    int pend_kind = -1;                   // events of the last call not read yet: 0 cutoff, 1 knn
    // device mirrors for the _host entry points
    void *h_dev[9] = {nullptr};
    size_t h_cap[9] = {0};
};

struct mg_graph {
    mg_ctx *ctx;
    int kind;
    float r_c;
    int32_t k;
    const int32_t *struct_ptr;
    int32_t n_struct, n_atoms;
    float *d_hint = nullptr;
    int have_hint = 0;
};

#include <stdio.h>
#define MG_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { if (getenv("MG_DEBUG")) fprintf(stderr, "[matgraph] %s:%d %s\n", __FILE__, __LINE__, cudaGetErrorString(e_)); cudaGetLastError(); return MG_ERR_CUDA; } } while (0)

static mg_status decode_status(unsigned bits) {
    if (bits & MGS_NONFINITE) return MG_ERR_NONFINITE;
    if (bits & MGS_SINGULAR) return MG_ERR_SINGULAR_LATTICE;
    if (bits & MGS_OFFSET) return MG_ERR_OFFSET_RANGE;
    if (bits & MGS_UNSUPPORTED) return MG_ERR_UNSUPPORTED;
    if (bits & MGS_CAPACITY) return MG_ERR_CAPACITY;
    return MG_OK;
}

extern "C" const char *mg_status_string(mg_status s) {
    switch (s) {
        case MG_OK: return "ok";
        case MG_ERR_INVALID_ARG: return "invalid argument";
        case MG_ERR_CUDA: return "CUDA error (no device, launch or allocation failure)";
        case MG_ERR_SINGULAR_LATTICE: return "singular lattice";
        case MG_ERR_NONFINITE: return "non-finite lattice or position";
        case MG_ERR_OFFSET_RANGE: return "search box needs |tau| > 127";
        case MG_ERR_CAPACITY: return "edge capacity exceeded";
        case MG_ERR_UNSUPPORTED: return "unsupported k or structure size";
        case MG_ERR_TOO_LARGE: return "more atoms or edges than the static scratch of mg_symmetrize_static holds";
    }
    return "unknown status";
}

extern "C" mg_status mg_create(mg_ctx **out, int device) {
    if (!out) return MG_ERR_INVALID_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return MG_ERR_CUDA;
    }
    MG_CUDA(cudaSetDevice(device));
    mg_ctx *c = new (std::nothrow) mg_ctx();
    if (!c) return MG_ERR_CUDA;
    c->device = device;
    c->pdl = getenv("MATGRAPH_NO_PDL") ? 0 : 1;
    // test knob: a smaller mask scratch per range makes the emit launch evaluate masks again
    c->mask_words = MG_MASK_WORDS;
    if (const char *mw = getenv("MATGRAPH_MASK_WORDS")) {
        const int v = atoi(mw);
        if (v >= 0 && v <= MG_MASK_WORDS) c->mask_words = v;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess || prop.major < 10) { delete c; return MG_ERR_CUDA; }
    c->sm_count = prop.multiProcessorCount;
    if (cudaMalloc(&c->d_ctl, 16 * sizeof(unsigned)) != cudaSuccess ||
        cudaMemset(c->d_ctl, 0, 16 * sizeof(unsigned)) != cudaSuccess ||
        cudaMalloc(&c->d_count, sizeof(long long)) != cudaSuccess) { mg_destroy(c); return MG_ERR_CUDA; }
    if (cudaFuncSetAttribute(mg_cutoff_emit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(MG_WARPS * sizeof(EmitSmem))) != cudaSuccess) { mg_destroy(c); return MG_ERR_CUDA; }
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->cutoff_occ, mg_cutoff_emit_kernel, MG_BLOCK, (MG_WARPS * sizeof(EmitSmem)));
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->count_occ, mg_cutoff_count_kernel, MG_BLOCK, 0);
    if (cudaFuncSetAttribute(mg_knn_pairs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)(MG_WARPS * sizeof(KnnSmem))) != cudaSuccess) { mg_destroy(c); return MG_ERR_CUDA; }
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->knnp_occ, mg_knn_pairs_kernel, MG_BLOCK, (MG_WARPS * sizeof(KnnSmem)));
    {                                       // the kernel for k > 16 (knn_large.cu): the same grid for both
        int occ_l = 0;
        if (mg_knn_large_setup(&occ_l) != cudaSuccess || occ_l < 1) { mg_destroy(c); return MG_ERR_CUDA; }
        if (occ_l < c->knnp_occ) c->knnp_occ = occ_l;
        if (mg_knn_bins_setup(&c->knnb_occ) != cudaSuccess || c->knnb_occ < 1) { mg_destroy(c); return MG_ERR_CUDA; }
    }
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->knn_occ[0], mg_knn_small_kernel<1>, MG_BLOCK, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->knn_occ[1], mg_knn_small_kernel<2>, MG_BLOCK, 0);
    {
        const int occ = c->cutoff_occ < c->count_occ ? c->cutoff_occ : c->count_occ;
        c->cut_warps = c->sm_count * occ * MG_WARPS;
        if (occ >= 1 && (cudaMalloc(&c->d_wtotal, (MG_OVER * c->cut_warps + 1 + 64) * sizeof(unsigned)) != cudaSuccess ||
                         cudaMemset(c->d_wtotal, 0, (MG_OVER * c->cut_warps + 1 + 64) * sizeof(unsigned)) != cudaSuccess ||
                         cudaMalloc(&c->d_wstart, MG_OVER * c->cut_warps * sizeof(int2)) != cudaSuccess ||
                         cudaMalloc(&c->d_wmask, (size_t)MG_OVER * c->cut_warps * MG_MASK_WORDS * sizeof(unsigned)) != cudaSuccess ||
                         cudaMalloc(&c->d_wclock, 64 * (size_t)(c->cut_warps + 2048) * sizeof(unsigned)) != cudaSuccess)) { mg_destroy(c); return MG_ERR_CUDA; }
    }
    c->write_kernel = getenv("MATGRAPH_WRITE_KERNEL") ? 1 : 0;
    c->force_scan = getenv("MATGRAPH_FUSED") ? 1 : 0;
    c->force_legacy = getenv("MATGRAPH_LEGACY") ? 1 : 0;
    if (cudaFuncSetAttribute(mg_cutoff_scan_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)sizeof(ScanSmem)) != cudaSuccess ||
        cudaFuncSetAttribute(mg_cutoff_scan_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)sizeof(ScanSmem)) != cudaSuccess) { mg_destroy(c); return MG_ERR_CUDA; }
    {                                       // both instances run with the same grid: the smaller of their occupancies
        int occ_b = 0, occ_p = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_b, mg_cutoff_scan_kernel<true>, MGS_BLOCK, sizeof(ScanSmem));
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_p, mg_cutoff_scan_kernel<false>, MGS_BLOCK, sizeof(ScanSmem));
        c->fused_occ = occ_b < occ_p ? occ_b : occ_p;
    }
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->write_occ, mg_cutoff_write_kernel, MGWR_BLOCK, 0);
    if (c->fused_occ < 1 || c->write_occ < 1) { mg_destroy(c); return MG_ERR_CUDA; }
    {
        const size_t nc = (size_t)c->sm_count * c->fused_occ * MGS_WAVES;
        if (cudaMalloc(&c->d_slots, nc * sizeof(unsigned long long)) != cudaSuccess ||
            cudaMemset(c->d_slots, 0, nc * sizeof(unsigned long long)) != cudaSuccess ||
            false) { mg_destroy(c); return MG_ERR_CUDA; }
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device);
        c->fused_coop = coop && !getenv("MATGRAPH_NO_COOP");
    }
    if (c->cutoff_occ < 1 || c->count_occ < 1 || c->knnp_occ < 1 || c->knn_occ[0] < 1 || c->knn_occ[1] < 1) { mg_destroy(c); return MG_ERR_CUDA; }
    *out = c;
    return MG_OK;
}

extern "C" void mg_destroy(mg_ctx *c) {
    if (!c) return;
    cudaSetDevice(c->device);
    cudaFree(c->d_ctl);
    cudaFree(c->d_wtotal);
    cudaFree(c->d_wstart);
    cudaFree(c->d_wmask);
    cudaFree(c->d_wclock);
    cudaFree(c->d_slots);
    cudaFree(c->d_symflag);
    cudaFree(c->d_symcnt);
    cudaFree(c->d_scanpart);
    cudaFree(c->d_pool);
    cudaFree(c->d_codes);
    cudaFree(c->d_slice_row);
    cudaFree(c->d_pos64);
    cudaFree(c->d_xw4);
    cudaFree(c->d_xs4);
    cudaFree(c->d_binstart);
    cudaFree(c->d_binlist);
    cudaFree(c->d_lat64);
    cudaFree(c->d_crec);
    cudaFree(c->d_bpre);
    cudaFree(c->d_rec);
    cudaFree(c->d_atom_struct);
    cudaFree(c->d_rowptr_tmp);
    cudaFree(c->d_count);
    for (int i = 0; i < 9; ++i) cudaFree(c->h_dev[i]);
    for (int i = 0; i < 5; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    delete c;
}

extern "C" mg_status mg_reserve(mg_ctx *c, int32_t n_struct, int32_t n_atoms) {
    if (!c || n_struct < 0 || n_atoms < 0) return MG_ERR_INVALID_ARG;
    MG_CUDA(cudaSetDevice(c->device));
    if ((size_t)n_struct + 1 > c->crec_cap) {
        const size_t cap = (size_t)n_struct + 1025;
        cudaFree(c->d_crec); cudaFree(c->d_bpre); cudaFree(c->d_binlist);
        c->d_crec = nullptr; c->d_bpre = nullptr; c->d_binlist = nullptr; c->crec_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_crec, cap * sizeof(CutRec)));
        MG_CUDA(cudaMalloc(&c->d_binlist, cap * sizeof(int)));
        MG_CUDA(cudaMalloc(&c->d_bpre, (cap / MG_CP_BLOCK + 3) * sizeof(unsigned long long)));
        c->crec_cap = cap;
    }
    if ((size_t)n_struct + 1 > c->rec_cap) {
        const size_t cap = (size_t)n_struct + 1025;
        cudaFree(c->d_rec);
        c->d_rec = nullptr; c->rec_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_rec, cap * sizeof(StructRec)));
        c->rec_cap = cap;
    }
    if ((size_t)n_atoms + 1 > c->atom_cap) {
        const size_t cap = (size_t)n_atoms + 1025;
        cudaFree(c->d_atom_struct);
        c->d_atom_struct = nullptr; c->atom_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_atom_struct, cap * sizeof(int32_t)));
        c->atom_cap = cap;
    }
    if ((size_t)n_atoms + 1 > c->atom64_cap) {
        const size_t cap = (size_t)n_atoms + 1025;
        cudaFree(c->d_pos64); cudaFree(c->d_xw4); cudaFree(c->d_xs4);
        c->d_pos64 = nullptr; c->d_xw4 = nullptr; c->d_xs4 = nullptr; c->atom64_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_pos64, cap * 4 * sizeof(double)));
        MG_CUDA(cudaMalloc(&c->d_xw4, cap * sizeof(float4)));
        MG_CUDA(cudaMalloc(&c->d_xs4, cap * sizeof(float4)));
        c->atom64_cap = cap;
    }
    if ((size_t)n_atoms + 2 * (size_t)n_struct + 2 > c->bin_cap) {
        const size_t cap = (size_t)n_atoms + 2 * (size_t)n_struct + 4098;
        cudaFree(c->d_binstart);
        c->d_binstart = nullptr; c->bin_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_binstart, cap * sizeof(int)));
        c->bin_cap = cap;
    }
    if ((size_t)n_struct + 1 > c->lat64_cap) {
        const size_t cap = (size_t)n_struct + 1025;
        cudaFree(c->d_lat64);
        c->d_lat64 = nullptr; c->lat64_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_lat64, cap * 9 * sizeof(double)));
        c->lat64_cap = cap;
    }
    if ((size_t)mgo_scan_blocks(n_atoms) > c->scanpart_cap) {
        const size_t cap = (size_t)mgo_scan_blocks(n_atoms) + 64;
        cudaFree(c->d_scanpart);
        c->d_scanpart = nullptr; c->scanpart_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_scanpart, cap * sizeof(long long)));
        c->scanpart_cap = cap;
    }
    if ((size_t)n_atoms + 1 > c->rowptr_cap) {
        const size_t cap = (size_t)n_atoms + 1025;
        cudaFree(c->d_rowptr_tmp);
        c->d_rowptr_tmp = nullptr; c->rowptr_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_rowptr_tmp, cap * sizeof(int32_t)));
        c->rowptr_cap = cap;
    }
    return MG_OK;
}

#ifdef MG_PHASE_CLOCKS
// Tuning aid (not part of the public header): per-warp cycles and range starts of the last cutoff call.
extern "C" int mg_debug_cut_warps(mg_ctx *c, unsigned *clocks_host, int *starts_host, int max_warps) {
    if (!c) return -1;
    cudaDeviceSynchronize();
    const int n = c->last_cut_warps < max_warps ? c->last_cut_warps : max_warps;
    if (n > 0) {
        cudaMemcpy(clocks_host, c->d_wclock, (size_t)n * 4, cudaMemcpyDeviceToHost);
        cudaMemcpy(clocks_host + max_warps, c->d_wclock + c->last_cut_warps, (size_t)n * 4, cudaMemcpyDeviceToHost);
        cudaMemcpy(starts_host, c->d_wstart, (size_t)n * 8, cudaMemcpyDeviceToHost);
    }
    return c->last_cut_warps;
}

extern "C" int mg_debug_clock_words(mg_ctx *c, unsigned *host, int n_words) {
    if (!c) return -1;
    cudaDeviceSynchronize();
    cudaMemcpy(host, c->d_wclock, (size_t)n_words * 4, cudaMemcpyDeviceToHost);
    return c->cut_warps;
}

extern "C" int mg_debug_cut_masks(mg_ctx *c, unsigned *host, int n_words) {
    if (!c) return -1;
    cudaDeviceSynchronize();
    cudaMemcpy(host, c->d_wmask, (size_t)n_words * 4, cudaMemcpyDeviceToHost);
    return 0;
}

#endif

extern "C" int64_t mg_launch_count(const mg_ctx *c) { return c ? c->launches : 0; }

static bool bad_inputs(const mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                       int32_t n_struct, int32_t n_atoms) {
    if (!c || n_struct < 0 || n_atoms < 0 || !sp) return true;
    if (n_struct > 0 && !lat) return true;
    if (n_atoms > 0 && !pos) return true;
    return false;
}

static bool bad_edges(const mg_edges *o, long long need) {
    if (!o || !o->row_ptr || !o->n_edges || o->capacity < 0) return true;
    if (o->capacity > 0 && (!o->src || !o->dst || !o->offset || !o->vec)) return true;
    return o->capacity < need;
}

// Profiling aid: with mg_set_profile(ctx, 1) every graph call brackets its kernels with CUDA events on
// the caller's stream; the durations are collected at the next call (or mg_profile_read).
static void prof_collect(mg_ctx *c) {
    if (c->pend_kind < 0) return;
    if (cudaEventSynchronize(c->ev[3]) == cudaSuccess) {
        float ms = 0.f;
        if (c->pend_kind == 0) {
            for (int i = 0; i < 3; ++i)
                if (cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]) == cudaSuccess) { c->prof_ms[i] += ms; c->prof_n[i] += 1; }
        } else {
            if (cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]) == cudaSuccess) { c->prof_ms[0] += ms; c->prof_n[0] += 1; }
            if (cudaEventElapsedTime(&ms, c->ev[1], c->ev[3]) == cudaSuccess) { c->prof_ms[3] += ms; c->prof_n[3] += 1; }
        }
    }
    cudaGetLastError();
    c->pend_kind = -1;
}

extern "C" mg_status mg_set_profile(mg_ctx *c, int on) {
    if (!c) return MG_ERR_INVALID_ARG;
    MG_CUDA(cudaSetDevice(c->device));
    prof_collect(c);
    if (on && !c->ev[0])
        for (int i = 0; i < 5; ++i) MG_CUDA(cudaEventCreate(&c->ev[i]));
    c->profile = on ? 1 : 0;
    for (int i = 0; i < 4; ++i) { c->prof_ms[i] = 0; c->prof_n[i] = 0; }
    return MG_OK;
}

extern "C" mg_status mg_profile_read(mg_ctx *c, double *mean_ms4, int64_t *count4) {
    if (!c || !mean_ms4) return MG_ERR_INVALID_ARG;
    MG_CUDA(cudaSetDevice(c->device));
    prof_collect(c);
    for (int i = 0; i < 4; ++i) {
        mean_ms4[i] = c->prof_n[i] ? c->prof_ms[i] / (double)c->prof_n[i] : 0.0;
        if (count4) count4[i] = c->prof_n[i];
    }
    return MG_OK;
}

// Launch a kernel that consumes the output of the kernel before it on the same stream with
// programmatic dependent launch: its CTAs may be scheduled while the producer drains and wait in
// mg_grid_dependency_wait() (common.cuh), which hides the launch latency of the dependent kernel.
template <class Args>
static cudaError_t launch_after(mg_ctx *c, void (*kern)(const Args), int grid, int block, size_t smem,
                                cudaStream_t st, const Args &a, bool cooperative = false) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    int n = 0;
    if (c->pdl) {
        at[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[n].val.programmaticStreamSerializationAllowed = 1;
        ++n;
    }
    if (cooperative) {                     // all CTAs resident at once: they wait on one another's slots
        at[n].id = cudaLaunchAttributeCooperative;
        at[n].val.cooperative = 1;
        ++n;
    }
    cfg.attrs = at;
    cfg.numAttrs = n;
    return cudaLaunchKernelEx(&cfg, kern, a);
}

static mg_status launch_prep(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                             int32_t n_struct, int32_t n_atoms, float r_c, cudaStream_t st) {
    PrepArgs P;
    P.pos = pos; P.lattice = lat; P.struct_ptr = sp; P.n_struct = n_struct; P.n_atoms = n_atoms;
    P.rec = c->d_rec; P.atom_struct = c->d_atom_struct; P.status = c->d_ctl + 4;
    mg_prep_kernel<<<(n_struct + MG_PREP_BLOCK / 32 - 1) / (MG_PREP_BLOCK / 32), MG_PREP_BLOCK, 0, st>>>(P);
    MG_CUDA(cudaGetLastError());
    c->launches += 1;
    return MG_OK;
}

static mg_status launch_cutoff(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                               int32_t n_struct, int32_t n_atoms, float r_c, const mg_edges *o,
                               int count_only, cudaStream_t st, const float *radii = nullptr) {
    MG_CUDA(cudaSetDevice(c->device));
    mg_status rs = mg_reserve(c, n_struct, n_atoms);
    if (rs != MG_OK) return rs;
    if (n_struct == 0) {
        MG_CUDA(cudaMemsetAsync(o->row_ptr, 0, sizeof(int32_t), st));
        MG_CUDA(cudaMemsetAsync(o->n_edges, 0, sizeof(long long), st));
        return MG_OK;
    }
    const int n_blocks = (n_struct + MG_CP_BLOCK - 1) / MG_CP_BLOCK;
    const bool prof = c->profile && !count_only;
    // Two cutoff paths: the scan kernel (cut_scan.cuh) and the count + emit pair (cutoff_pairs.cuh).  The pair is
    // ahead on batches of small cells (BASELINE configs[2]: 73 against 81 us per call), the scan kernel on large
    // structures; MATGRAPH_FUSED=1 / MATGRAPH_LEGACY=1 force one of them.
    const bool use_scan = radii || c->force_scan || (!c->force_legacy && n_struct > 0 && n_atoms / n_struct > MG_SMALL_MAX_ATOMS);
    // ... and the scan kernel in its instance with cell lists (cut_bins.cuh) for batches of large structures; the other
    // instance takes a large structure among small ones by its generic rows
    const bool use_bins = use_scan && n_atoms / n_struct > MG_SMALL_MAX_ATOMS;
    if (prof) { prof_collect(c); cudaEventRecord(c->ev[0], st); }
    {
        CutPrepArgs P;
        P.lattice = lat; P.struct_ptr = sp; P.n_struct = n_struct; P.n_atoms = n_atoms; P.r_c = r_c;
        P.k = 0; P.hint = nullptr; P.use_hint = 0; P.rows_cost = use_scan ? 1 : 0;
        P.pos = pos; P.xw4 = use_scan ? c->d_xw4 : nullptr; P.n_sblocks = n_blocks; P.radii = radii;
        P.binlist = use_bins ? c->d_binlist : nullptr;     // (NULL: no structure gets a cell list)
        P.rec = c->d_crec; P.bpre = c->d_bpre; P.ctl = c->d_ctl; P.status = c->d_ctl + 4;
        // (scan path: extra blocks wrap the coordinates of the batch's atoms)
        const int xblocks = use_scan ? (n_atoms + 8 * MG_CP_BLOCK - 1) / (8 * MG_CP_BLOCK) : 0;
        MG_CUDA(launch_after(c, mg_cut_prep_kernel, n_blocks + (xblocks < 1024 ? xblocks : 1024), MG_CP_BLOCK, 0, st, P));
        c->launches += 1;
    }
    if (use_scan) {
        // the code stream holds one 8-byte code per edge the caller's arrays can take
        const size_t need = count_only ? 0 : (size_t)o->capacity;
        if (c->write_kernel && need > c->code_cap) {
            cudaFree(c->d_codes); cudaFree(c->d_slice_row);
            c->d_codes = nullptr; c->d_slice_row = nullptr; c->code_cap = 0;
            const size_t cap = need + need / 8 + 4096;
            MG_CUDA(cudaMalloc(&c->d_codes, cap * sizeof(uint2)));
            MG_CUDA(cudaMalloc(&c->d_slice_row, (cap / MGS_SLICE + 2) * sizeof(int4)));
            c->code_cap = cap;
        }
        int grid = c->sm_count * c->fused_occ;
        const int cap_grid = (n_atoms + MGS_WARPS * MGS_WAVES) / (MGS_WARPS * MGS_WAVES);   // >= 1 row per range
        if (grid > cap_grid) grid = cap_grid;
        // pool: the edges the caller can take, in chunks, plus one partly filled chunk per warp
        const size_t want_chunks = count_only ? 0 : need / MGS_CHUNK + (size_t)grid * MGS_WARPS * MGS_WAVES + 8;
        if (want_chunks > c->pool_chunks) {
            cudaFree(c->d_pool);
            c->d_pool = nullptr; c->pool_chunks = 0;
            const size_t cap = want_chunks + want_chunks / 8;
            MG_CUDA(cudaMalloc(&c->d_pool, cap * MGS_CHUNK * sizeof(uint2)));
            c->pool_chunks = cap;
        }
        if (use_bins) {                     // K2: the cell lists of the large structures (cut_bins.cuh)
            BinArgs B;
            B.rec = c->d_crec; B.xw4 = c->d_xw4; B.xs4 = c->d_xs4; B.bin_start = c->d_binstart;
            B.n_struct = n_struct; B.binlist = c->d_binlist; B.ctl = c->d_ctl;
            const int bgrid = n_struct < 2 * c->sm_count ? n_struct : 2 * c->sm_count;
            MG_CUDA(launch_after(c, mg_cut_bin_kernel, bgrid, MGB_BLOCK, 0, st, B));
            c->launches += 1;
        }
        ScanArgs F;
        F.xs4 = c->d_xs4; F.bin_start = c->d_binstart;
        F.pos = pos; F.lattice = lat; F.xw4 = c->d_xw4; F.n_struct = n_struct; F.n_atoms = n_atoms; F.radii = radii;
        F.row_ptr = o->row_ptr; F.capacity = o->capacity; F.n_edges = (long long *)o->n_edges;
        F.rec = c->d_crec; F.bpre = c->d_bpre; F.n_blocks = n_blocks;
        F.pool = c->d_pool;
        // (test knob MATGRAPH_MASK_WORDS < 4096: a pool this small, so that warps list their rows again)
        F.n_pool = count_only ? 0 : (c->mask_words < MG_MASK_WORDS ? c->mask_words : (int)(c->pool_chunks < 0x7FFFFFFF ? c->pool_chunks : 0x7FFFFFFF));
        F.slots = c->d_slots; F.ctl = c->d_ctl; F.status = c->d_ctl + 4;
        F.count_only = count_only;
        F.src = o->src; F.dst = o->dst; F.offset = o->offset; F.vec = o->vec; F.dist = o->dist;
        F.write_here = c->write_kernel ? 0 : 1;
        F.codes = c->d_codes; F.slice_row = c->d_slice_row; F.atom_struct = c->d_atom_struct;
        F.pos64 = c->d_pos64; F.lat64 = c->d_lat64;
        F.dbg = c->d_wclock;
        if (prof) cudaEventRecord(c->ev[1], st);
        void (*scan_kernel)(const ScanArgs) = use_bins ? mg_cutoff_scan_kernel<true> : mg_cutoff_scan_kernel<false>;
        cudaError_t e = launch_after(c, scan_kernel, grid, MGS_BLOCK, sizeof(ScanSmem), st, F, c->fused_coop != 0);
        if (e != cudaSuccess && c->fused_coop) {        // cooperative + programmatic launch refused together
            cudaGetLastError();
            c->fused_coop = 0;
            e = launch_after(c, scan_kernel, grid, MGS_BLOCK, sizeof(ScanSmem), st, F, false);
        }
        MG_CUDA(e);
        c->launches += 1;
        if (prof) cudaEventRecord(c->ev[2], st);
        if (!count_only && o->capacity > 0 && c->write_kernel) {
            WriteArgs W;
            W.codes = c->d_codes; W.slice_row = c->d_slice_row; W.atom_struct = c->d_atom_struct;
            W.pos64 = c->d_pos64; W.lat64 = c->d_lat64; W.row_ptr = o->row_ptr;
            W.n_edges = (const long long *)o->n_edges; W.n_atoms = n_atoms; W.capacity = o->capacity;
            W.src = o->src; W.dst = o->dst; W.offset = o->offset; W.vec = o->vec; W.dist = o->dist;
            const long long n_slices = (o->capacity + MGS_SLICE - 1) / MGS_SLICE;
            long long wgrid = (n_slices + MGWR_BLOCK / 32 - 1) / (MGWR_BLOCK / 32);
            const long long wmax = (long long)c->sm_count * c->write_occ;
            if (wgrid > wmax) wgrid = wmax;
            MG_CUDA(launch_after(c, mg_cutoff_write_kernel, (int)wgrid, MGWR_BLOCK, 0, st, W));
            c->launches += 1;
        }
        if (prof) { cudaEventRecord(c->ev[3], st); c->pend_kind = 0; }
        return MG_OK;
    }
    CutoffArgs A;
    A.pos = pos; A.lattice = lat;
    A.n_struct = n_struct; A.n_atoms = n_atoms; A.r_c = r_c;
    A.row_ptr = o->row_ptr; A.src = o->src; A.dst = o->dst; A.offset = o->offset;
    A.vec = o->vec; A.dist = o->dist; A.capacity = o->capacity; A.n_edges = (long long *)o->n_edges;
    A.rec = c->d_crec; A.bpre = c->d_bpre; A.n_blocks = n_blocks;
    A.wtotal = c->d_wtotal; A.gtotal = c->d_wtotal + MG_OVER * c->cut_warps + 1; A.wstart = c->d_wstart; A.wmask = c->d_wmask; A.mask_words = c->mask_words; A.wclock = c->d_wclock;
    A.ctl = c->d_ctl; A.status = c->d_ctl + 4;
    A.count_only = count_only;
    // one contiguous range of rows per warp; small batches use fewer warps (>= 1 row each)
    int grid = c->cut_warps / MG_WARPS;
    const int cap_grid = (n_atoms + MG_WARPS) / MG_WARPS;
    if (grid > cap_grid) grid = cap_grid;
    A.n_warps = grid * MG_WARPS;
    A.n_ranges = MG_OVER * A.n_warps;
    c->last_cut_warps = A.n_warps;
    if (prof) cudaEventRecord(c->ev[1], st);
    MG_CUDA(launch_after(c, mg_cutoff_count_kernel, grid, MG_BLOCK, 0, st, A));
    c->launches += 1;
    if (prof) cudaEventRecord(c->ev[2], st);
    if (!count_only) {
        MG_CUDA(launch_after(c, mg_cutoff_emit_kernel, grid, MG_BLOCK, MG_WARPS * sizeof(EmitSmem), st, A));
        c->launches += 1;
    }
    if (prof) { cudaEventRecord(c->ev[3], st); c->pend_kind = 0; }
    return MG_OK;
}

extern "C" mg_status mg_cutoff_graph(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                                     int32_t n_struct, int32_t n_atoms, float r_c, const mg_edges *o,
                                     void *stream) {
    if (bad_inputs(c, pos, lat, sp, n_struct, n_atoms) || bad_edges(o, 0) || !(r_c > 0.f) || !isfinite(r_c))
        return MG_ERR_INVALID_ARG;
    return launch_cutoff(c, pos, lat, sp, n_struct, n_atoms, r_c, o, 0, (cudaStream_t)stream);
}

extern "C" mg_status mg_cutoff_graph_radii(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                                           int32_t n_struct, int32_t n_atoms, const float *radii, const mg_edges *o,
                                           void *stream) {
    if (bad_inputs(c, pos, lat, sp, n_struct, n_atoms) || bad_edges(o, 0) || (n_atoms > 0 && !radii)) return MG_ERR_INVALID_ARG;
    return launch_cutoff(c, pos, lat, sp, n_struct, n_atoms, 1.f, o, 0, (cudaStream_t)stream, radii);
}

extern "C" mg_status mg_cutoff_count(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                                     int32_t n_struct, int32_t n_atoms, float r_c,
                                     int64_t *n_edges_host, void *stream) {
    if (bad_inputs(c, pos, lat, sp, n_struct, n_atoms) || !n_edges_host || !(r_c > 0.f) || !isfinite(r_c))
        return MG_ERR_INVALID_ARG;
    mg_status rs = mg_reserve(c, n_struct, n_atoms);
    if (rs != MG_OK) return rs;
    mg_edges o;
    memset(&o, 0, sizeof(o));
    o.row_ptr = c->d_rowptr_tmp;
    o.n_edges = (int64_t *)c->d_count;
    rs = launch_cutoff(c, pos, lat, sp, n_struct, n_atoms, r_c, &o, 1, (cudaStream_t)stream);
    if (rs != MG_OK) return rs;
    long long v = 0;
    MG_CUDA(cudaMemcpyAsync(&v, c->d_count, sizeof(v), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    MG_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    *n_edges_host = v;
    return MG_OK;
}

static mg_status launch_knn(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                            int32_t n_struct, int32_t n_atoms, int32_t k, const mg_edges *o,
                            float *hint, int use_hint, cudaStream_t st) {
    MG_CUDA(cudaSetDevice(c->device));
    mg_status rs = mg_reserve(c, n_struct, n_atoms);
    if (rs != MG_OK) return rs;
    if (n_struct > 0 && n_atoms / n_struct > MG_SMALL_MAX_ATOMS) {
        // a batch of large structures (any k): one warp per row through the cell list (knn_bins.cu); four launches: prep (which
        // also wraps the coordinates and picks the slab counts), the sort by bin, the rows, the reset of the list
        const int n_blocks = (n_struct + MG_CP_BLOCK - 1) / MG_CP_BLOCK;
        CutPrepArgs P;
        P.lattice = lat; P.struct_ptr = sp; P.n_struct = n_struct; P.n_atoms = n_atoms; P.r_c = 0.f;
        P.k = k; P.hint = hint; P.use_hint = use_hint; P.rows_cost = 0;
        P.pos = pos; P.xw4 = c->d_xw4; P.n_sblocks = n_blocks; P.radii = nullptr; P.binlist = c->d_binlist;
        P.rec = c->d_crec; P.bpre = c->d_bpre; P.ctl = c->d_ctl; P.status = c->d_ctl + 4;
        const int xblocks = (n_atoms + 8 * MG_CP_BLOCK - 1) / (8 * MG_CP_BLOCK);
        MG_CUDA(launch_after(c, mg_cut_prep_kernel, n_blocks + (xblocks < 1024 ? xblocks : 1024), MG_CP_BLOCK, 0, st, P));
        BinArgs B;
        B.rec = c->d_crec; B.xw4 = c->d_xw4; B.xs4 = c->d_xs4; B.bin_start = c->d_binstart;
        B.n_struct = n_struct; B.binlist = c->d_binlist; B.ctl = c->d_ctl;
        const int bgrid = n_struct < 2 * c->sm_count ? n_struct : 2 * c->sm_count;
        MG_CUDA(launch_after(c, mg_cut_bin_kernel, bgrid, MGB_BLOCK, 0, st, B));
        KnnBinsArgs A;
        A.pos = pos; A.lattice = lat; A.struct_ptr = sp; A.n_struct = n_struct; A.n_atoms = n_atoms; A.k = k;
        A.row_ptr = o->row_ptr; A.src = o->src; A.dst = o->dst; A.offset = o->offset; A.vec = o->vec; A.dist = o->dist;
        A.n_edges = (long long *)o->n_edges; A.hint = hint; A.rec = c->d_crec; A.xw4 = c->d_xw4; A.xs4 = c->d_xs4;
        A.bin_start = c->d_binstart; A.status = c->d_ctl + 4;
        int grid = c->sm_count * c->knnb_occ;
        const int cap_grid = (n_atoms + MG_WARPS - 1) / MG_WARPS;
        if (grid > cap_grid) grid = cap_grid;
        MG_CUDA(mg_knn_bins_launch(&A, grid, st, c->pdl));
        MG_CUDA(cudaMemsetAsync(c->d_ctl + 13, 0, sizeof(unsigned), st));      // (the list of binned structures: empty again)
        c->launches += 3;
        return MG_OK;
    }
    if (k <= 32 && n_struct > 0) {                      // pair-lane kernel (knn_pairs.cuh)
        const int n_blocks = (n_struct + MG_CP_BLOCK - 1) / MG_CP_BLOCK;
        if (c->profile) { prof_collect(c); cudaEventRecord(c->ev[0], st); }
        CutPrepArgs P;
        P.lattice = lat; P.struct_ptr = sp; P.n_struct = n_struct; P.n_atoms = n_atoms; P.r_c = 0.f;
        P.k = k; P.hint = hint; P.use_hint = use_hint; P.rows_cost = 0;
        P.pos = pos; P.xw4 = nullptr; P.n_sblocks = n_blocks; P.radii = nullptr; P.binlist = nullptr;
        P.rec = c->d_crec; P.bpre = c->d_bpre; P.ctl = c->d_ctl; P.status = c->d_ctl + 4;
        MG_CUDA(launch_after(c, mg_cut_prep_kernel, n_blocks, MG_CP_BLOCK, 0, st, P));
        c->launches += 1;
        KnnPairsArgs A;
        A.pos = pos; A.lattice = lat; A.struct_ptr = sp;
        A.n_struct = n_struct; A.n_atoms = n_atoms; A.k = k;
        A.row_ptr = o->row_ptr; A.src = o->src; A.dst = o->dst; A.offset = o->offset;
        A.vec = o->vec; A.dist = o->dist; A.n_edges = (long long *)o->n_edges;
        A.hint = hint; A.rec = c->d_crec; A.bpre = c->d_bpre; A.n_blocks = n_blocks;
        A.status = c->d_ctl + 4;
        A.dbg = c->d_wclock;
        int grid = c->sm_count * c->knnp_occ;
        const int cap_grid = (n_atoms + MG_WARPS) / MG_WARPS;
        if (grid > cap_grid) grid = cap_grid;
        A.n_warps = grid * MG_WARPS;
        if (c->profile) cudaEventRecord(c->ev[1], st);
        if (k > 16) MG_CUDA(mg_knn_large_launch(&A, sizeof(A), grid, st, c->pdl));
        else MG_CUDA(launch_after(c, mg_knn_pairs_kernel, grid, MG_BLOCK, MG_WARPS * sizeof(KnnSmem), st, A));
        c->launches += 1;
        if (c->profile) { cudaEventRecord(c->ev[3], st); c->pend_kind = 1; }
        return MG_OK;
    }
    if (n_struct > 0) {
        rs = launch_prep(c, pos, lat, sp, n_struct, n_atoms, 0.f, st);
        if (rs != MG_OK) return rs;
    }
    KnnArgs A;
    A.pos = pos; A.lattice = lat; A.struct_ptr = sp;
    A.n_struct = n_struct; A.n_atoms = n_atoms; A.k = k;
    A.row_ptr = o->row_ptr; A.src = o->src; A.dst = o->dst; A.offset = o->offset;
    A.vec = o->vec; A.dist = o->dist; A.n_edges = (long long *)o->n_edges;
    A.radius_hint = hint; A.use_hint = use_hint;
    A.rec = c->d_rec; A.atom_struct = c->d_atom_struct;
    A.ctl = c->d_ctl; A.status = c->d_ctl + 4;
    const int kpl = k <= 32 ? 0 : 1;
    int grid = c->sm_count * c->knn_occ[kpl];
    if (grid > (n_atoms + MG_WARPS - 1) / MG_WARPS) grid = (n_atoms + MG_WARPS - 1) / MG_WARPS;
    if (grid < 1) grid = 1;
    if (kpl == 0) mg_knn_small_kernel<1><<<grid, MG_BLOCK, 0, st>>>(A);
    else mg_knn_small_kernel<2><<<grid, MG_BLOCK, 0, st>>>(A);
    MG_CUDA(cudaGetLastError());
    c->launches += 1;
    return MG_OK;
}

extern "C" mg_status mg_knn_graph(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                                  int32_t n_struct, int32_t n_atoms, int32_t k, const mg_edges *o,
                                  void *stream) {
    if (k < 1 || k > MG_MAX_K) return MG_ERR_INVALID_ARG;
    if (bad_inputs(c, pos, lat, sp, n_struct, n_atoms) || bad_edges(o, (long long)k * n_atoms))
        return MG_ERR_INVALID_ARG;
    return launch_knn(c, pos, lat, sp, n_struct, n_atoms, k, o, nullptr, 0, (cudaStream_t)stream);
}

extern "C" mg_status mg_graph_create(mg_ctx *c, int kind, float r_c, int32_t k, const int32_t *sp,
                                     int32_t n_struct, int32_t n_atoms, mg_graph **out) {
    if (!out) return MG_ERR_INVALID_ARG;
    *out = nullptr;
    if (!c || !sp || n_struct < 0 || n_atoms < 0) return MG_ERR_INVALID_ARG;
    if (kind == MG_KIND_CUTOFF) { if (!(r_c > 0.f) || !isfinite(r_c)) return MG_ERR_INVALID_ARG; }
    else if (kind == MG_KIND_KNN) { if (k < 1 || k > MG_MAX_K) return MG_ERR_INVALID_ARG; }
    else return MG_ERR_INVALID_ARG;
    mg_status rs = mg_reserve(c, n_struct, n_atoms);
    if (rs != MG_OK) return rs;
    mg_graph *g = new (std::nothrow) mg_graph();
    if (!g) return MG_ERR_CUDA;
    g->ctx = c; g->kind = kind; g->r_c = r_c; g->k = k;
    g->struct_ptr = sp; g->n_struct = n_struct; g->n_atoms = n_atoms;
    if (kind == MG_KIND_KNN && n_atoms > 0) {
        const size_t nh = (size_t)(n_atoms > n_struct ? n_atoms : n_struct) + 1;   // per atom (k > 32) or per structure
        if (cudaMalloc(&g->d_hint, nh * sizeof(float)) != cudaSuccess ||
            cudaMemset(g->d_hint, 0, nh * sizeof(float)) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(g->d_hint);
            delete g;
            return MG_ERR_CUDA;
        }
    }
    *out = g;
    return MG_OK;
}

extern "C" void mg_graph_destroy(mg_graph *g) {
    if (!g) return;
    cudaSetDevice(g->ctx->device);
    cudaFree(g->d_hint);
    delete g;
}

extern "C" mg_status mg_update_graph(mg_ctx *c, mg_graph *g, const float *pos, const float *lat,
                                     const mg_edges *o, void *stream) {
    if (!c || !g || g->ctx != c) return MG_ERR_INVALID_ARG;
    if (bad_inputs(c, pos, lat, g->struct_ptr, g->n_struct, g->n_atoms)) return MG_ERR_INVALID_ARG;
    if (g->kind == MG_KIND_CUTOFF) {
        if (bad_edges(o, 0)) return MG_ERR_INVALID_ARG;
        return launch_cutoff(c, pos, lat, g->struct_ptr, g->n_struct, g->n_atoms, g->r_c, o, 0,
                             (cudaStream_t)stream);
    }
    if (bad_edges(o, (long long)g->k * g->n_atoms)) return MG_ERR_INVALID_ARG;
    mg_status rs = launch_knn(c, pos, lat, g->struct_ptr, g->n_struct, g->n_atoms, g->k, o, g->d_hint,
                              g->have_hint, (cudaStream_t)stream);
    if (rs == MG_OK) g->have_hint = 1;
    return rs;
}

// ---- operations on a finished graph (graph_ops.cuh) -------------------------------------------------
extern "C" mg_status mg_symmetrize(mg_ctx *c, const mg_edges *in, int32_t n_atoms, const mg_edges *out, void *stream) {
    if (!c || n_atoms < 0 || !in || !in->row_ptr || !in->n_edges || in->capacity < 0 || bad_edges(out, 0)) return MG_ERR_INVALID_ARG;
    if (in->capacity > 0 && (!in->src || !in->dst || !in->offset || !in->vec)) return MG_ERR_INVALID_ARG;
    if (out->dist && !in->dist) return MG_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    MG_CUDA(cudaSetDevice(c->device));
    if ((size_t)in->capacity + 1 > c->symflag_cap) {
        cudaFree(c->d_symflag);
        c->d_symflag = nullptr; c->symflag_cap = 0;
        const size_t cap = (size_t)in->capacity + (size_t)in->capacity / 8 + 1024;
        MG_CUDA(cudaMalloc(&c->d_symflag, cap));
        c->symflag_cap = cap;
    }
    if ((size_t)n_atoms + 1 > c->symcnt_cap) {
        cudaFree(c->d_symcnt);
        c->d_symcnt = nullptr; c->symcnt_cap = 0;
        const size_t cap = (size_t)n_atoms + 1025;
        MG_CUDA(cudaMalloc(&c->d_symcnt, 2 * cap * sizeof(int)));
        c->symcnt_cap = cap;
    }
    if ((size_t)mgo_scan_blocks(n_atoms) > c->scanpart_cap) {
        const size_t cap = (size_t)mgo_scan_blocks(n_atoms) + 64;
        cudaFree(c->d_scanpart);
        c->d_scanpart = nullptr; c->scanpart_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_scanpart, cap * sizeof(long long)));
        c->scanpart_cap = cap;
    }
    MG_CUDA(cudaMemsetAsync(c->d_symcnt, 0, 2 * c->symcnt_cap * sizeof(int), st));
    SymArgs A;
    A.row_ptr = in->row_ptr; A.src = in->src; A.dst = in->dst; A.offset = in->offset; A.vec = in->vec; A.dist = in->dist;
    A.n_edges_in = (const long long *)in->n_edges; A.cap_in = in->capacity; A.n_atoms = n_atoms;
    A.o_row_ptr = out->row_ptr; A.o_src = out->src; A.o_dst = out->dst; A.o_offset = out->offset; A.o_vec = out->vec;
    A.o_dist = out->dist; A.capacity = out->capacity; A.n_edges_out = (long long *)out->n_edges;
    A.flag = c->d_symflag; A.extra = c->d_symcnt; A.fill = c->d_symcnt + c->symcnt_cap; A.status = c->d_ctl + 4;
    A.part = c->d_scanpart;
    long long want = (in->capacity + MGO_BLOCK - 1) / MGO_BLOCK;
    const int grid = (int)(want < 1 ? 1 : (want > (long long)c->sm_count * 16 ? (long long)c->sm_count * 16 : want));
    MG_CUDA(launch_after(c, mg_sym_flag_kernel, grid, MGO_BLOCK, 0, st, A));
    MG_CUDA(launch_after(c, mg_sym_part_kernel, mgo_scan_blocks(n_atoms), MGO_SCAN_BLOCK, 0, st, A));
    MG_CUDA(launch_after(c, mg_sym_scan_kernel, mgo_scan_blocks(n_atoms), MGO_SCAN_BLOCK, 0, st, A));
    MG_CUDA(launch_after(c, mg_sym_emit_kernel, grid, MGO_BLOCK, 0, st, A));
    c->launches += 4;
    return MG_OK;
}

extern "C" mg_status mg_triplets_graph(mg_ctx *c, const int32_t *row_ptr, int32_t n_atoms, const mg_triplets *out, void *stream) {
    if (!c || !row_ptr || n_atoms < 0 || !out || !out->tri_ptr || !out->n_triplets || out->capacity < 0) return MG_ERR_INVALID_ARG;
    if (out->capacity > 0 && (!out->edge_a || !out->edge_b)) return MG_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    MG_CUDA(cudaSetDevice(c->device));
    if ((size_t)mgo_scan_blocks(n_atoms) > c->scanpart_cap) {
        const size_t cap = (size_t)mgo_scan_blocks(n_atoms) + 64;
        cudaFree(c->d_scanpart);
        c->d_scanpart = nullptr; c->scanpart_cap = 0;
        MG_CUDA(cudaMalloc(&c->d_scanpart, cap * sizeof(long long)));
        c->scanpart_cap = cap;
    }
    TripArgs A;
    A.part = c->d_scanpart;
    A.row_ptr = row_ptr; A.n_atoms = n_atoms; A.tri_ptr = (long long *)out->tri_ptr;
    A.edge_a = out->edge_a; A.edge_b = out->edge_b; A.capacity = out->capacity;
    A.n_triplets = (long long *)out->n_triplets; A.status = c->d_ctl + 4;
    MG_CUDA(launch_after(c, mg_trip_part_kernel, mgo_scan_blocks(n_atoms), MGO_SCAN_BLOCK, 0, st, A));
    MG_CUDA(launch_after(c, mg_trip_scan_kernel, mgo_scan_blocks(n_atoms), MGO_SCAN_BLOCK, 0, st, A));
    const long long want = ((long long)n_atoms * 32 + MGO_BLOCK - 1) / MGO_BLOCK;
    const int grid = (int)(want < 1 ? 1 : (want > (long long)c->sm_count * 8 ? (long long)c->sm_count * 8 : want));
    MG_CUDA(launch_after(c, mg_trip_emit_kernel, grid, MGO_BLOCK, 0, st, A));
    c->launches += 3;
    return MG_OK;
}

// ---- mg_symmetrize without allocation (include/matgraph.h) -------------------------------------------
// The scratch of the three symmetrize kernels in a file-scope device array: a status word (one 256-byte
// line), the two counters per atom (extra | fill, packed behind one another for the call's n_atoms) and
// one flag byte per input edge.  Every GPU that loads the library holds it until the process exits.
#define MGST_HEAD 256
static_assert(64 + (MG_STATIC_MAX_ATOMS / MGO_CHUNK + 1) * sizeof(long long) <= MGST_HEAD, "the chunk totals fit the header");
#define MGST_COUNTERS (2 * (size_t)MG_STATIC_MAX_ATOMS * sizeof(int) + 512)
#define MGST_BYTES (MGST_HEAD + MGST_COUNTERS + (size_t)MG_STATIC_MAX_EDGES + 256)
static __device__ __align__(256) unsigned char mg_static_scratch[MGST_BYTES];

// In host code `mg_static_scratch` is a stand-in, not a device address: the address the kernels get is
// looked up once per device, with that device current.
#define MGST_MAX_DEVICES 64
static std::mutex g_static_lock;
static unsigned char *g_static_ptr[MGST_MAX_DEVICES];
static int g_static_sms[MGST_MAX_DEVICES];

extern "C" mg_status mg_symmetrize_static(int32_t device, const mg_edges *in, int32_t n_atoms, const mg_edges *out,
                                          void *stream) {
    if (device < 0 || device >= MGST_MAX_DEVICES || n_atoms < 0 || !in || !in->row_ptr || !in->n_edges || in->capacity < 0 ||
        bad_edges(out, 0))
        return MG_ERR_INVALID_ARG;
    if (in->capacity > 0 && (!in->src || !in->dst || !in->offset || !in->vec)) return MG_ERR_INVALID_ARG;
    if (out->dist && !in->dist) return MG_ERR_INVALID_ARG;
    if (n_atoms > MG_STATIC_MAX_ATOMS || in->capacity > (long long)MG_STATIC_MAX_EDGES) return MG_ERR_TOO_LARGE;
    cudaStream_t st = (cudaStream_t)stream;
    MG_CUDA(cudaSetDevice(device));
    unsigned char *base;
    int sms;
    {
        std::lock_guard<std::mutex> guard(g_static_lock);
        if (!g_static_ptr[device]) {
            void *p = nullptr;
            int n = 0;
            MG_CUDA(cudaGetSymbolAddress(&p, mg_static_scratch));
            MG_CUDA(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device));
            if (!p || n < 1) return MG_ERR_CUDA;
            g_static_sms[device] = n;
            g_static_ptr[device] = (unsigned char *)p;
        }
        base = g_static_ptr[device];
        sms = g_static_sms[device];
    }
    // the array keeps the last call's contents: status word and both counter arrays start at zero
    const size_t na = ((size_t)n_atoms + 63) & ~(size_t)63;               // counters of a call: [na] extra | [na] fill
    MG_CUDA(cudaMemsetAsync(base, 0, MGST_HEAD + 2 * na * sizeof(int), st));
    SymArgs A;
    A.row_ptr = in->row_ptr; A.src = in->src; A.dst = in->dst; A.offset = in->offset; A.vec = in->vec; A.dist = in->dist;
    A.n_edges_in = (const long long *)in->n_edges; A.cap_in = in->capacity; A.n_atoms = n_atoms;
    A.o_row_ptr = out->row_ptr; A.o_src = out->src; A.o_dst = out->dst; A.o_offset = out->offset; A.o_vec = out->vec;
    A.o_dist = out->dist; A.capacity = out->capacity; A.n_edges_out = (long long *)out->n_edges;
    A.status = reinterpret_cast<unsigned *>(base);
    A.part = reinterpret_cast<long long *>(base + 64);          // (MG_STATIC_MAX_ATOMS / MGO_CHUNK = 8 chunk totals)
    A.extra = reinterpret_cast<int *>(base + MGST_HEAD);
    A.fill = A.extra + na;
    A.flag = base + MGST_HEAD + MGST_COUNTERS;       // (every flag the emit kernel reads is written by the flag kernel)
    long long want = (in->capacity + MGO_BLOCK - 1) / MGO_BLOCK;
    const int grid = (int)(want < 1 ? 1 : (want > (long long)sms * 16 ? (long long)sms * 16 : want));
    mg_sym_flag_kernel<<<grid, MGO_BLOCK, 0, st>>>(A);
    mg_sym_part_kernel<<<mgo_scan_blocks(n_atoms), MGO_SCAN_BLOCK, 0, st>>>(A);
    mg_sym_scan_kernel<<<mgo_scan_blocks(n_atoms), MGO_SCAN_BLOCK, 0, st>>>(A);
    mg_sym_emit_kernel<<<grid, MGO_BLOCK, 0, st>>>(A);
    MG_CUDA(cudaGetLastError());
    return MG_OK;
}

extern "C" mg_status mg_check(mg_ctx *c, void *stream) {
    if (!c) return MG_ERR_INVALID_ARG;
    MG_CUDA(cudaSetDevice(c->device));
    unsigned bits = 0;
    MG_CUDA(cudaMemcpyAsync(&bits, c->d_ctl + 4, sizeof(bits), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    MG_CUDA(cudaMemsetAsync(c->d_ctl + 4, 0, sizeof(unsigned), (cudaStream_t)stream));
    MG_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    return decode_status(bits);
}

// ---- host-buffer entry points -------------------------------------------------------------
static mg_status host_buf(mg_ctx *c, int slot, size_t bytes) {
    if (bytes <= c->h_cap[slot]) return MG_OK;
    cudaFree(c->h_dev[slot]);
    c->h_dev[slot] = nullptr; c->h_cap[slot] = 0;
    const size_t cap = bytes + bytes / 4 + 256;
    MG_CUDA(cudaMalloc(&c->h_dev[slot], cap));
    c->h_cap[slot] = cap;
    return MG_OK;
}

static mg_status run_host(mg_ctx *c, int kind, const float *pos, const float *lat, const int32_t *sp,
                          int32_t n_struct, int32_t n_atoms, float r_c, int32_t k, const mg_edges *oh) {
    if (!c || n_struct < 0 || n_atoms < 0 || !sp || (n_struct > 0 && !lat) || (n_atoms > 0 && !pos))
        return MG_ERR_INVALID_ARG;
    if (bad_edges(oh, kind == MG_KIND_KNN ? (long long)k * n_atoms : 0)) return MG_ERR_INVALID_ARG;
    MG_CUDA(cudaSetDevice(c->device));
    const size_t cap = (size_t)oh->capacity;
    const size_t sz[9] = {(size_t)n_atoms * 12 + 4, (size_t)n_struct * 36 + 4, ((size_t)n_struct + 1) * 4,
                          ((size_t)n_atoms + 1) * 4, cap * 4 + 4, cap * 4 + 4, cap * 3 + 4, cap * 12 + 4,
                          (oh->dist ? cap * 4 : 0) + 16};
    for (int i = 0; i < 9; ++i) { mg_status rs = host_buf(c, i, sz[i]); if (rs != MG_OK) return rs; }
    cudaStream_t st = 0;
    MG_CUDA(cudaMemcpyAsync(c->h_dev[0], pos, (size_t)n_atoms * 12, cudaMemcpyHostToDevice, st));
    MG_CUDA(cudaMemcpyAsync(c->h_dev[1], lat, (size_t)n_struct * 36, cudaMemcpyHostToDevice, st));
    MG_CUDA(cudaMemcpyAsync(c->h_dev[2], sp, ((size_t)n_struct + 1) * 4, cudaMemcpyHostToDevice, st));
    mg_edges od;
    od.row_ptr = (int32_t *)c->h_dev[3]; od.src = (int32_t *)c->h_dev[4]; od.dst = (int32_t *)c->h_dev[5];
    od.offset = (int8_t *)c->h_dev[6]; od.vec = (float *)c->h_dev[7];
    od.dist = oh->dist ? (float *)((char *)c->h_dev[8] + 16) : nullptr;
    od.capacity = oh->capacity; od.n_edges = (int64_t *)c->h_dev[8];
    mg_status rs;
    if (kind == MG_KIND_CUTOFF)
        rs = mg_cutoff_graph(c, (const float *)c->h_dev[0], (const float *)c->h_dev[1],
                             (const int32_t *)c->h_dev[2], n_struct, n_atoms, r_c, &od, st);
    else
        rs = mg_knn_graph(c, (const float *)c->h_dev[0], (const float *)c->h_dev[1],
                          (const int32_t *)c->h_dev[2], n_struct, n_atoms, k, &od, st);
    if (rs != MG_OK) return rs;
    long long ne = 0;
    MG_CUDA(cudaMemcpyAsync(&ne, od.n_edges, 8, cudaMemcpyDeviceToHost, st));
    MG_CUDA(cudaMemcpyAsync(oh->row_ptr, od.row_ptr, ((size_t)n_atoms + 1) * 4, cudaMemcpyDeviceToHost, st));
    MG_CUDA(cudaStreamSynchronize(st));
    *oh->n_edges = ne;
    const size_t m = (size_t)(ne < oh->capacity ? ne : oh->capacity);
    if (m) {
        MG_CUDA(cudaMemcpyAsync(oh->src, od.src, m * 4, cudaMemcpyDeviceToHost, st));
        MG_CUDA(cudaMemcpyAsync(oh->dst, od.dst, m * 4, cudaMemcpyDeviceToHost, st));
        MG_CUDA(cudaMemcpyAsync(oh->offset, od.offset, m * 3, cudaMemcpyDeviceToHost, st));
        MG_CUDA(cudaMemcpyAsync(oh->vec, od.vec, m * 12, cudaMemcpyDeviceToHost, st));
        if (oh->dist) MG_CUDA(cudaMemcpyAsync(oh->dist, od.dist, m * 4, cudaMemcpyDeviceToHost, st));
    }
    return mg_check(c, st);
}

extern "C" mg_status mg_cutoff_graph_host(mg_ctx *c, const float *pos, const float *lat,
                                          const int32_t *sp, int32_t n_struct, int32_t n_atoms,
                                          float r_c, const mg_edges *oh) {
    if (!(r_c > 0.f) || !isfinite(r_c)) return MG_ERR_INVALID_ARG;
    return run_host(c, MG_KIND_CUTOFF, pos, lat, sp, n_struct, n_atoms, r_c, 0, oh);
}

extern "C" mg_status mg_knn_graph_host(mg_ctx *c, const float *pos, const float *lat, const int32_t *sp,
                                       int32_t n_struct, int32_t n_atoms, int32_t k, const mg_edges *oh) {
    if (k < 1 || k > MG_MAX_K) return MG_ERR_INVALID_ARG;
    return run_host(c, MG_KIND_KNN, pos, lat, sp, n_struct, n_atoms, 0.f, k, oh);
}
