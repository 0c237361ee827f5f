// knn_large.cu — the pair-lane KNN kernel for k > 16 (knn_pairs_kernel.inc with MG_KNN_LARGE 1) as a module of its own,
// and the two host functions matgraph.cu reaches it through.  Everything the shared headers define lives in a
// namespace here, so their other kernels (compiled again, unused) do not clash with matgraph.cu's at link time.
#include "../../include/matgraph.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

namespace mg_knn_large_tu {
#define MG_KNN_LARGE_TU 1
#include "common.cuh"
#include "cut_prep.cuh"
#include "cutoff_pairs.cuh"
#include "knn_small.cuh"
#include "knn_pairs.cuh"
}  // namespace mg_knn_large_tu

using mg_knn_large_tu::KnnPairsArgs;
using mg_knn_large_tu::KnnSmem;

// Opt the kernel in to its shared memory; *occ: resident CTAs per SM.  Call once per device, that device current.
__attribute__((visibility("hidden"))) cudaError_t mg_knn_large_setup(int *occ) {
    const size_t smem = MG_WARPS * sizeof(KnnSmem);
    cudaError_t e = cudaFuncSetAttribute(mg_knn_large_tu::mg_knn_pairs_large_kernel,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, mg_knn_large_tu::mg_knn_pairs_large_kernel, MG_BLOCK, smem);
}

// `args`: a KnnPairsArgs of matgraph.cu (the same struct: one header), `pdl`: programmatic dependent launch.
__attribute__((visibility("hidden"))) cudaError_t mg_knn_large_launch(const void *args, size_t args_bytes, int grid,
                                                                      cudaStream_t st, int pdl) {
    KnnPairsArgs a;
    if (args_bytes != sizeof(a)) return cudaErrorInvalidValue;
    memcpy(&a, args, sizeof(a));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(MG_BLOCK);
    cfg.dynamicSmemBytes = MG_WARPS * sizeof(KnnSmem);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, mg_knn_large_tu::mg_knn_pairs_large_kernel, a);
}
