// knn_bins_args.cuh — arguments of mg_knn_bins_kernel (knn_bins.cu), the KNN kernel for batches of large structures.
// A plain struct and nothing else: matgraph.cu fills it, knn_bins.cu (a module of its own) reads it.
#pragma once
#include <stdint.h>

struct KnnBinsArgs {
    const float *pos;              // [n_atoms, 3] as given
    const float *lattice;          // [n_struct, 9]
    const int32_t *struct_ptr;     // [n_struct + 1]
    int n_struct, n_atoms, k;
    int32_t *row_ptr, *src, *dst;
    int8_t *offset;
    float *vec, *dist;             // dist may be NULL
    long long *n_edges;
    float *hint;                   // [n_struct] or NULL: largest k-th distance per structure (atomicMax)
    const void *rec;               // CutRec [n_struct] of mg_cut_prep_kernel (k > 0: radius, bins)
    const void *xw4;               // float4 [n_atoms] wrapped coordinates + packed integer parts (cut_prep.cuh)
    const void *xs4;               // float4 [n_atoms] the same in bin order, .w = atom and integer parts (cut_bins.cuh)
    const int *bin_start;          // [n_atoms + 2 n_struct + 2]
    unsigned *status;
};
