// prep.cuh — K1 (per-structure search bounds) + K6 (batching): one thread per structure.
//
//  * plane spacings h_a = V / |a_b x a_c| in FP64 from the FP32 lattice, validity (finite, V > 1e-9),
//  * cutoff box n_a = floor(r_c / h_a + spread_a)  (<= ceil(r_c/h_a) for x in [0,1); spread_a =
//    max_i x_ia - min_i x_ia makes the bound hold for coordinates outside the unit cell, R6/R14),
//  * the rounding window [lo2, hi2) of the FP32 distance filter,
//  * a scheduling cost per source row; the LAST block to finish turns the costs into an exclusive
//    prefix sum P (uint64) — cutoff chunk c owns the rows whose cost offset lies in
//    [c * MG_CHUNK_COST, (c+1) * MG_CHUNK_COST) — and publishes the number of chunks,
//  * atom -> structure map for the warp-per-atom KNN kernel.
#pragma once
#include "common.cuh"

struct PrepArgs {
    const float *pos;
    const float *lattice;
    const int32_t *struct_ptr;
    int n_struct, n_atoms;
    float r_c;                  // <= 0: KNN call (no cutoff box)
    StructRec *rec;             // [n_struct]
    unsigned long long *cost_prefix;   // [n_struct + 1]
    int32_t *atom_struct;       // [n_atoms]
    unsigned *ctl;              // [5] blocks done, [6] n_chunks
    unsigned *status;
};

#define MG_PREP_BLOCK 128

__global__ void __launch_bounds__(MG_PREP_BLOCK)
mg_prep_kernel(const PrepArgs A) {
    const int s = blockIdx.x * MG_PREP_BLOCK + threadIdx.x;
    if (s < A.n_struct) {
        StructRec r;
        const int first = A.struct_ptr[s];
        const int N = A.struct_ptr[s + 1] - first;
        r.first = first;
        r.natoms = N;
        float lat[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) lat[c] = A.lattice[9 * (size_t)s + c];
        double vol = 0.0, h[3] = {1.0, 1.0, 1.0};
        unsigned err = mg_cell_spacings(lat, &vol, h);
        bool finite = true;
        float xabs = 1.f;
#pragma unroll
        for (int a = 0; a < 3; ++a) { r.xmin[a] = 0.f; r.xmax[a] = 0.f; }
        for (int i = 0; i < N; ++i) {
            A.atom_struct[first + i] = s;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float v = A.pos[3 * (size_t)(first + i) + a];
                finite = finite && isfinite(v);
                r.xmin[a] = i ? fminf(r.xmin[a], v) : v;
                r.xmax[a] = i ? fmaxf(r.xmax[a], v) : v;
                xabs = fmaxf(xabs, fabsf(v));
            }
        }
        if (!finite) err |= MGS_NONFINITE;
        if (N > MG_SMALL_MAX_ATOMS) err |= MGS_UNSUPPORTED;
        double M = 0.0;
        r.ncell = 0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            r.n[a] = 0;
            r.h_dn[a] = __double2float_rd(h[a] * (1.0 - 1e-6));
            r.invh_up[a] = __double2float_ru((1.0 + 1e-6) / h[a]);
            r.amax[a] = fmaxf(fabsf(lat[3 * a]), fmaxf(fabsf(lat[3 * a + 1]), fabsf(lat[3 * a + 2])));
        }
        if (!err && A.r_c > 0.f) {
            int nc = 1;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double spread = (double)r.xmax[a] - (double)r.xmin[a];
                const double nn = floor((double)A.r_c / h[a] * (1.0 + 1e-9) + spread);
                if (!(nn <= 127.0)) { err |= MGS_OFFSET; break; }
                r.n[a] = (int)nn;
                nc *= 2 * r.n[a] + 1;
                M += (nn + 2.0 * (double)xabs) * (double)r.amax[a];
            }
            if (!err) r.ncell = nc;
        }
        // every FP32 rounding in p_j, p_i, q = p_j - p_i, T_tau and q + T is <= 2^-24 M; 12 per
        // component; candidates inside the window go to FP64
        const double W = 3.5 * 12.0 * 5.9604644775390625e-8 * M + 2e-6 * (double)A.r_c;
        const double lo = (double)A.r_c - W, hi = (double)A.r_c + W;
        r.lo2 = lo > 0.0 ? __double2float_rd(lo * lo * (1.0 - 1e-6)) : 0.f;
        r.hi2 = __double2float_ru(hi * hi * (1.0 + 1e-6));
        r.volume = (float)vol;
        r.err = err;
        if (err) atomicOr(A.status, err);
        const unsigned work = (unsigned)N * (unsigned)((r.ncell + 31) & ~31);
        // a row never costs more than one chunk budget, so every chunk window holds a row start
        // and the number of chunks is <= n_atoms + 1 (the host sizes the descriptors by that)
        r.rowcost = N > 0 ? min(work + MG_ROW_OVERHEAD + MG_STRUCT_OVERHEAD / (unsigned)N, MG_CHUNK_COST) : 0u;
#pragma unroll
        for (int c = 0; c < 6; ++c) r.pad[c] = 0;
        A.rec[s] = r;
        A.cost_prefix[s + 1] = (unsigned long long)N * r.rowcost;   // scanned below
    }
    // ---- last block: exclusive prefix sum of the structure costs
    __shared__ unsigned long long part[MG_PREP_BLOCK];
    __shared__ bool last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(A.ctl + 5, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last) return;
    __threadfence();
    const int S = A.n_struct;
    const int per = (S + MG_PREP_BLOCK - 1) / MG_PREP_BLOCK;
    const int b = threadIdx.x * per, e = min(S, b + per);
    unsigned long long sum = 0;
    for (int t = b; t < e; ++t) sum += __ldcg(A.cost_prefix + t + 1);
    part[threadIdx.x] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long run = 0;
        for (int t = 0; t < MG_PREP_BLOCK; ++t) { const unsigned long long v = part[t]; part[t] = run; run += v; }
        A.cost_prefix[0] = 0ull;
        A.ctl[6] = (unsigned)(run / MG_CHUNK_COST) + 1u;
        A.ctl[5] = 0u;
    }
    __syncthreads();
    unsigned long long run = part[threadIdx.x];
    for (int t = b; t < e; ++t) {
        run += __ldcg(A.cost_prefix + t + 1);
        A.cost_prefix[t + 1] = run;                 // inclusive at s+1 == exclusive prefix of s+1
    }
}
