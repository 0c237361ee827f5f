// prep.cuh — K1 (per-structure search bounds) + K6 (batching): one WARP per structure.
//
//  * plane spacings h_a = V / |a_b x a_c| in FP64 from the FP32 lattice, validity (finite, V > 1e-9),
//  * cutoff box n_a = floor(r_c / h_a + spread_a)  (<= ceil(r_c/h_a) for x in [0,1); spread_a =
//    max_i x_ia - min_i x_ia makes the bound hold for coordinates outside the unit cell, R6/R14),
//  * the rounding window [lo2, hi2) of the FP32 distance filter,
//  * the split of the structure's source rows into cutoff TASKS of about MG_TASK_BUDGET
//    candidates (<= MG_TASK_ROWS rows, expected edges within the per-warp stash); the LAST block to
//    finish turns the task counts into an exclusive prefix sum and publishes the number of tasks,
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
    unsigned *task_prefix;      // [n_struct + 1]
    int32_t *atom_struct;       // [n_atoms]
    unsigned *ctl;              // [5] blocks done, [6] number of tasks
    unsigned *status;
};

#define MG_PREP_BLOCK 128

__global__ void __launch_bounds__(MG_PREP_BLOCK)
mg_prep_kernel(const PrepArgs A) {
    const int lane = threadIdx.x & 31;
    const int s = blockIdx.x * (MG_PREP_BLOCK / 32) + (threadIdx.x >> 5);
    if (s < A.n_struct) {
        const int first = A.struct_ptr[s];
        const int N = A.struct_ptr[s + 1] - first;
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        float xabs = 1.f;
        bool finite = true;
        for (int j = lane; j < N; j += 32) {
            A.atom_struct[first + j] = s;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float v = A.pos[3 * (size_t)(first + j) + a];
                finite = finite && isfinite(v);
                lo[a] = fminf(lo[a], v);
                hi[a] = fmaxf(hi[a], v);
                xabs = fmaxf(xabs, fabsf(v));
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                lo[a] = fminf(lo[a], __shfl_xor_sync(0xFFFFFFFFu, lo[a], o));
                hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xFFFFFFFFu, hi[a], o));
            }
            xabs = fmaxf(xabs, __shfl_xor_sync(0xFFFFFFFFu, xabs, o));
        }
        finite = __all_sync(0xFFFFFFFFu, finite);
        if (lane == 0) {
            StructRec r;
            r.first = first;
            r.natoms = N;
            float lat[9];
#pragma unroll
            for (int c = 0; c < 9; ++c) lat[c] = A.lattice[9 * (size_t)s + c];
            double vol = 0.0, h[3] = {1.0, 1.0, 1.0};
            unsigned err = mg_cell_spacings(lat, &vol, h);
            if (!finite) err |= MGS_NONFINITE;
            if (N > MG_SMALL_MAX_ATOMS) err |= MGS_UNSUPPORTED;
            double M = 0.0;
            r.ncell = 0;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                r.xmin[a] = N ? lo[a] : 0.f;
                r.xmax[a] = N ? hi[a] : 0.f;
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
            const double wl = (double)A.r_c - W, wh = (double)A.r_c + W;
            r.lo2 = wl > 0.0 ? __double2float_rd(wl * wl * (1.0 - 1e-6)) : 0.f;
            r.hi2 = __double2float_ru(wh * wh * (1.0 + 1e-6));
            r.volume = (float)vol;
            r.err = err;
            if (err) atomicOr(A.status, err);
            // ---- task split: rows per task from the candidate budget and the stash
            int rpt = MG_TASK_ROWS, cap = 0;
            if (r.ncell > 0) {
                const unsigned rowwork = (unsigned)N * (unsigned)((r.ncell + 7) & ~7);
                rpt = (int)(MG_TASK_BUDGET / rowwork);
                // expected row length lambda = N (4/3) pi r_c^3 / V, plus slack
                const float lam = (float)N * 4.18879f * A.r_c * A.r_c * A.r_c / r.volume;
                cap = min(MG_WS, (int)(1.25f * lam) + 24);
                rpt = max(1, min(rpt, min(MG_TASK_ROWS, MG_WS / cap)));
            }
            r.rpt = rpt;
            r.cap = cap;
#pragma unroll
            for (int c = 0; c < 5; ++c) r.pad[c] = 0;
            A.rec[s] = r;
            A.task_prefix[s + 1] = (unsigned)((N + rpt - 1) / rpt);   // scanned below
        }
    }
    // ---- last block: exclusive prefix sum of the task counts
    __shared__ unsigned part[MG_PREP_BLOCK];
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
    unsigned sum = 0;
    for (int t = b; t < e; ++t) sum += __ldcg(A.task_prefix + t + 1);
    // block-wide exclusive scan of the partial sums
    unsigned incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) part[threadIdx.x >> 5] = incl;
    __syncthreads();
    unsigned woff = 0;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) woff += part[w];
    unsigned run = woff + incl - sum;
    if (threadIdx.x == MG_PREP_BLOCK - 1) {
        A.task_prefix[0] = 0u;
        A.ctl[6] = woff + incl;
        A.ctl[5] = 0u;
    }
    for (int t = b; t < e; ++t) {
        run += __ldcg(A.task_prefix + t + 1);
        A.task_prefix[t + 1] = run;                 // inclusive at s+1 == exclusive prefix of s+1
    }
}
