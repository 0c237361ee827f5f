// cut_bins.cuh — K2: fractional-coordinate cell list of the large structures (SURVEY.md 8(a) K2,
// BASELINE.json north_star "Binning: fractional-coordinate cell-list binning per structure").
//
// A structure above the staging limit (more than MG_SMALL_MAX_ATOMS atoms) whose per-pair sub-box is one
// cell (m_a = 1 on every axis, i.e. rho_a = r_c / h_a < 1/2: the minimum-image regime, cut_prep.cuh) is
// binned along each axis a into nb_a equal slabs of the WRAPPED fractional coordinate, nb_a <=
// 2 / rho_a, so a slab is at least rho_a / 2 wide.  An edge (i, j, tau) has |x_ja - x_ia + tau_a| <
// rho_a (cut_prep.cuh), so on the circle [0, 1) the two atoms are less than two slabs apart and the slab
// of j is one of the five slabs b_i - 2 .. b_i + 2 (mod nb_a): a source row visits 5 x 5 x 5 of the
// nb_0 nb_1 nb_2 bins instead of all of them.  An axis with fewer than six slabs would be visited whole,
// so it gets one slab.  (The pruning only REMOVES candidates that cannot be edges; every candidate left is
// decided exactly as before: FP32 filter, FP64 inside the rounding window, R23.)
//
// This file: the bin index of a coordinate (shared with the scan kernel's rows, cut_scan.cuh) and the
// kernel that sorts a structure's atoms by bin: one block per structure; per-warp histograms in shared
// memory, exclusive scan, stable scatter (atoms of a bin stay in index order, so the result does not depend on
// the timing of atomics).  Output, per structure s with first atom f: bin_start[f + 2 s + b], b in
// [0, nbins], positions LOCAL to the structure, and at b = nbins + 1 a flag: 1 if every atom is finite and
// within 15 cells of the origin (then no offset of an edge can leave int8 and the rows need not check);
// xs4[f + p] = the p-th atom in bin order: wrapped coordinates, and in .w its local index j and the
// integer parts k_a of its coordinates, j | (k_0 + 16) << 16 | (k_1 + 16) << 21 | (k_2 + 16) << 26
// (mgb_pack): a row of the scan kernel needs nothing else about a candidate.
#pragma once
#include "common.cuh"
#include "cut_prep.cuh"

#define MGB_MAXBINS 4096           // bins of a structure (16 slabs per axis)

// slab of the wrapped coordinate x in [0, 1] (1.0 is the same point of the circle as 0.0; NaN -> slab 0)
__device__ __forceinline__ int mgb_axis(float x, int nb) {
    const int b = (int)__fmul_rn(x, (float)nb);
    return b >= nb ? b - nb : (b < 0 ? 0 : b);
}

__device__ __forceinline__ int mgb_bin(const float4 x, int nb0, int nb1, int nb2) {
    return (mgb_axis(x.x, nb0) * nb1 + mgb_axis(x.y, nb1)) * nb2 + mgb_axis(x.z, nb2);
}

// .w of a sorted entry from the packed integer parts of cut_prep.cuh (10 bits each, biased by 512; the
// structure's atoms are within 15 cells of the origin, else the entry is not used) and the atom's index
__device__ __forceinline__ int mgb_pack(int kk, int j) {
    return j | ((((kk & 1023) - 496) & 31) << 16) | (((((kk >> 10) & 1023) - 496) & 31) << 21) | (((((kk >> 20) & 1023) - 496) & 31) << 26);
}

struct BinArgs {
    const CutRec *rec;
    const float4 *xw4;         // [n_atoms] wrapped coordinates (cut_prep.cuh)
    float4 *xs4;               // [n_atoms] the same, in bin order inside each binned structure
    int *bin_start;            // [n_atoms + 2 n_struct + 2]
    const int *binlist;        // the structures to sort (written by the prep kernel), ctl[13] of them
    const unsigned *ctl;
    int n_struct;
};

#define MGB_BLOCK 512
#define MGB_HWORDS 24000           // 16-bit counters of a block: warps x (bins + 32)

// One block per listed structure.  The atoms are cut into W contiguous segments, one per warp (W <= 16, fewer when
// the structure has so many bins that W rows of counters do not fit); a warp counts its segment into its
// own row of 16-bit counters, the block turns the counters into cursors in (bin, warp) order, and every
// warp scatters its segment in index order: atoms of a bin stay sorted by index, whatever the timing.
__global__ void __launch_bounds__(MGB_BLOCK)
mg_cut_bin_kernel(const BinArgs A) {
    mg_grid_dependency_wait();                  // rec and xw4 are the prep kernel's
    __shared__ unsigned short h[MGB_HWORDS];
    __shared__ int s_wsum[MGB_BLOCK / 32];
    __shared__ int s_carry, s_bad;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_list = min((int)A.ctl[13], A.n_struct);   // (a batch of small cells: zero, every block leaves at once)
    for (int q = blockIdx.x; q < n_list; q += gridDim.x) {
        const int s = A.binlist[q];
        if ((unsigned)s >= (unsigned)A.n_struct) continue;
        const CutRec *R = A.rec + s;
        const int bins = R->bins;
        if (!(bins >> 24)) continue;            // (the same for every thread of the block)
        const int nb0 = bins & 0xFF, nb1 = (bins >> 8) & 0xFF, nb2 = (bins >> 16) & 0xFF, nbins = nb0 * nb1 * nb2;
        const int first = R->first, N = R->natoms;
        const float4 *x = A.xw4 + first;
        int *bs = A.bin_start + first + 2 * s;
        const int stride = nbins + 32;
        const int W = min(MGB_BLOCK / 32, MGB_HWORDS / stride);              // >= 5 (MGB_MAXBINS)
        const int seg = (((N + W - 1) / W) + 31) & ~31;
        const int j_lo = warp * seg, j_hi = min(N, j_lo + seg);
        __syncthreads();
        for (int q = tid; q < W * stride; q += MGB_BLOCK) h[q] = 0;
        if (tid == 0) { s_carry = 0; s_bad = 0; }
        __syncthreads();
        unsigned short *row = h + warp * stride;
        // ---- count: the lanes of a trip that share a bin add their number once
        bool bad = false;
        if (warp < W)
            for (int j0 = j_lo; j0 < j_hi; j0 += 32) {
                const int j = j0 + lane;
                int b = nbins + lane;                   // lanes past the end: a bin of their own
                if (j < j_hi) {
                    const float4 xj = x[j];
                    const int kk = __float_as_int(xj.w);
                    bad = bad || kk == 0 || abs((kk & 1023) - 512) > 15 || abs(((kk >> 10) & 1023) - 512) > 15 ||
                          abs(((kk >> 20) & 1023) - 512) > 15;
                    b = mgb_bin(xj, nb0, nb1, nb2);
                }
                const unsigned peers = __match_any_sync(0xFFFFFFFFu, b);
                if (lane == 31 - __clz(peers)) row[b] = (unsigned short)(row[b] + __popc(peers));
                __syncwarp();
            }
        if (bad) s_bad = 1;
        __syncthreads();
        // ---- counters -> cursors: bins in order, inside a bin the warps in order
        for (int b0 = 0; b0 < nbins; b0 += MGB_BLOCK) {
            const int b = b0 + tid;
            int tot = 0;
            if (b < nbins)
                for (int w = 0; w < W; ++w) tot += h[w * stride + b];
            int incl = tot;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                if (lane >= o) incl += t;
            }
            if (lane == 31) s_wsum[warp] = incl;
            __syncthreads();
            int off = s_carry;
            for (int w = 0; w < warp; ++w) off += s_wsum[w];
            int cur = off + incl - tot;
            if (b < nbins) {
                bs[b] = cur;
                for (int w = 0; w < W; ++w) {
                    const int c = h[w * stride + b];
                    h[w * stride + b] = (unsigned short)cur;
                    cur += c;
                }
            }
            __syncthreads();
            if (tid == MGB_BLOCK - 1) s_carry = off + incl;
            __syncthreads();
        }
        if (tid == 0) { bs[nbins] = N; bs[nbins + 1] = s_bad ? 0 : 1; }
        // ---- scatter, every warp its segment in index order
        if (warp < W)
            for (int j0 = j_lo; j0 < j_hi; j0 += 32) {
                const int j = j0 + lane;
                const bool v = j < j_hi;
                float4 xj = make_float4(0.f, 0.f, 0.f, 0.f);
                int b = nbins + lane;
                if (v) { xj = x[j]; b = mgb_bin(xj, nb0, nb1, nb2); }
                const unsigned peers = __match_any_sync(0xFFFFFFFFu, b);
                const int p = (int)row[b] + __popc(peers & ((1u << lane) - 1u));
                __syncwarp();
                if (lane == 31 - __clz(peers)) row[b] = (unsigned short)(p + 1);   // the last lane of the group leaves the cursor
                if (v) { xj.w = __int_as_float(mgb_pack(__float_as_int(xj.w), j)); A.xs4[first + p] = xj; }
                __syncwarp();
            }
    }
}
