// knn_bins.cu — k-nearest-neighbour graph (k <= 64) for batches of LARGE structures: one warp per source row, candidates
// from the fractional-coordinate cell list of cut_bins.cuh (SURVEY.md 8(a) K2 + K5; "route KNN for
// N > 64 through the same structure instead of the row-by-row fallback").
//
// mg_cut_prep_kernel (k > 0) picks the structure's search radius R (density, or the hint of the last mg_update_graph call)
// and, where the structure has more than MG_SMALL_MAX_ATOMS atoms and R / h_a < 1/2 on every axis (one image per pair),
// its slab counts; mg_cut_bin_kernel sorts the atoms by bin.  A row then looks at the 5 x 5 x 5 bins around its own
// (every image closer than R is in one of them, cut_bins.cuh): the nearest image of each candidate, d2 in FP32, hits
// (d2 < R^2) to the warp's stash; the k smallest by the generic selection of knn_pairs.cuh (FP32 keys, exact FP64 d2 for the
// k first and every hit FP32 cannot tell from the k-th, final order (d2, dst, tau)).  Alg. 1 line 4: a row whose k-th
// distance is not safely inside R — and every row of a structure without a cell list — goes to the growing-radius routine.
// Scanning all N atoms over 27 cells, that routine alone took 4.7 ms for the 20 430 rows of BASELINE configs[3].
//
// A module of its own (like knn_large.cu): nothing here touches the kernels of the headline.
#include "../../include/matgraph.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

#include "knn_bins_args.cuh"

namespace mg_knn_bins_tu {
#include "common.cuh"
#include "cut_prep.cuh"
#include "cut_bins.cuh"
#include "cutoff_pairs.cuh"
#include "knn_small.cuh"
#include "knn_pairs.cuh"

#define MGKB_HITS 640              // hits of a row the table area of the warp's shared memory holds (atom, offset bytes)
#define MGKB_BOX_MAX 512           // cells of a per-pair sub-box the rows of a structure without a cell list walk

// tau of a hit: codes = rint(u_a) mod 4 (2 bits per axis), ki = the source's packed integer parts (cut_prep.cuh), wj = .w
// of the target's sorted entry (cut_bins.cuh): tau = -rint(u) + k_i - k_j.
__device__ __forceinline__ void mgkb_tau(unsigned codes, int ki, int wj, int tau[3]) {
    tau[0] = 1 - (int)((codes + 1u) & 3u) + ((ki & 1023) - 512) - (((wj >> 16) & 31) - 16);
    tau[1] = 1 - (int)(((codes >> 2) + 1u) & 3u) + (((ki >> 10) & 1023) - 512) - (((wj >> 21) & 31) - 16);
    tau[2] = 1 - (int)(((codes >> 4) + 1u) & 3u) + (((ki >> 20) & 1023) - 512) - (((wj >> 26) & 31) - 16);
}

__device__ __forceinline__ unsigned mgkb_pack_tau(const int tau[3]) {
    return ((unsigned)(tau[0] + 128) << 16) | ((unsigned)(tau[1] + 128) << 8) | (unsigned)(tau[2] + 128);
}

// Hits of row i of structure s (first atom `first`) -> ks.stash (key = d2 bits | hit number) and the table area (atom,
// offset bytes).  Returns their number (more than MGKB_HITS: the caller gives up).
__device__ __forceinline__ int mgkb_find(KnnSmem &ks, const KnnBinsArgs &A, const CutRec *R, int s, int first, int i,
                                         const float a[9], float r2, int lane) {
    const float4 *xw = reinterpret_cast<const float4 *>(A.xw4) + first, *xs = reinterpret_cast<const float4 *>(A.xs4) + first;
    const int *bs = A.bin_start + first + 2 * s;
    const int nb0 = R->bins & 0xFF, nb1 = (R->bins >> 8) & 0xFF, nb2 = (R->bins >> 16) & 0xFF;
    const float4 xi = xw[i];
    // the row's columns of bins: exclusive prefix of their lengths, first run (start, length), start of the second
    int *tp = reinterpret_cast<int *>(&ks.xd[0][0]), *ta1 = tp + 32, *tn1 = tp + 64, *ta2 = tp + 96;
    const int s0 = nb0 > 1 ? 5 : 1, s1 = nb1 > 1 ? 5 : 1, ncol = s0 * s1;
    int a1 = 0, n1 = 0, a2 = 0, n2 = 0;
    if (lane < ncol) {
        const int q = s1 == 5 ? lane / 5 : lane;
        int c0 = mgb_axis(xi.x, nb0) + (s0 == 5 ? q - 2 : 0), c1 = mgb_axis(xi.y, nb1) + (s1 == 5 ? lane - 5 * q - 2 : 0);
        c0 += c0 < 0 ? nb0 : 0; c0 -= c0 >= nb0 ? nb0 : 0;
        c1 += c1 < 0 ? nb1 : 0; c1 -= c1 >= nb1 ? nb1 : 0;
        const int *col = bs + (c0 * nb1 + c1) * nb2;
        if (nb2 == 1) { a1 = col[0]; n1 = col[1] - a1; }
        else {
            const int lo = mgb_axis(xi.z, nb2) - 2, hi = lo + 4;            // nb2 >= 6: the five slabs are distinct
            if (lo < 0) { a1 = col[0]; n1 = col[hi + 1] - a1; a2 = col[nb2 + lo]; n2 = col[nb2] - a2; }
            else if (hi >= nb2) { a1 = col[lo]; n1 = col[nb2] - a1; a2 = col[0]; n2 = col[hi - nb2 + 1] - a2; }
            else { a1 = col[lo]; n1 = col[hi + 1] - a1; }
        }
    }
    int incl = n1 + n2;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += t;
    }
    const int total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    __syncwarp();
    tp[lane] = incl - (n1 + n2); ta1[lane] = a1; tn1[lane] = n1; ta2[lane] = a2;   // (lanes >= ncol: prefix = total)
    __syncwarp();
    // the candidates, lane <-> candidate: nearest image f = u - rint(u) (rint by the 1.5 * 2^23 trick, whose low
    // mantissa bits are rint(u) mod 4), d2 in FP32
    uint2 *meta = reinterpret_cast<uint2 *>(ks.w.T);
    const unsigned lt = (1u << lane) - 1u;
    int run = 0;
    for (int v0 = 0; v0 < total; v0 += 32) {
        const int v = v0 + lane;
        bool hit = false;
        unsigned long long key = 0ull;
        uint2 m = make_uint2(0u, 0u);
        if (v < total) {
            int c = 0;                                                        // the last column with tp[c] <= v
#pragma unroll
            for (int st = 16; st; st >>= 1) c += tp[c + st] <= v ? st : 0;    // (ncol <= 25: tp[26 .. 31] = total > v)
            const int r = v - tp[c], n1c = tn1[c];
            const float4 xj = xs[r < n1c ? ta1[c] + r : ta2[c] + (r - n1c)];
            const float u0 = __fsub_rn(xj.x, xi.x), u1 = __fsub_rn(xj.y, xi.y), u2 = __fsub_rn(xj.z, xi.z);
            const float m0 = __fadd_rn(u0, 12582912.f), m1 = __fadd_rn(u1, 12582912.f), m2 = __fadd_rn(u2, 12582912.f);
            const float f0 = __fsub_rn(u0, __fsub_rn(m0, 12582912.f)), f1 = __fsub_rn(u1, __fsub_rn(m1, 12582912.f)),
                        f2 = __fsub_rn(u2, __fsub_rn(m2, 12582912.f));
            const float vx = __fmaf_rn(f2, a[6], __fmaf_rn(f1, a[3], __fmul_rn(f0, a[0])));
            const float vy = __fmaf_rn(f2, a[7], __fmaf_rn(f1, a[4], __fmul_rn(f0, a[1])));
            const float vz = __fmaf_rn(f2, a[8], __fmaf_rn(f1, a[5], __fmul_rn(f0, a[2])));
            const float d2 = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmul_rn(vx, vx)));
            hit = d2 < r2 && (__float_as_int(xj.w) & 0xFFFF) != i;           // (i, i, 0) is not an edge (R3)
            key = (unsigned long long)__float_as_uint(d2) << 32;
            if (hit) {                                                        // the hit's atom and offset
                int tau[3];
                mgkb_tau((__float_as_uint(m0) & 3u) | ((__float_as_uint(m1) & 3u) << 2) | ((__float_as_uint(m2) & 3u) << 4),
                         __float_as_int(xi.w), __float_as_int(xj.w), tau);
                m = make_uint2(__float_as_uint(xj.w) & 0xFFFFu, mgkb_pack_tau(tau));
            }
        }
        const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
        if (hit) {
            const int pos = run + __popc(bal & lt);
            if (pos < MGKB_HITS) { ks.stash[pos] = key | (unsigned)pos; meta[pos] = m; }
        }
        run += __popc(bal);
    }
    __syncwarp();
    return run;
}
// The same for a structure WITHOUT a cell list (several images per pair: R / h_a >= 1/2 on some axis, or atoms far from
// the origin): lanes over (target, cell) of the per-pair sub-box of cut_prep.cuh — u = x_j - x_i (wrapped), first cell
// lo_a = floor(-rho_a - u_a) + 1, m_a cells from there — every target, no pruning.  Offsets outside int8 or a non-finite
// coordinate: gives up (the growing-radius routine decides and reports).
__device__ __forceinline__ int mgkb_find_box(KnnSmem &ks, const KnnBinsArgs &A, const CutRec *R, int first, int N, int i,
                                             const float a[9], float r2, int lane) {
    const float4 *xw = reinterpret_cast<const float4 *>(A.xw4) + first;
    const float4 xi = xw[i];
    const int ki = __float_as_int(xi.w);
    const float rho0 = R->rho[0], rho1 = R->rho[1], rho2 = R->rho[2];
    const int m1 = (R->m >> 8) & 0xFF, m2 = (R->m >> 16) & 0xFF, mloc = R->mloc, M12 = m1 * m2;
    const bool wide = mloc >= 32;
    const int J = wide ? 1 : 32 / mloc, jl = wide ? 0 : lane / mloc, npass = wide ? (mloc + 31) >> 5 : 1;
    uint2 *meta = reinterpret_cast<uint2 *>(ks.w.T);
    const unsigned lt = (1u << lane) - 1u;
    int run = 0;
    bool bad = ki == 0;
    for (int ps = 0; ps < npass; ++ps) {
        const int c = wide ? 32 * ps + lane : lane - jl * mloc;
        const bool cv = wide ? c < mloc : jl < J;
        const int t0 = c / M12, rr = c - t0 * M12, t1 = rr / m2, t2 = rr - t1 * m2;
        for (int j0 = 0; j0 < N; j0 += J) {
            const int j = j0 + jl;
            bool hit = false;
            unsigned long long key = 0ull;
            uint2 m = make_uint2(0u, 0u);
            if (cv && j < N) {
                const float4 xj = xw[j];
                const int kj = __float_as_int(xj.w);
                const float u0 = __fsub_rn(xj.x, xi.x), u1 = __fsub_rn(xj.y, xi.y), u2 = __fsub_rn(xj.z, xi.z);
                const float e0 = floorf(__fsub_rn(-rho0, u0)) + 1.f, e1 = floorf(__fsub_rn(-rho1, u1)) + 1.f,
                            e2 = floorf(__fsub_rn(-rho2, u2)) + 1.f;
                const float f0 = __fadd_rn(u0, e0 + (float)t0), f1 = __fadd_rn(u1, e1 + (float)t1), f2 = __fadd_rn(u2, e2 + (float)t2);
                const float vx = __fmaf_rn(f2, a[6], __fmaf_rn(f1, a[3], __fmul_rn(f0, a[0])));
                const float vy = __fmaf_rn(f2, a[7], __fmaf_rn(f1, a[4], __fmul_rn(f0, a[1])));
                const float vz = __fmaf_rn(f2, a[8], __fmaf_rn(f1, a[5], __fmul_rn(f0, a[2])));
                const float d2 = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmul_rn(vx, vx)));
                int tau[3];
                tau[0] = (int)e0 + t0 + (ki & 1023) - (kj & 1023);
                tau[1] = (int)e1 + t1 + ((ki >> 10) & 1023) - ((kj >> 10) & 1023);
                tau[2] = (int)e2 + t2 + ((ki >> 20) & 1023) - ((kj >> 20) & 1023);
                bad = bad || kj == 0 || tau[0] < -127 || tau[1] < -127 || tau[2] < -127 || tau[0] > 127 || tau[1] > 127 || tau[2] > 127;
                hit = !bad && d2 < r2 && !(i == j && (tau[0] | tau[1] | tau[2]) == 0);   // (i, i, 0) is not an edge (R3)
                key = (unsigned long long)__float_as_uint(d2) << 32;
                m = make_uint2((unsigned)j, mgkb_pack_tau(tau));
            }
            const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
            if (hit) {
                const int pos = run + __popc(bal & lt);
                if (pos < MGKB_HITS) { ks.stash[pos] = key | (unsigned)pos; meta[pos] = m; }
            }
            run += __popc(bal);
        }
    }
    __syncwarp();
    return __any_sync(0xFFFFFFFFu, bad) ? MGKB_HITS + 1 : run;
}

// One row through the cell list.  Returns false if the row did not settle inside R (the caller hands it to the growing-
// radius routine); *dk: its k-th distance.
__device__ __forceinline__ bool mgkb_row(KnnSmem &ks, const KnnBinsArgs &A, const CutRec *R, int s, int first, int N, int i,
                                         bool binned, int lane, float *dk) {
    const int K = A.k, gi = first + i;
    const float *lat = A.lattice + 9 * (size_t)s;
    float a[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) a[c] = __ldg(lat + c);
    const float rad = R->radius, r2 = __fmul_rn(rad, rad);
    // FP32 error bound of d2 near R^2 (R23): every image with true d2 < R^2 - win is a hit; a k-th key below
    // R^2 - 2 win is safe
    const float win = 1.1920929e-7f * (2.f * rad * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * rad * rad);
    const float lim2 = __fmaf_rn(-2.f, win, r2);
    const int total = binned ? mgkb_find(ks, A, R, s, first, i, a, r2, lane) : mgkb_find_box(ks, A, R, first, N, i, a, r2, lane);
    if (total < K || total > MGKB_HITS) return false;
    // the 32 smallest FP32 keys (Alg. 2's "sort, keep k", 32 at a time)
    mg_key key = mg_sort32(lane < total ? ks.stash[lane] : MG_KEY_INF, lane);
    for (int c = 32; c < total; c += 32) {
        mg_key keys1[1] = {key};
        mg_knn_merge<1>(keys1, c + lane < total ? ks.stash[c + lane] : MG_KEY_INF, lane);
        key = keys1[0];
    }
    const mg_key kth = __shfl_sync(0xFFFFFFFFu, key, K - 1);
    const float kth_d2 = __uint_as_float((unsigned)(kth >> 32));
    if (kth == MG_KEY_INF || !(kth_d2 < lim2)) return false;
    // exact FP64 d2 of the k first and of every hit FP32 cannot tell from the k-th; final order (d2, dst, tau)
    const bool amb = lane >= K && key != MG_KEY_INF && __uint_as_float((unsigned)(key >> 32)) <= __fmaf_rn(2.f, win, kth_d2);
    const int nsel = K + __popc(__ballot_sync(0xFFFFFFFFu, amb));
    const uint2 *meta = reinterpret_cast<const uint2 *>(ks.w.T);
    int j = 0, tau[3] = {0, 0, 0};
    unsigned long long ord = ~0ull;
    double dd = 1e300, vv[3] = {0.0, 0.0, 0.0};
    if (lane < nsel) {
        const uint2 m = meta[(unsigned)key];                                 // (the key's low word is the hit's number)
        j = (int)m.x;
        tau[0] = (int)(m.y >> 16) - 128; tau[1] = (int)((m.y >> 8) & 0xFFu) - 128; tau[2] = (int)(m.y & 0xFFu) - 128;
        double xi[3], xj[3], L[9];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            xi[c] = (double)A.pos[3 * (size_t)gi + c];
            xj[c] = (double)A.pos[3 * (size_t)(first + j) + c];
        }
#pragma unroll
        for (int c = 0; c < 9; ++c) L[c] = (double)a[c];
        dd = mg_knn_exact_d2(xi, xj, tau[0], tau[1], tau[2], L, vv);
        ord = ((unsigned long long)(unsigned)j << 24) | ((unsigned)(tau[0] + 128) << 16) | ((unsigned)(tau[1] + 128) << 8) |
              (unsigned)(tau[2] + 128);
    }
    int rank = 0;
    for (int l = 0; l < nsel; ++l) {
        const double od = __shfl_sync(0xFFFFFFFFu, dd, l);
        const unsigned long long oo = __shfl_sync(0xFFFFFFFFu, ord, l);
        rank += (od < dd || (od == dd && oo < ord)) ? 1 : 0;
    }
    float dkk = 0.f;
    if (lane < nsel && rank < K) {
        const long long e = (long long)K * gi + rank;
        A.src[e] = gi;
        A.dst[e] = first + j;
        A.offset[3 * e] = (int8_t)tau[0]; A.offset[3 * e + 1] = (int8_t)tau[1]; A.offset[3 * e + 2] = (int8_t)tau[2];
        A.vec[3 * e] = (float)vv[0]; A.vec[3 * e + 1] = (float)vv[1]; A.vec[3 * e + 2] = (float)vv[2];
        if (A.dist) A.dist[e] = __fsqrt_rn((float)dd);
        if (rank == K - 1) dkk = __fsqrt_ru(__double2float_ru(dd));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dkk = fmaxf(dkk, __shfl_xor_sync(0xFFFFFFFFu, dkk, o));
    *dk = dkk;
    return true;
}
// The same with KPL sorted FP32 keys per lane (k <= 32 KPL; slot q of lane l holds rank 32 q + l), for 32 < k <= 64.  Out
// of line and apart from mgkb_row: as one template, inlined, the rows of k <= 32 ran 13 % slower (config 3, k = 12: 94.8
// against 82.5 us per call).
template <int KPL>
__device__ __noinline__ bool mgkb_row_wide(KnnSmem &ks, const KnnBinsArgs &A, const CutRec *R, int s, int first, int N, int i,
                                         bool binned, int lane, float *dk) {
    const int K = A.k, gi = first + i;
    const float *lat = A.lattice + 9 * (size_t)s;
    float a[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) a[c] = __ldg(lat + c);
    const float rad = R->radius, r2 = __fmul_rn(rad, rad);
    // FP32 error bound of d2 near R^2 (R23): every image with true d2 < R^2 - win is a hit; a k-th key below
    // R^2 - 2 win is safe
    const float win = 1.1920929e-7f * (2.f * rad * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * rad * rad);
    const float lim2 = __fmaf_rn(-2.f, win, r2);
    const int total = binned ? mgkb_find(ks, A, R, s, first, i, a, r2, lane) : mgkb_find_box(ks, A, R, first, N, i, a, r2, lane);
    if (total < K || total > MGKB_HITS) return false;
    // the 32 KPL smallest FP32 keys (Alg. 2's "sort, keep k", 32 at a time)
    mg_key keys[KPL];
    if (KPL == 1) {
        keys[0] = mg_sort32(lane < total ? ks.stash[lane] : MG_KEY_INF, lane);
        for (int c = 32; c < total; c += 32) mg_knn_merge<KPL>(keys, c + lane < total ? ks.stash[c + lane] : MG_KEY_INF, lane);
    } else {
#pragma unroll
        for (int q = 0; q < KPL; ++q) keys[q] = MG_KEY_INF;
        for (int c = 0; c < total; c += 32) mg_knn_merge<KPL>(keys, c + lane < total ? ks.stash[c + lane] : MG_KEY_INF, lane);
    }
    const mg_key kth = __shfl_sync(0xFFFFFFFFu, keys[(K - 1) >> 5], (K - 1) & 31);
    const float kth_d2 = __uint_as_float((unsigned)(kth >> 32));
    if (kth == MG_KEY_INF || !(kth_d2 < lim2)) return false;
    // exact FP64 d2 of the k first and of every hit FP32 cannot tell from the k-th; final order (d2, dst, tau)
    int nsel = K;
#pragma unroll
    for (int q = 0; q < KPL; ++q) {
        const bool amb = 32 * q + lane >= K && keys[q] != MG_KEY_INF &&
                         __uint_as_float((unsigned)(keys[q] >> 32)) <= __fmaf_rn(2.f, win, kth_d2);
        nsel += __popc(__ballot_sync(0xFFFFFFFFu, amb));
    }
    const uint2 *meta = reinterpret_cast<const uint2 *>(ks.w.T);
    int j[KPL], tau[KPL][3];
    unsigned long long ord[KPL];
    double dd[KPL], vv[KPL][3];
    double xi[3], L[9];
#pragma unroll
    for (int c = 0; c < 3; ++c) xi[c] = (double)A.pos[3 * (size_t)gi + c];
#pragma unroll
    for (int c = 0; c < 9; ++c) L[c] = (double)a[c];
#pragma unroll
    for (int q = 0; q < KPL; ++q) {
        j[q] = 0; tau[q][0] = tau[q][1] = tau[q][2] = 0; ord[q] = ~0ull; dd[q] = 1e300;
        vv[q][0] = vv[q][1] = vv[q][2] = 0.0;
        if (32 * q + lane < nsel) {
            const uint2 m = meta[(unsigned)keys[q]];                         // (the key's low word is the hit's number)
            j[q] = (int)m.x;
            tau[q][0] = (int)(m.y >> 16) - 128; tau[q][1] = (int)((m.y >> 8) & 0xFFu) - 128; tau[q][2] = (int)(m.y & 0xFFu) - 128;
            double xj[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) xj[c] = (double)A.pos[3 * (size_t)(first + j[q]) + c];
            dd[q] = mg_knn_exact_d2(xi, xj, tau[q][0], tau[q][1], tau[q][2], L, vv[q]);
            ord[q] = ((unsigned long long)(unsigned)j[q] << 24) | m.y;
        }
    }
    // (the FP32 keys mostly are the final order already: one look at each entry's predecessor tells, and only a row where
    // FP64 or the tie-break disagrees counts, as in knn_small.cuh)
    int rank[KPL];
    bool ok = true;
#pragma unroll
    for (int q = 0; q < KPL; ++q) {
        rank[q] = 32 * q + lane;
        double pd = __shfl_up_sync(0xFFFFFFFFu, dd[q], 1);
        unsigned long long po = __shfl_up_sync(0xFFFFFFFFu, ord[q], 1);
        if (q > 0) {
            const double ld = __shfl_sync(0xFFFFFFFFu, dd[q > 0 ? q - 1 : 0], 31);
            const unsigned long long lo = __shfl_sync(0xFFFFFFFFu, ord[q > 0 ? q - 1 : 0], 31);
            if (lane == 0) { pd = ld; po = lo; }
        }
        if (32 * q + lane < nsel) ok = ok && (32 * q + lane == 0 || pd < dd[q] || (pd == dd[q] && po < ord[q]));
    }
    if (!__all_sync(0xFFFFFFFFu, ok)) {
#pragma unroll
        for (int q = 0; q < KPL; ++q) rank[q] = 0;
#pragma unroll
        for (int q2 = 0; q2 < KPL; ++q2) {
            const int cnt2 = min(32, nsel - 32 * q2);
            for (int l = 0; l < cnt2; ++l) {
                const double od = __shfl_sync(0xFFFFFFFFu, dd[q2], l);
                const unsigned long long oo = __shfl_sync(0xFFFFFFFFu, ord[q2], l);
#pragma unroll
                for (int q = 0; q < KPL; ++q) rank[q] += (od < dd[q] || (od == dd[q] && oo < ord[q])) ? 1 : 0;
            }
        }
    }
    float dkk = 0.f;
#pragma unroll
    for (int q = 0; q < KPL; ++q)
        if (32 * q + lane < nsel && rank[q] < K) {
            const long long e = (long long)K * gi + rank[q];
            A.src[e] = gi;
            A.dst[e] = first + j[q];
            A.offset[3 * e] = (int8_t)tau[q][0]; A.offset[3 * e + 1] = (int8_t)tau[q][1]; A.offset[3 * e + 2] = (int8_t)tau[q][2];
            A.vec[3 * e] = (float)vv[q][0]; A.vec[3 * e + 1] = (float)vv[q][1]; A.vec[3 * e + 2] = (float)vv[q][2];
            if (A.dist) A.dist[e] = __fsqrt_rn((float)dd[q]);
            if (rank[q] == K - 1) dkk = __fsqrt_ru(__double2float_ru(dd[q]));
        }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dkk = fmaxf(dkk, __shfl_xor_sync(0xFFFFFFFFu, dkk, o));
    *dk = dkk;
    return true;
}

// The growing-radius routine of knn_small.cuh for one row with two sorted keys per lane (32 < k <= 64): what
// mg_knn_row_fallback of knn_pairs.cuh is for k <= 32, the same steps.
__device__ __noinline__ void mgkb_grow2(KnnSmem &ks, const KnnPairsArgs &A, int s, int first, int N, int i, int lane) {
    const float *lat9 = A.lattice + 9 * (size_t)s;
    float4 *sp = reinterpret_cast<float4 *>(ks.w.T);
    mg_key *buf = reinterpret_cast<mg_key *>(ks.w.T + MG_SMALL_MAX_ATOMS);
    StructRec R;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
    __syncwarp();
    const bool big = N > MG_SMALL_MAX_ATOMS;      // too large to stage: positions on the fly
    for (int j = lane; j < N; j += 32) {
        const float *x = A.pos + 3 * (size_t)(first + j);
        const float x0 = x[0], x1 = x[1], x2 = x[2];
        lo[0] = fminf(lo[0], x0); lo[1] = fminf(lo[1], x1); lo[2] = fminf(lo[2], x2);
        hi[0] = fmaxf(hi[0], x0); hi[1] = fmaxf(hi[1], x1); hi[2] = fmaxf(hi[2], x2);
        if (big) continue;
        float4 p;
        p.x = __fmaf_rn(x2, lat9[6], __fmaf_rn(x1, lat9[3], __fmul_rn(x0, lat9[0])));
        p.y = __fmaf_rn(x2, lat9[7], __fmaf_rn(x1, lat9[4], __fmul_rn(x0, lat9[1])));
        p.z = __fmaf_rn(x2, lat9[8], __fmaf_rn(x1, lat9[5], __fmul_rn(x0, lat9[2])));
        p.w = 0.f;
        sp[j] = p;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xFFFFFFFFu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xFFFFFFFFu, hi[a], o));
        }
    __syncwarp();
    float lat[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) lat[c] = lat9[c];
    double vol = 1.0, h[3] = {1.0, 1.0, 1.0};
    mg_cell_spacings(lat, &vol, h);                   // the lattice is valid: prep checked it
    R.first = first;
    R.natoms = N;
    R.volume = (float)vol;
    R.err = 0u;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        R.xmin[a] = lo[a];
        R.xmax[a] = hi[a];
        R.h_dn[a] = __double2float_rd(h[a] * (1.0 - 1e-6));
        R.invh_up[a] = __double2float_ru((1.0 + 1e-6) / h[a]);
        R.amax[a] = fmaxf(fabsf(lat[3 * a]), fmaxf(fabsf(lat[3 * a + 1]), fabsf(lat[3 * a + 2])));
    }
    KnnArgs K;
    K.pos = A.pos; K.lattice = A.lattice; K.struct_ptr = A.struct_ptr;
    K.n_struct = A.n_struct; K.n_atoms = A.n_atoms; K.k = A.k;
    K.row_ptr = A.row_ptr; K.src = A.src; K.dst = A.dst; K.offset = A.offset;
    K.vec = A.vec; K.dist = A.dist; K.n_edges = A.n_edges;
    float *slot = reinterpret_cast<float *>(ks.w.T + MG_SMALL_MAX_ATOMS + 16);   // k-th distance comes back here
    K.radius_hint = A.hint ? slot - (first + i) : nullptr; K.use_hint = 0;
    K.rec = nullptr; K.atom_struct = nullptr; K.ctl = nullptr; K.status = A.status;
    mg_knn_source<2>(K, R, lat9, big ? nullptr : sp, buf, i, lane);
    __syncwarp();
    if (A.hint && lane == 0) atomicMax(reinterpret_cast<int *>(A.hint + s), __float_as_int(*slot));
    __syncwarp();
}

__global__ void __launch_bounds__(MG_BLOCK)
mg_knn_bins_kernel(const __grid_constant__ KnnBinsArgs A) {
    mg_grid_dependency_wait();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    KnnSmem &ks = reinterpret_cast<KnnSmem *>(smem_raw)[warp];
    const int K = A.k;
    for (long long t = (long long)blockIdx.x * MG_BLOCK + threadIdx.x; t <= A.n_atoms; t += (long long)gridDim.x * MG_BLOCK)
        A.row_ptr[t] = (int)((long long)K * t);
    if (blockIdx.x == 0 && threadIdx.x == 0) *A.n_edges = (long long)K * A.n_atoms;
    // what the growing-radius routine wants to know (knn_pairs.cuh)
    KnnPairsArgs P;
    P.pos = A.pos; P.lattice = A.lattice; P.struct_ptr = A.struct_ptr; P.n_struct = A.n_struct; P.n_atoms = A.n_atoms; P.k = K;
    P.row_ptr = A.row_ptr; P.src = A.src; P.dst = A.dst; P.offset = A.offset; P.vec = A.vec; P.dist = A.dist;
    P.n_edges = A.n_edges; P.hint = A.hint; P.rec = reinterpret_cast<const CutRec *>(A.rec); P.bpre = nullptr; P.n_blocks = 0;
    P.n_warps = 0; P.status = A.status; P.dbg = nullptr;
    const CutRec *rec = reinterpret_cast<const CutRec *>(A.rec);
    const int gw = (int)blockIdx.x * MG_WARPS + warp, nw = (int)gridDim.x * MG_WARPS;
    for (int g = gw; g < A.n_atoms; g += nw) {
        // the row's structure: the last s with struct_ptr[s] <= g (empty structures share their start with the next one)
        int lo = 0, hi = A.n_struct;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(A.struct_ptr + mid) <= g) lo = mid; else hi = mid;
        }
        const int s = lo;
        const CutRec *R = rec + s;
        const int first = R->first, N = R->natoms, i = g - first;
        if (R->mloc <= 0) {                    // invalid lattice / positions: placeholder row (src = dst, zero vec); mg_check reports
            for (int e = lane; e < K; e += 32) {
                const long long o = (long long)K * g + e;
                A.src[o] = g; A.dst[o] = g;
                A.offset[3 * o] = 0; A.offset[3 * o + 1] = 0; A.offset[3 * o + 2] = 0;
                A.vec[3 * o] = 0.f; A.vec[3 * o + 1] = 0.f; A.vec[3 * o + 2] = 0.f;
                if (A.dist) A.dist[o] = 0.f;
            }
            continue;
        }
        // a cell list, and every atom of the structure finite and within 15 cells of the origin (cut_bins.cuh)
        const int bins = R->bins;
        bool binned = (bins >> 24) != 0;
        if (binned) binned = A.bin_start[first + 2 * s + (bins & 0xFF) * ((bins >> 8) & 0xFF) * ((bins >> 16) & 0xFF) + 1] != 0;
        float dk = 0.f;
        __syncwarp();
        // (no cell list: every target over the per-pair sub-box, unless that is thousands of cells)
        const bool list = binned || R->mloc <= MGKB_BOX_MAX;
        if (list && (K <= 32 ? mgkb_row(ks, A, R, s, first, N, i, binned, lane, &dk)
                             : mgkb_row_wide<2>(ks, A, R, s, first, N, i, binned, lane, &dk))) {
            if (A.hint && lane == 0 && dk > 0.f) atomicMax(reinterpret_cast<int *>(A.hint + s), __float_as_int(dk));
            continue;
        }
        __syncwarp();
        if (K <= 32) mg_knn_row_fallback(ks, P, s, first, N, i, lane);    // (the growing-radius routine; sets the hint itself)
        else mgkb_grow2(ks, P, s, first, N, i, lane);
    }
}
}  // namespace mg_knn_bins_tu

using mg_knn_bins_tu::KnnSmem;

// Opt the kernel in to its shared memory; *occ: resident CTAs per SM.  Call once per device, that device current.
__attribute__((visibility("hidden"))) cudaError_t mg_knn_bins_setup(int *occ) {
    const size_t smem = MG_WARPS * sizeof(KnnSmem);
    cudaError_t e = cudaFuncSetAttribute(mg_knn_bins_tu::mg_knn_bins_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, mg_knn_bins_tu::mg_knn_bins_kernel, MG_BLOCK, smem);
}

// `pdl`: programmatic dependent launch (the kernel waits for the bin kernel before it reads anything).
__attribute__((visibility("hidden"))) cudaError_t mg_knn_bins_launch(const KnnBinsArgs *a, int grid, cudaStream_t st, int pdl) {
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
    return cudaLaunchKernelEx(&cfg, mg_knn_bins_tu::mg_knn_bins_kernel, *a);
}
