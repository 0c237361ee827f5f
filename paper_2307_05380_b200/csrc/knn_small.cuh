// knn_small.cuh — k-nearest-neighbour multigraph by a growing-radius search, one warp per source atom (k up to 64;
// structures of <= MG_SMALL_MAX_ATOMS atoms are staged in shared memory, larger ones are read in place).
//
// Problem: per source the k smallest keys (d, dst, tau_x, tau_y, tau_z) over all periodic images
// except (i,i,0) (Alg. 2 lines 2-5, made deterministic: DESIGN.md R2, R8).
// Method (Alg. 1, re-designed): one WARP per source atom, no block-level
// synchronisation.  The ordered stack of Alg. 2 lives in registers — a sorted list of 64-bit keys
// (d2 bits | dst | tau), one or two per lane.  The warp explores the box of cells that provably
// holds every image closer than a search radius R (n_a = floor(R/h_a + spread_a); every unexplored
// image is farther than R_safe = min_a (n_a + 1 - spread_a) h_a >= R: closest_distance of Alg. 1
// line 4, R11): lanes <-> cells, loop over target atoms j, candidates with d <= R that
// beat the current k-th key are appended to a 32-entry shared-memory buffer; a full buffer is
// bitonic-sorted and merged into the list (Alg. 2's "concatenate, sort, keep k", batched).
// If fewer than k images lie within R the radius grows and the search starts again (Alg. 1's
// while loop).  R starts from the atomic density, or from the previous k-th distance when
// mg_update_graph supplies it.  The FP32 keys select the k entries; their final order and the
// emitted vec / dist use the exact FP64 distance.
#pragma once
#include "common.cuh"

#define MG_KEY_INF 0xFFFFFFFFFFFFFFFFull

struct KnnArgs {
    const float *pos;
    const float *lattice;
    const int32_t *struct_ptr;
    int n_struct, n_atoms;
    int k;
    int32_t *row_ptr, *src, *dst;
    int8_t *offset;
    float *vec, *dist;
    long long *n_edges;
    float *radius_hint;         // [n_atoms] k-th distance of the previous call, or NULL
    int use_hint;               // read radius_hint as the first search radius
    const StructRec *rec;
    const int32_t *atom_struct;
    unsigned *ctl;              // [2] next atom, [3] CTAs done
    unsigned *status;
};

typedef unsigned long long mg_key;

__device__ __forceinline__ mg_key mg_kmin(mg_key a, mg_key b) { return a < b ? a : b; }
__device__ __forceinline__ mg_key mg_kmax(mg_key a, mg_key b) { return a < b ? b : a; }

// ascending bitonic sort of one key per lane
__device__ __forceinline__ mg_key mg_sort32(mg_key v, int lane) {
#pragma unroll
    for (int k2 = 2; k2 <= 32; k2 <<= 1) {      // "flip" form: the lower lane of every exchange takes the minimum
        {
            const mg_key p = __shfl_xor_sync(0xFFFFFFFFu, v, k2 - 1);
            v = (lane & (k2 >> 1)) == 0 ? mg_kmin(v, p) : mg_kmax(v, p);
        }
#pragma unroll
        for (int j = k2 >> 2; j > 0; j >>= 1) {
            const mg_key p = __shfl_xor_sync(0xFFFFFFFFu, v, j);
            v = (lane & j) == 0 ? mg_kmin(v, p) : mg_kmax(v, p);
        }
    }
    return v;
}

// ascending sort of a bitonic sequence
__device__ __forceinline__ mg_key mg_sort_bitonic(mg_key v, int lane) {
#pragma unroll
    for (int j = 16; j > 0; j >>= 1) {
        const mg_key p = __shfl_xor_sync(0xFFFFFFFFu, v, j);
        v = (lane & j) == 0 ? mg_kmin(v, p) : mg_kmax(v, p);
    }
    return v;
}

// Merge up to 32 unsorted keys (one per lane, MG_KEY_INF = none) into the sorted list
// (slot s of lane l holds rank 32 s + l); what falls off the end is dropped.
template <int KPL>
__device__ __forceinline__ void mg_knn_merge(mg_key (&keys)[KPL], mg_key b, int lane) {
    b = mg_sort32(b, lane);
    mg_key rb = __shfl_sync(0xFFFFFFFFu, b, 31 - lane);
    if (KPL == 1) {
        keys[0] = mg_sort_bitonic(mg_kmin(keys[0], rb), lane);
    } else {
        mg_key t = mg_sort_bitonic(mg_kmin(keys[KPL - 1], rb), lane);   // 32 smallest of (top slot, b)
        const mg_key rt = __shfl_sync(0xFFFFFFFFu, t, 31 - lane);
        const mg_key lo = mg_kmin(keys[0], rt), hi = mg_kmax(keys[0], rt);
        keys[0] = mg_sort_bitonic(lo, lane);
        keys[KPL - 1] = mg_sort_bitonic(hi, lane);
    }
}

// Key of the growing-radius search: FP32 d2 bits | j * ncell + c, c the index of the image's cell in
// the explored box (lexicographic in tau), so that the low word orders like (dst, tau_x, tau_y, tau_z)
// for structures of any size (an 8-bit dst field would wrap above 256 atoms).  The caller makes sure
// that natoms * ncell fits 32 bits.
__device__ __forceinline__ mg_key mg_knn_key(float d2, unsigned tie) {
    return ((mg_key)__float_as_uint(d2) << 32) | (mg_key)tie;
}

// FP32 cartesian position of atom j of the structure (x . L, the same arithmetic as the staged copy).
__device__ __forceinline__ float4 mg_knn_cart(const float *xs, const float *lat9, int j) {
    const float x0 = xs[3 * j], x1 = xs[3 * j + 1], x2 = xs[3 * j + 2];
    float4 p;
    p.x = __fmaf_rn(x2, lat9[6], __fmaf_rn(x1, lat9[3], __fmul_rn(x0, lat9[0])));
    p.y = __fmaf_rn(x2, lat9[7], __fmaf_rn(x1, lat9[4], __fmul_rn(x0, lat9[1])));
    p.z = __fmaf_rn(x2, lat9[8], __fmaf_rn(x1, lat9[5], __fmul_rn(x0, lat9[2])));
    p.w = 0.f;
    return p;
}

// Search + emit for source atom gi = R.first + i; sp = this warp's cartesian positions of the
// structure (nullptr: evaluated on the fly from pos, for structures too large to stage),
// buf = this warp's 32-entry candidate buffer.  Called by a full warp.
template <int KPL>
__device__ inline void mg_knn_source(const KnnArgs &A, const StructRec &R, const float *lat9,
                                     const float4 *sp, mg_key *buf, int i, int lane) {
    const int N = R.natoms, k = A.k, gi = R.first + i;
    const int kslot = (k - 1) >> 5, klane = (k - 1) & 31;
    const float *xs = A.pos + 3 * (size_t)R.first;
    const float4 pi = sp ? sp[i] : mg_knn_cart(xs, lat9, i);
    float a[3][3], lo_off[3], hi_off[3], spread[3];
    float xabs = 1.f;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
#pragma unroll
        for (int c = 0; c < 3; ++c) a[r][c] = lat9[3 * r + c];
        const float xi = xs[3 * i + r];
        lo_off[r] = R.xmin[r] - xi;                  // only used for pruning, with h rounded down
        hi_off[r] = R.xmax[r] - xi;                  // and a safety factor
        spread[r] = __fadd_ru(R.xmax[r], -R.xmin[r]);
        xabs = fmaxf(xabs, fmaxf(fabsf(R.xmin[r]), fabsf(R.xmax[r])));
    }
    float Rad;
    if (A.use_hint && A.radius_hint[gi] > 0.f) Rad = 1.03f * A.radius_hint[gi] + 1e-3f;
    else Rad = 1.25f * cbrtf(0.2387324f * (float)(k + 1) * R.volume / (float)N);
    mg_key keys[KPL];
    mg_key thr;
    bool failed = false, too_big = false;
    int n[3] = {0, 0, 0};
    for (;;) {
        // ---- box that holds every image with d < Rad
        float rsafe = 3.0e38f, M = 0.f;
        bool range_ok = true;
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            float nn = floorf(__fmaf_ru(Rad, R.invh_up[r], spread[r]));
            if (!(nn <= 127.f)) { range_ok = false; nn = 127.f; }
            n[r] = (int)nn;
            rsafe = fminf(rsafe, __fmul_rd(__fadd_rd(nn + 1.f, -spread[r]), R.h_dn[r]));
            M += (nn + 2.f * xabs) * R.amax[r];
        }
        const float W = 3.5f * 12.f * 5.9604645e-8f * M * 1.01f;   // FP32 error bound of a distance
        const float lim = fminf(Rad, rsafe);
        const float lim2 = __fmul_ru(lim, lim);
#pragma unroll
        for (int s = 0; s < KPL; ++s) keys[s] = MG_KEY_INF;
        thr = MG_KEY_INF;
        float thr_d2 = lim2;
        int nb = 0;
        const int D1 = 2 * n[1] + 1, D2 = 2 * n[2] + 1;
        const int ncell = (2 * n[0] + 1) * D1 * D2;
        if ((unsigned long long)N * (unsigned long long)ncell > 0xFFFFFFFFull) { too_big = true; break; }
        const float inv12 = 1.f / (float)(D1 * D2), inv2 = 1.f / (float)D2;
        for (int c0 = 0; c0 < ncell; c0 += 32) {
            const int c = c0 + lane;
            const bool big = ncell >= (1 << 20);            // float reciprocal is exact below 2^20 only
            const int u0 = big ? c / (D1 * D2) : __float2int_rz(((float)c + 0.5f) * inv12), rem = c - u0 * (D1 * D2);
            const int u1 = big ? rem / D2 : __float2int_rz(((float)rem + 0.5f) * inv2);
            const int t0 = u0 - n[0], t1 = u1 - n[1], t2 = rem - u1 * D2 - n[2];
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            // lower bound of the distance to any image in this cell: max_a gap_a h_a
            const float g0 = fmaxf(0.f, fmaxf(f0 + lo_off[0], -(f0 + hi_off[0]))) * R.h_dn[0];
            const float g1 = fmaxf(0.f, fmaxf(f1 + lo_off[1], -(f1 + hi_off[1]))) * R.h_dn[1];
            const float g2 = fmaxf(0.f, fmaxf(f2 + lo_off[2], -(f2 + hi_off[2]))) * R.h_dn[2];
            const float lb = fmaxf(g0, fmaxf(g1, g2)) * 0.99999f;
            const bool alive = c < ncell && lb * lb <= thr_d2;
            if (!__any_sync(0xFFFFFFFFu, alive)) continue;
            const float Tx = __fmaf_rn(f2, a[2][0], __fmaf_rn(f1, a[1][0], __fmul_rn(f0, a[0][0])));
            const float Ty = __fmaf_rn(f2, a[2][1], __fmaf_rn(f1, a[1][1], __fmul_rn(f0, a[0][1])));
            const float Tz = __fmaf_rn(f2, a[2][2], __fmaf_rn(f1, a[1][2], __fmul_rn(f0, a[0][2])));
            const bool home = (t0 | t1 | t2) == 0;
            for (int j = 0; j < N; ++j) {
                const float4 pj = sp ? sp[j] : mg_knn_cart(xs, lat9, j);
                const float d2 = mg_d2(__fsub_rn(pj.x, pi.x), __fsub_rn(pj.y, pi.y),
                                       __fsub_rn(pj.z, pi.z), Tx, Ty, Tz);
                bool cand = alive && d2 <= thr_d2 && !(home && j == i);
                const mg_key key = mg_knn_key(d2, (unsigned)j * (unsigned)ncell + (unsigned)c);
                cand = cand && key < thr;
                const unsigned m = __ballot_sync(0xFFFFFFFFu, cand);
                if (m) {
                    const int pos = nb + __popc(m & ((1u << lane) - 1u));
                    if (cand && pos < 32) buf[pos] = key;
                    nb += __popc(m);
                    if (nb >= 32) {                       // buffer full: sort + merge (Alg. 2)
                        __syncwarp();
                        mg_knn_merge<KPL>(keys, buf[lane], lane);
                        thr = __shfl_sync(0xFFFFFFFFu, keys[kslot], klane);
                        if (thr != MG_KEY_INF) thr_d2 = fminf(lim2, __uint_as_float((unsigned)(thr >> 32)));
                        __syncwarp();
                        if (cand && pos >= 32) buf[pos - 32] = key;
                        nb -= 32;
                    }
                }
            }
        }
        if (nb > 0) {
            __syncwarp();
            mg_knn_merge<KPL>(keys, lane < nb ? buf[lane] : MG_KEY_INF, lane);
            thr = __shfl_sync(0xFFFFFFFFu, keys[kslot], klane);
            __syncwarp();
        }
        // ---- Alg. 1 line 4: stop when the k-th distance is inside the fully explored radius
        if (thr != MG_KEY_INF) {
            const float dk = sqrtf(__uint_as_float((unsigned)(thr >> 32)));
            if (__fadd_ru(dk, 2.f * W) <= lim) break;
        }
        if (!range_ok) { failed = true; break; }
        Rad = 1.3f * fmaxf(Rad, rsafe) + 4.f * W;
    }
    if (failed && lane == 0) atomicOr(A.status, MGS_OFFSET);
    if (too_big) {                                      // natoms * box cells does not fit the key
        if (lane == 0) atomicOr(A.status, MGS_UNSUPPORTED);
#pragma unroll
        for (int s = 0; s < KPL; ++s) keys[s] = MG_KEY_INF;
    }
    // tie word -> (j, tau): cell index c = ((t0 + n0) D1 + t1 + n1) D2 + t2 + n2 of the last box
    const unsigned D1f = 2u * (unsigned)n[1] + 1u, D2f = 2u * (unsigned)n[2] + 1u;
    const unsigned ncellf = (2u * (unsigned)n[0] + 1u) * D1f * D2f;
    // ---- exact FP64 distance of the selected entries, final order by (d, dst, tau), emit
    double dmax = 0.0;
    double dd[KPL], vv[KPL][3];
    int jj[KPL], tt[KPL][3];
#pragma unroll
    for (int s = 0; s < KPL; ++s) {
        const unsigned tie = (unsigned)keys[s];
        const bool valid = 32 * s + lane < k && keys[s] != MG_KEY_INF;
        dd[s] = 1e300;
        jj[s] = 0; tt[s][0] = tt[s][1] = tt[s][2] = 0;
        if (valid) {
            const unsigned j = tie / ncellf, c = tie - j * ncellf;
            const unsigned u0 = c / (D1f * D2f), rem = c - u0 * (D1f * D2f), u1 = rem / D2f;
            jj[s] = (int)j;
            tt[s][0] = (int)u0 - n[0]; tt[s][1] = (int)u1 - n[1]; tt[s][2] = (int)(rem - u1 * D2f) - n[2];
            mg_exact_vec(xs + 3 * i, xs + 3 * jj[s], tt[s][0], tt[s][1], tt[s][2], lat9, vv[s]);
            // ranked by the FP64 SQUARED distance (the pair-lane kernel does the same: no FP64 square root)
            dd[s] = __dadd_rn(__dadd_rn(__dmul_rn(vv[s][0], vv[s][0]), __dmul_rn(vv[s][1], vv[s][1])), __dmul_rn(vv[s][2], vv[s][2]));
        }
    }
    // (two keys per lane: ranking 64 entries by counting is 1.5 k instructions a row, a fifth of the k = 64 kernel —
    // but the FP32 keys mostly ARE the final order; one look at each entry's predecessor tells, and only a row where
    // FP64 or the tie-break disagrees with the FP32 order, or one with placeholders, counts)
    bool in_order = false;
    if (KPL > 1) {
        bool ok = true;
#pragma unroll
        for (int s = 0; s < KPL; ++s) {
            const int r = 32 * s + lane;
            const unsigned tie = (unsigned)keys[s];
            double pd = __shfl_up_sync(0xFFFFFFFFu, dd[s], 1);
            unsigned pt = __shfl_up_sync(0xFFFFFFFFu, tie, 1);
            if (s > 0) {
                const double ld = __shfl_sync(0xFFFFFFFFu, dd[s > 0 ? s - 1 : 0], 31);
                const unsigned lt = __shfl_sync(0xFFFFFFFFu, (unsigned)keys[s > 0 ? s - 1 : 0], 31);
                if (lane == 0) { pd = ld; pt = lt; }
            }
            if (r < k) ok = ok && keys[s] != MG_KEY_INF && (r == 0 || pd < dd[s] || (pd == dd[s] && pt < tie));
        }
        in_order = __all_sync(0xFFFFFFFFu, ok);
    }
#pragma unroll
    for (int s = 0; s < KPL; ++s) {
        const int r = 32 * s + lane;
        const unsigned tie = (unsigned)keys[s];
        const bool valid = r < k && keys[s] != MG_KEY_INF;
        int rank = 0;
        if (KPL > 1 && in_order) rank = r;
        else {
#pragma unroll
            for (int s2 = 0; s2 < KPL; ++s2) {
                const unsigned tie2 = (unsigned)keys[s2];
                const int cnt2 = min(32, k - 32 * s2);
                for (int l = 0; l < cnt2; ++l) {
                    const double od = __shfl_sync(0xFFFFFFFFu, dd[s2], l);
                    const unsigned ot = __shfl_sync(0xFFFFFFFFu, tie2, l);
                    rank += (od < dd[s] || (od == dd[s] && ot < tie)) ? 1 : 0;
                }
            }
        }
        if (r < k) {
            const long long e = (long long)k * gi + (valid ? rank : r);
            const int j = valid ? jj[s] : i;
            A.src[e] = gi;
            A.dst[e] = R.first + j;
            A.offset[3 * e] = valid ? (int8_t)tt[s][0] : (int8_t)0;
            A.offset[3 * e + 1] = valid ? (int8_t)tt[s][1] : (int8_t)0;
            A.offset[3 * e + 2] = valid ? (int8_t)tt[s][2] : (int8_t)0;
            A.vec[3 * e] = valid ? (float)vv[s][0] : 0.f;
            A.vec[3 * e + 1] = valid ? (float)vv[s][1] : 0.f;
            A.vec[3 * e + 2] = valid ? (float)vv[s][2] : 0.f;
            // (dist = sqrt in FP32 of the FP64 squared distance, like the pair-lane kernel: a row gives the same bits
            // whichever routine produced it)
            if (A.dist) A.dist[e] = valid ? __fsqrt_rn((float)dd[s]) : 0.f;
            if (valid) dmax = fmax(dmax, dd[s]);
        }
    }
    if (A.radius_hint) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(0xFFFFFFFFu, dmax, o));
        if (lane == 0) A.radius_hint[gi] = __fsqrt_ru(__double2float_ru(dmax));
    }
}

template <int KPL>
__global__ void __launch_bounds__(MG_BLOCK)
mg_knn_small_kernel(const KnnArgs A) {
    __shared__ float4 s_p[MG_WARPS][MG_SMALL_MAX_ATOMS];
    __shared__ mg_key s_buf[MG_WARPS][32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (long long t = (long long)blockIdx.x * MG_BLOCK + tid; t <= A.n_atoms; t += (long long)gridDim.x * MG_BLOCK)
        A.row_ptr[t] = (int)((long long)A.k * t);
    if (blockIdx.x == 0 && tid == 0) *A.n_edges = (long long)A.k * A.n_atoms;
    float4 *sp = s_p[warp];
    for (;;) {
        int g = 0;
        if (lane == 0) g = (int)atomicAdd(A.ctl + 2, 1u);
        g = __shfl_sync(0xFFFFFFFFu, g, 0);
        if (g >= A.n_atoms) break;
        const int s = A.atom_struct[g];
        const StructRec R = A.rec[s];
        const float *lat9 = A.lattice + 9 * (size_t)s;
        const int i = g - R.first;
        if (R.err) {
            // invalid lattice / unsupported size: placeholder rows (src = dst, zero vec); mg_check reports
            for (int e = lane; e < A.k; e += 32) {
                const long long o = (long long)A.k * g + e;
                A.src[o] = g; A.dst[o] = g;
                A.offset[3 * o] = 0; A.offset[3 * o + 1] = 0; A.offset[3 * o + 2] = 0;
                A.vec[3 * o] = 0.f; A.vec[3 * o + 1] = 0.f; A.vec[3 * o + 2] = 0.f;
                if (A.dist) A.dist[o] = 0.f;
            }
            continue;
        }
        // (a structure above the staging limit: cartesian positions evaluated on the fly)
        const bool big = R.natoms > MG_SMALL_MAX_ATOMS;
        __syncwarp();
        for (int j = lane; j < (big ? 0 : R.natoms); j += 32) {
            const float *x = A.pos + 3 * (size_t)(R.first + j);
            const float x0 = x[0], x1 = x[1], x2 = x[2];
            float4 p;
            p.x = __fmaf_rn(x2, lat9[6], __fmaf_rn(x1, lat9[3], __fmul_rn(x0, lat9[0])));
            p.y = __fmaf_rn(x2, lat9[7], __fmaf_rn(x1, lat9[4], __fmul_rn(x0, lat9[1])));
            p.z = __fmaf_rn(x2, lat9[8], __fmaf_rn(x1, lat9[5], __fmul_rn(x0, lat9[2])));
            p.w = 0.f;
            sp[j] = p;
        }
        __syncwarp();
        mg_knn_source<KPL>(A, R, lat9, big ? nullptr : sp, s_buf[warp], i, lane);
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(A.ctl + 3, 1u) == gridDim.x - 1) { A.ctl[2] = 0u; A.ctl[3] = 0u; }
    }
}
