// knn_small.cuh — k-nearest-neighbour multigraph for structures of <= MG_SMALL_MAX_ATOMS atoms.
//
// Problem: per source the k smallest keys (d, dst, tau_x, tau_y, tau_z) over all periodic images
// except (i,i,0) (Alg. 2 lines 2-5, made deterministic: DESIGN.md R2, R8).
// Method (Alg. 1, re-designed): one warp per source atom keeps the ordered stack
// of Alg. 2 in REGISTERS — a sorted list of 64-bit keys, one or two per lane — and explores an
// expanding box of cells: lanes <-> cells, loop over target atoms j.  After a box of half widths
// n_a every unexplored image is farther than R_safe = min_a (n_a + 1 - spread_a) h_a
// (closest_distance of Alg. 1 line 4; proof in DESIGN.md R11), so the search stops as soon as the
// k-th distance is <= R_safe; otherwise the box grows to the current k-th distance ("the search
// radius decreases over time"), which is then guaranteed to finish.
// The FP32 keys select the k entries; their final order and the emitted vec / dist use the exact
// FP64 distance.
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
    unsigned *ticket;           // [0] next chunk, [1] CTAs done
    unsigned *status;
};

struct KnnSmem {
    float4 p[MG_SMALL_MAX_ATOMS];
    float x[MG_SMALL_MAX_ATOMS * 3];
    float lat[9];
    double h[3];
    double vol;
    float xmin[3], xmax[3];
    int chunk, first, natoms;
    unsigned err;
};

// Insert `key` into the warp-resident sorted list (slot s of lane l holds rank 32 s + l).
template <int KPL>
__device__ __forceinline__ void mg_knn_insert(unsigned long long (&keys)[KPL], unsigned long long key,
                                              int lane) {
#pragma unroll
    for (int s = 0; s < KPL; ++s) {
        const unsigned less = __ballot_sync(0xFFFFFFFFu, keys[s] < key);
        const int pos = __popc(less);                    // sorted: the smaller keys are a lane prefix
        const unsigned long long up = __shfl_up_sync(0xFFFFFFFFu, keys[s], 1);
        const unsigned long long last = __shfl_sync(0xFFFFFFFFu, keys[s], 31);
        if (pos < 32) {
            if (lane == pos) keys[s] = key;
            else if (lane > pos) keys[s] = up;
            key = last;                                  // evicted rank 31 goes to the next slot
        }
    }
}

__device__ __forceinline__ unsigned long long mg_knn_key(float d2, int j, int t0, int t1, int t2) {
    return ((unsigned long long)__float_as_uint(d2) << 32) | ((unsigned long long)(unsigned)j << 24) |
           ((unsigned long long)(unsigned)(t0 + 128) << 16) | ((unsigned)(t1 + 128) << 8) |
           (unsigned)(t2 + 128);
}

// Search + emit for one source atom i of the staged structure; called by a full warp.
template <int KPL>
__device__ inline void mg_knn_source(const KnnSmem &sm, const KnnArgs &A, int i, int lane) {
    const int N = sm.natoms, k = A.k;
    const int kslot = (k - 1) >> 5, klane = (k - 1) & 31;
    unsigned long long keys[KPL];
#pragma unroll
    for (int s = 0; s < KPL; ++s) keys[s] = MG_KEY_INF;
    unsigned long long thr = MG_KEY_INF;
    float thr_d2 = __int_as_float(0x7f800000);
    const float4 pi = sm.p[i];
    float a[3][3], hf[3], lo_off[3], hi_off[3];
    double spread[3], amax[3];
    float xabs = 1.f;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
#pragma unroll
        for (int c = 0; c < 3; ++c) a[r][c] = sm.lat[3 * r + c];
        hf[r] = __double2float_rd(sm.h[r] * (1.0 - 1e-6));
        const float xi = sm.x[3 * i + r];
        lo_off[r] = sm.xmin[r] - xi;                 // exact or rounded: only used for pruning,
        hi_off[r] = sm.xmax[r] - xi;                 // with hf rounded down and a safety factor
        spread[r] = (double)sm.xmax[r] - (double)sm.xmin[r];
        amax[r] = fmax(fabs((double)a[r][0]), fmax(fabs((double)a[r][1]), fabs((double)a[r][2])));
        xabs = fmaxf(xabs, fmaxf(fabsf(sm.xmin[r]), fabsf(sm.xmax[r])));
    }
    const int gi = sm.first + i;
    double R;
    if (A.use_hint && A.radius_hint[gi] > 0.f) R = 1.05 * (double)A.radius_hint[gi] + 1e-3;
    else R = 1.1 * cbrt(0.2387324146 * (double)(k + 1) * sm.vol / (double)N);
    int nprev[3] = {-1, -1, -1};
    bool failed = false;
    for (;;) {
        int n[3];
        double rsafe = 1e300, M = 0.0;
        bool range_ok = true;
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            double nn = floor(R / sm.h[r] * (1.0 + 1e-6) + spread[r]);
            if (nn < (double)nprev[r]) nn = (double)nprev[r];
            if (!(nn <= 127.0)) { range_ok = false; nn = 127.0; }
            n[r] = (int)nn;
            rsafe = fmin(rsafe, (nn + 1.0 - spread[r]) * sm.h[r]);
            M += (nn + 2.0 * (double)xabs) * amax[r];
        }
        const double W = 3.5 * 12.0 * 5.9604644775390625e-8 * M;
        const int D1 = 2 * n[1] + 1, D2 = 2 * n[2] + 1;
        const int ncell = (2 * n[0] + 1) * D1 * D2;
        for (int c0 = 0; c0 < ncell; c0 += 32) {
            const int c = c0 + lane;
            const int u0 = c / (D1 * D2), rem = c - u0 * (D1 * D2), u1 = rem / D2;
            const int t0 = u0 - n[0], t1 = u1 - n[1], t2 = rem - u1 * D2 - n[2];
            bool alive = c < ncell && !(abs(t0) <= nprev[0] && abs(t1) <= nprev[1] && abs(t2) <= nprev[2]);
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            // lower bound of the distance to any image in this cell: max_a gap_a h_a
            const float g0 = fmaxf(0.f, fmaxf(f0 + lo_off[0], -(f0 + hi_off[0]))) * hf[0];
            const float g1 = fmaxf(0.f, fmaxf(f1 + lo_off[1], -(f1 + hi_off[1]))) * hf[1];
            const float g2 = fmaxf(0.f, fmaxf(f2 + lo_off[2], -(f2 + hi_off[2]))) * hf[2];
            const float lb = fmaxf(g0, fmaxf(g1, g2)) * 0.99999f;
            alive = alive && lb * lb <= thr_d2;
            if (!__any_sync(0xFFFFFFFFu, alive)) continue;
            const float Tx = __fmaf_rn(f2, a[2][0], __fmaf_rn(f1, a[1][0], __fmul_rn(f0, a[0][0])));
            const float Ty = __fmaf_rn(f2, a[2][1], __fmaf_rn(f1, a[1][1], __fmul_rn(f0, a[0][1])));
            const float Tz = __fmaf_rn(f2, a[2][2], __fmaf_rn(f1, a[1][2], __fmul_rn(f0, a[0][2])));
            const bool home = (t0 | t1 | t2) == 0;
            for (int j = 0; j < N; ++j) {
                const float4 pj = sm.p[j];
                const float d2 = mg_d2(__fsub_rn(pj.x, pi.x), __fsub_rn(pj.y, pi.y),
                                       __fsub_rn(pj.z, pi.z), Tx, Ty, Tz);
                bool cand = alive && d2 <= thr_d2 && !(home && j == i);
                const unsigned long long key = cand ? mg_knn_key(d2, j, t0, t1, t2) : MG_KEY_INF;
                cand = key < thr;
                unsigned m = __ballot_sync(0xFFFFFFFFu, cand);
                if (m) {
                    while (m) {
                        const int srcl = __ffs(m) - 1;
                        m &= m - 1;
                        const unsigned long long kk = __shfl_sync(0xFFFFFFFFu, key, srcl);
                        if (kk < thr) {
                            mg_knn_insert<KPL>(keys, kk, lane);
                            thr = __shfl_sync(0xFFFFFFFFu, keys[kslot], klane);
                        }
                    }
                    if (thr != MG_KEY_INF) thr_d2 = __uint_as_float((unsigned)(thr >> 32));
                }
            }
        }
        nprev[0] = n[0]; nprev[1] = n[1]; nprev[2] = n[2];
        if (thr != MG_KEY_INF) {
            const double dk = sqrt((double)thr_d2) + W;
            if (dk <= rsafe) break;
            if (!range_ok) { failed = true; break; }
            R = dk * (1.0 + 1e-6);
        } else {
            if (!range_ok) { failed = true; break; }
            R = fmax(1.5 * R, 1.01 * rsafe);
        }
    }
    if (failed && lane == 0) atomicOr(A.status, MGS_OFFSET);
    // ---- exact FP64 distance of the selected entries, final order by (d, dst, tau), emit
    double dmax = 0.0;
#pragma unroll
    for (int s = 0; s < KPL; ++s) {
        const int r = 32 * s + lane;
        const bool valid = r < k && keys[s] != MG_KEY_INF;
        const unsigned tie = (unsigned)keys[s];
        const int j = valid ? (int)((tie >> 24) & 0xFFu) : i;
        const int t0 = valid ? (int)((tie >> 16) & 0xFFu) - 128 : 0;
        const int t1 = valid ? (int)((tie >> 8) & 0xFFu) - 128 : 0;
        const int t2 = valid ? (int)(tie & 0xFFu) - 128 : 0;
        double v[3];
        double d = mg_exact_vec(sm.x + 3 * i, sm.x + 3 * j, t0, t1, t2, sm.lat, v);
        if (!valid) d = 1e300;
        int rank = 0;
#pragma unroll
        for (int s2 = 0; s2 < KPL; ++s2) {
            // my own slot-s2 values, to be broadcast
            const unsigned tie2 = (unsigned)keys[s2];
            const bool valid2 = 32 * s2 + lane < k && keys[s2] != MG_KEY_INF;
            double d2v = 1e300;
            if (s2 == s) d2v = d;
            else if (valid2) {
                double vv[3];
                d2v = mg_exact_vec(sm.x + 3 * i, sm.x + 3 * (int)((tie2 >> 24) & 0xFFu),
                                   (int)((tie2 >> 16) & 0xFFu) - 128, (int)((tie2 >> 8) & 0xFFu) - 128,
                                   (int)(tie2 & 0xFFu) - 128, sm.lat, vv);
            }
            const int cnt2 = min(32, k - 32 * s2);
            for (int l = 0; l < cnt2; ++l) {
                const double od = __shfl_sync(0xFFFFFFFFu, d2v, l);
                const unsigned ot = __shfl_sync(0xFFFFFFFFu, tie2, l);
                rank += (od < d || (od == d && ot < tie)) ? 1 : 0;
            }
        }
        if (r < k) {
            const long long e = (long long)k * gi + (valid ? rank : r);
            A.src[e] = gi;
            A.dst[e] = sm.first + j;
            A.offset[3 * e] = (int8_t)t0; A.offset[3 * e + 1] = (int8_t)t1; A.offset[3 * e + 2] = (int8_t)t2;
            A.vec[3 * e] = valid ? (float)v[0] : 0.f;
            A.vec[3 * e + 1] = valid ? (float)v[1] : 0.f;
            A.vec[3 * e + 2] = valid ? (float)v[2] : 0.f;
            if (A.dist) A.dist[e] = valid ? (float)d : 0.f;
            if (valid) dmax = fmax(dmax, d);
        }
    }
    if (A.radius_hint) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) dmax = fmax(dmax, __shfl_xor_sync(0xFFFFFFFFu, dmax, o));
        if (lane == 0) A.radius_hint[gi] = __double2float_ru(dmax);
    }
}

template <int KPL>
__global__ void __launch_bounds__(MG_BLOCK)
mg_knn_small_kernel(const KnnArgs A) {
    __shared__ KnnSmem sm;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (long long t = (long long)blockIdx.x * MG_BLOCK + tid; t <= A.n_atoms; t += (long long)gridDim.x * MG_BLOCK)
        A.row_ptr[t] = (int)((long long)A.k * t);
    if (blockIdx.x == 0 && tid == 0) *A.n_edges = (long long)A.k * A.n_atoms;
    for (;;) {
        __syncthreads();
        if (tid == 0) sm.chunk = (int)atomicAdd(A.ticket, 1u);
        __syncthreads();
        const int s = sm.chunk;
        if (s >= A.n_struct) break;
        if (tid == 0) {
            sm.first = A.struct_ptr[s];
            sm.natoms = A.struct_ptr[s + 1] - sm.first;
        }
        if (tid >= 32 && tid < 41) sm.lat[tid - 32] = A.lattice[9 * (size_t)s + (tid - 32)];
        __syncthreads();
        int N = sm.natoms;
        if (N > MG_SMALL_MAX_ATOMS) {
            if (tid == 0) atomicOr(A.status, MGS_UNSUPPORTED);
            continue;
        }
        if (tid < 3 * N) sm.x[tid] = A.pos[3 * (size_t)sm.first + tid];
        __syncthreads();
        if (tid == 0) {
            double vol;
            sm.err = mg_cell_spacings(sm.lat, &vol, sm.h);
            sm.vol = vol;
            bool finite = true;
            for (int a = 0; a < 3; ++a) {
                float lo = 0.f, hi = 0.f;
                for (int i = 0; i < N; ++i) {
                    const float v = sm.x[3 * i + a];
                    finite = finite && isfinite(v);
                    lo = i ? fminf(lo, v) : v;
                    hi = i ? fmaxf(hi, v) : v;
                }
                sm.xmin[a] = lo; sm.xmax[a] = hi;
            }
            if (!finite) sm.err |= MGS_NONFINITE;
            if (sm.err) atomicOr(A.status, sm.err);
        }
        __syncthreads();
        if (tid < N) {
            const float x0 = sm.x[3 * tid], x1 = sm.x[3 * tid + 1], x2 = sm.x[3 * tid + 2];
            float4 p;
            p.x = __fmaf_rn(x2, sm.lat[6], __fmaf_rn(x1, sm.lat[3], __fmul_rn(x0, sm.lat[0])));
            p.y = __fmaf_rn(x2, sm.lat[7], __fmaf_rn(x1, sm.lat[4], __fmul_rn(x0, sm.lat[1])));
            p.z = __fmaf_rn(x2, sm.lat[8], __fmaf_rn(x1, sm.lat[5], __fmul_rn(x0, sm.lat[2])));
            p.w = 0.f;
            sm.p[tid] = p;
        }
        __syncthreads();
        if (sm.err) {
            // invalid lattice: rows are filled with placeholders (src = dst, zero vec); see mg_check
            for (int e = tid; e < N * A.k; e += MG_BLOCK) {
                const long long o = (long long)A.k * sm.first + e;
                A.src[o] = sm.first + e / A.k; A.dst[o] = sm.first + e / A.k;
                A.offset[3 * o] = 0; A.offset[3 * o + 1] = 0; A.offset[3 * o + 2] = 0;
                A.vec[3 * o] = 0.f; A.vec[3 * o + 1] = 0.f; A.vec[3 * o + 2] = 0.f;
                if (A.dist) A.dist[o] = 0.f;
            }
            continue;
        }
        for (int i = warp; i < N; i += MG_WARPS) mg_knn_source<KPL>(sm, A, i, lane);
    }
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(A.ticket + 1, 1u) == gridDim.x - 1) { A.ticket[0] = 0u; A.ticket[1] = 0u; }
    }
}
