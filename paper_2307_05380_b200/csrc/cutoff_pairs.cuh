// cutoff_pairs.cuh — cutoff graph (K3 distance filter + K4 count -> device-wide scan -> emit + K6
// batching) in two launches of autonomous WARPS: no block barriers, no spin waits,
// no tickets.  mg_cut_prep_kernel gives every source row an estimated cost; warp w of the grid owns
// the contiguous range of rows whose cost prefix falls in [w, w+1) * total / n_warps and walks it
// structure by structure (positions and the translation table are staged once per structure).
//
//   mg_cutoff_count_kernel  find phase over the warp's rows -> edges per warp; the last CTA out
//                           turns them into an exclusive scan (the device-wide scan of K4) and
//                           writes n_edges.
//   mg_cutoff_emit_kernel   find phase again, group of rows by group of rows, now with the hits
//                           compacted into a shared-memory stash in (row, j) order; the running
//                           offset gives row_ptr; emit.
//
//  find   lane <-> ordered pair (row i, target j).  For a pair only the integers
//         tau_a in (-rho_a - u_a, rho_a - u_a), u = x_j - x_i, rho_a = r_c / h_a can be edges
//         (cut_prep.cuh), i.e. a sub-box of m_0 m_1 m_2 cells that starts at lo(pair).  The lane
//         folds its own lo into q' = (u + lo) . L and then walks the SAME table of local
//         translations T_t = t . L, t in [0,m) (broadcast float4 loads from shared memory):
//         d2 = |q' + T_t|^2 in FP32 (3 FADD, 3 FFMA), hit mask in registers.  A lane that saw a
//         candidate inside the FP32 rounding window decides its cells again with the exact FP64
//         predicate, so the edge set equals Def. 3 evaluated in FP64.  A warp
//         scan of the hit counts gives every pair its place: the group's edges are ordered by
//         (row, j), 4-byte codes (tau + 128 bytes, j).
//  emit   lanes over consecutive edges of the group: decode, vec = (p_j - p_i) + tau . L in FP64
//         rounded once, coalesced stores of src, dst, offset, vec, dist.  A group whose edges do
//         not fit the stash is searched again, writing straight to global memory.
#pragma once
#include "common.cuh"
#include "cut_prep.cuh"

struct CutoffArgs {
    const float *pos;
    const float *lattice;
    int n_struct, n_atoms;
    float r_c;
    int32_t *row_ptr, *src, *dst;
    int8_t *offset;
    float *vec, *dist;
    long long capacity;
    long long *n_edges;
    const CutRec *rec;
    const unsigned long long *bpre;   // [n_blocks + 1] cost prefix over the prep blocks, [n_blocks] = total
    int n_blocks;
    int n_warps;                   // warps of the grid (same for both launches)
    unsigned *wtotal;              // [n_warps + 1] edges per warp -> exclusive scan
    int2 *wstart;                  // [n_warps] first (structure, row) of each warp's range
    unsigned *ctl;                 // [1] count CTAs done
    unsigned *status;
    int count_only;
};

#define MG_TLOC 128                // local translation table tile (cells) = 4 mask words
#define MG_MODE_COUNT 0
#define MG_MODE_STASH 1
#define MG_MODE_DIRECT 2

struct WarpSmem {
    float4 T[MG_TLOC];             // t . L (xyz), w unused
    unsigned tcode[MG_TLOC];       // (t0 << 24 | t1 << 16 | t2 << 8)
    float4 x[MG_SMALL_MAX_ATOMS];  // wrapped fractional coordinates, .w = packed integer parts
    int rowoff[MG_TASK_ROWS + 1];
};

struct EmitSmem {
    WarpSmem w;
    double pd[MG_SMALL_MAX_ATOMS][3];   // cartesian positions x . L in FP64
    unsigned stash[MG_STASH];
};

struct Task {
    int s, first, natoms, i0, nr;      // rows i0 .. i0 + nr - 1 of structure s
};

// q / n for 0 <= q < 2^20, 1 <= n (exact: (q + 0.5) / n is never within rounding of an integer)
__device__ __forceinline__ int mg_fdiv(int q, float inv_n) {
    return __float2int_rz(__fmul_rn((float)q + 0.5f, inv_n));
}

// Write one edge: vec = (p_j - p_i) + tau . L in FP64, rounded once (R24).
// b0, b1, b2 = tau + 128.
__device__ __forceinline__ void mg_emit_edge(const CutoffArgs &A, long long e, int gi, int gj,
                                             const double *pdi, const double *pdj, const double Ld[9],
                                             unsigned b0, unsigned b1, unsigned b2) {
    // (double)(b - 128) without a conversion instruction: 2^52 + b has b in its low mantissa word
    const double t0 = __hiloint2double(0x43300000, (int)b0) - 4503599627370624.0;
    const double t1 = __hiloint2double(0x43300000, (int)b1) - 4503599627370624.0;
    const double t2 = __hiloint2double(0x43300000, (int)b2) - 4503599627370624.0;
    const double v0 = fma(t2, Ld[6], fma(t1, Ld[3], fma(t0, Ld[0], pdj[0] - pdi[0])));
    const double v1 = fma(t2, Ld[7], fma(t1, Ld[4], fma(t0, Ld[1], pdj[1] - pdi[1])));
    const double v2 = fma(t2, Ld[8], fma(t1, Ld[5], fma(t0, Ld[2], pdj[2] - pdi[2])));
    const float f0 = (float)v0, f1 = (float)v1, f2 = (float)v2;
    A.src[e] = gi;
    A.dst[e] = gj;
    A.offset[3 * e] = (int8_t)(b0 ^ 0x80u); A.offset[3 * e + 1] = (int8_t)(b1 ^ 0x80u);
    A.offset[3 * e + 2] = (int8_t)(b2 ^ 0x80u);
    A.vec[3 * e] = f0; A.vec[3 * e + 1] = f1; A.vec[3 * e + 2] = f2;
    if (A.dist) A.dist[e] = __fsqrt_rn((float)fma(v2, v2, fma(v1, v1, v0 * v0)));
}

// Stage the structure of task k: wrapped fractional coordinates xw = x - floor(x) with the integer
// part packed in .w (10 bits per axis, biased by 512); with pd != nullptr also the FP64 cartesian
// positions of the coordinates AS GIVEN.  Returns false if a coordinate is non-finite or its
// integer part does not fit (then the structure emits nothing and the status word is set).
__device__ __forceinline__ bool mg_warp_stage(WarpSmem &sw, double (*pd)[3], const CutoffArgs &A, const Task &k,
                                              int lane) {
    const float *L = A.lattice + 9 * (size_t)k.s;
    bool ok = true;
    __syncwarp();
    for (int j = lane; j < k.natoms; j += 32) {
        const float *xp = A.pos + 3 * (size_t)(k.first + j);
        const float x0 = xp[0], x1 = xp[1], x2 = xp[2];
        const float g0 = floorf(x0), g1 = floorf(x1), g2 = floorf(x2);
        ok = ok && fabsf(g0) <= 500.f && fabsf(g1) <= 500.f && fabsf(g2) <= 500.f;   // false for NaN / inf
        const int kk = ((int)g0 + 512) | (((int)g1 + 512) << 10) | (((int)g2 + 512) << 20);
        sw.x[j] = make_float4(x0 - g0, x1 - g1, x2 - g2, __int_as_float(ok ? kk : 0));
        if (pd) {
            const double d0 = (double)x0, d1 = (double)x1, d2 = (double)x2;
            pd[j][0] = fma(d2, (double)__ldg(L + 6), fma(d1, (double)__ldg(L + 3), d0 * (double)__ldg(L + 0)));
            pd[j][1] = fma(d2, (double)__ldg(L + 7), fma(d1, (double)__ldg(L + 4), d0 * (double)__ldg(L + 1)));
            pd[j][2] = fma(d2, (double)__ldg(L + 8), fma(d1, (double)__ldg(L + 5), d0 * (double)__ldg(L + 2)));
        }
    }
    ok = __all_sync(0xFFFFFFFFu, ok);
    __syncwarp();
    return ok;
}

// Local translations of cells [tile0, tile0 + MG_TLOC) of the per-pair sub-box m0 x m1 x m2:
// T = t . L in FP32, tcode = packed t; the tail is padded with a far-away sentinel.
__device__ __forceinline__ void mg_warp_table(WarpSmem &sw, const float a[9], int m1, int m2, int mloc,
                                              int tile0, int lane) {
    const int M12 = m1 * m2;
    const float inv12 = 1.f / (float)M12, inv2 = 1.f / (float)m2;
    __syncwarp();
#pragma unroll
    for (int cc = 0; cc < MG_TLOC; cc += 32) {
        const int c = cc + lane, cell = tile0 + c;
        float4 T = make_float4(1e18f, 1e18f, 1e18f, 0.f);
        unsigned code = 0u;
        if (cell < mloc) {
            const bool big = mloc >= (1 << 20);          // float reciprocal is exact below 2^20 only
            const int t0 = big ? cell / M12 : mg_fdiv(cell, inv12), r = cell - t0 * M12;
            const int t1 = big ? r / m2 : mg_fdiv(r, inv2), t2 = r - t1 * m2;
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            T.x = __fmaf_rn(f2, a[6], __fmaf_rn(f1, a[3], __fmul_rn(f0, a[0])));
            T.y = __fmaf_rn(f2, a[7], __fmaf_rn(f1, a[4], __fmul_rn(f0, a[1])));
            T.z = __fmaf_rn(f2, a[8], __fmaf_rn(f1, a[5], __fmul_rn(f0, a[2])));
            code = ((unsigned)t0 << 24) | ((unsigned)t1 << 16) | ((unsigned)t2 << 8);
        }
        if (cc == 0 || tile0 + cc < mloc) { sw.T[c] = T; sw.tcode[c] = code; }
    }
    __syncwarp();
}

// Per-task constants of the find phase.
struct FindCtx {
    float a[9];            // lattice rows (FP32)
    const float *lat;      // the same, global
    float rho[3];
    int m;                 // m_0 | m_1 << 8 | m_2 << 16
    int mloc;
    float nr2, win;        // -r_c^2, rounding window of d2
};

// One block of 32 ordered pairs against the cells [0, ncl) of the current table tile: hit masks in
// registers (W words = 32 W cells).  Lanes that saw a candidate inside the rounding window decide
// their window cells with the exact FP64 predicate.
template <int W>
__device__ __forceinline__ void mg_pair_masks(const WarpSmem &sw, const CutoffArgs &A, const FindCtx &F,
                                              float qx, float qy, float qz, int gi, int gj,
                                              int l0, int l1, int l2, int ncl, unsigned (&mask)[W]) {
    bool near = false;
    const float nr2 = F.nr2, win = F.win;
#pragma unroll
    for (int w = 0; w < W; ++w) {
        mask[w] = 0u;
        const int n4 = min(8, max(0, (ncl - 32 * w + 3) >> 2));      // warp-uniform
        const float4 *Tp = sw.T + 32 * w;
        for (int g = 0; g < n4; ++g) {
            unsigned sub = 0u;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const float4 T = Tp[4 * g + c];
                const float vx = __fadd_rn(qx, T.x), vy = __fadd_rn(qy, T.y), vz = __fadd_rn(qz, T.z);
                const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, nr2)));
                if (y < win) sub |= 1u << c;
                near = near || fabsf(y) < win;
            }
            mask[w] |= sub << (4 * g);
        }
    }
    if (near) {                                   // rare: decide the window cells in FP64
        const float *xi = A.pos + 3 * (size_t)gi, *xj = A.pos + 3 * (size_t)gj;
        for (int c = 0; c < ncl; ++c) {
            const float4 T = sw.T[c];
            const float vx = __fadd_rn(qx, T.x), vy = __fadd_rn(qy, T.y), vz = __fadd_rn(qz, T.z);
            const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, nr2)));
            if (fabsf(y) < win) {
                const unsigned tc = sw.tcode[c];
                double v[3];
                const double d = mg_exact_vec(xi, xj, l0 + (int)(tc >> 24), l1 + (int)((tc >> 16) & 0xFFu),
                                              l2 + (int)((tc >> 8) & 0xFFu), F.lat, v);
                const unsigned bit = 1u << (c & 31);
#pragma unroll
                for (int w = 0; w < W; ++w)
                    if (w == (c >> 5)) mask[w] = d < (double)A.r_c ? (mask[w] | bit) : (mask[w] & ~bit);
            }
        }
    }
}

// Find phase over rows k.i0 .. k.i0 + k.nr - 1 of structure k.s (staged in sw).  Returns the number
// of edges.
//   MG_MODE_COUNT   nothing else
//   MG_MODE_STASH   edge codes -> stash (positions >= MG_STASH are dropped: the caller checks),
//                   row offsets inside the group -> sw.rowoff[0 .. nr], row_ptr = goff + offset
//   MG_MODE_DIRECT  edges straight to global memory at goff + position, row_ptr
// The tile loop is outside the pair loop only when the table does not fit (mloc > 32 W; then the
// caller passes one row at a time in the STASH / DIRECT modes, so the (row, j) order holds).
template <int W, int MODE>
__device__ __forceinline__ unsigned mg_warp_find(WarpSmem &sw, unsigned *stash, const double (*pd)[3],
                                                 const CutoffArgs &A, const Task &k, const FindCtx &F,
                                                 long long goff, int lane) {
    const int N = k.natoms, NP = k.nr * N;
    const float inv_N = 1.f / (float)N;
    const int m0 = F.m & 0xFF, m1 = (F.m >> 8) & 0xFF, m2 = (F.m >> 16) & 0xFF;
    double Ld[9];
    if (MODE == MG_MODE_DIRECT) {
#pragma unroll
        for (int c = 0; c < 9; ++c) Ld[c] = (double)F.a[c];
    }
    int run = 0;
    for (int tile0 = 0; tile0 < F.mloc; tile0 += 32 * W) {
        const int ncl = min(32 * W, F.mloc - tile0);
        if (F.mloc > 32 * W) mg_warp_table(sw, F.a, m1, m2, F.mloc, tile0, lane);
        for (int q0 = 0; q0 < NP; q0 += 32) {
            const int q = q0 + lane;
            const bool valid = q < NP;
            const int ri = valid ? mg_fdiv(q, inv_N) : 0;
            const int j = valid ? q - ri * N : 0;
            const int i = k.i0 + ri;
            const float4 xi = sw.x[i], xj = sw.x[j];
            // u = x_j - x_i (wrapped coordinates), first cell of the pair's sub-box: floor(-rho - u) + 1
            const float u0 = __fsub_rn(xj.x, xi.x), u1 = __fsub_rn(xj.y, xi.y), u2 = __fsub_rn(xj.z, xi.z);
            const float e0 = floorf(__fsub_rn(-F.rho[0], u0)) + 1.f, e1 = floorf(__fsub_rn(-F.rho[1], u1)) + 1.f,
                        e2 = floorf(__fsub_rn(-F.rho[2], u2)) + 1.f;
            const float f0 = __fadd_rn(u0, e0), f1 = __fadd_rn(u1, e1), f2 = __fadd_rn(u2, e2);
            float qx = __fmaf_rn(f2, F.a[6], __fmaf_rn(f1, F.a[3], __fmul_rn(f0, F.a[0])));
            float qy = __fmaf_rn(f2, F.a[7], __fmaf_rn(f1, F.a[4], __fmul_rn(f0, F.a[1])));
            float qz = __fmaf_rn(f2, F.a[8], __fmaf_rn(f1, F.a[5], __fmul_rn(f0, F.a[2])));
            // cell offsets relative to the coordinates AS GIVEN: tau = tau_wrapped + k_i - k_j
            const int ki = __float_as_int(xi.w), kj = __float_as_int(xj.w);
            const int l0 = (int)e0 + (ki & 1023) - (kj & 1023);
            const int l1 = (int)e1 + ((ki >> 10) & 1023) - ((kj >> 10) & 1023);
            const int l2 = (int)e2 + ((ki >> 20) & 1023) - ((kj >> 20) & 1023);
            const bool inrange = l0 >= -127 && l1 >= -127 && l2 >= -127 && l0 + m0 <= 128 &&
                                 l1 + m1 <= 128 && l2 + m2 <= 128;
            if (MODE == MG_MODE_COUNT && valid && !inrange) atomicOr(A.status, MGS_OFFSET);
            if (!valid || !inrange) { qx = 1e18f; qy = 1e18f; qz = 1e18f; }
            unsigned mask[W];
            mg_pair_masks<W>(sw, A, F, qx, qy, qz, k.first + i, k.first + j, l0, l1, l2, ncl, mask);
            if (i == j) {                           // (i,i,0) is not an edge (R3)
                const int cs = (-(int)e0 * m1 - (int)e1) * m2 - (int)e2 - tile0;
#pragma unroll
                for (int w = 0; w < W; ++w)
                    if (cs >= 32 * w && cs < 32 * w + 32) mask[w] &= ~(1u << (cs & 31));
            }
            int cnt = 0;
#pragma unroll
            for (int w = 0; w < W; ++w) cnt += __popc(mask[w]);
            if (MODE == MG_MODE_COUNT) {
                run += cnt;                         // per lane; reduced once at the end
            } else {
                int incl = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                    if (lane >= o) incl += v;
                }
                const int tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
                int pos = run + incl - cnt;
                if (valid && j == 0 && tile0 == 0) {
                    sw.rowoff[ri] = pos;
                    A.row_ptr[k.first + i] = (int)(goff + pos);
                }
                const unsigned paircode = ((unsigned)(l0 + 128) << 24) | ((unsigned)(l1 + 128) << 16) |
                                          ((unsigned)(l2 + 128) << 8) | (unsigned)j;
#pragma unroll
                for (int w = 0; w < W; ++w) {
                    unsigned mk = mask[w];
                    while (mk) {
                        const int b = __ffs(mk) - 1;
                        mk &= mk - 1;
                        const unsigned code = paircode + sw.tcode[32 * w + b];
                        if (MODE == MG_MODE_STASH) {
                            if (pos < MG_STASH) stash[pos] = code;
                        } else if (goff + pos < A.capacity) {
                            mg_emit_edge(A, goff + pos, k.first + i, k.first + j, pd[i], pd[j], Ld, code >> 24,
                                         (code >> 16) & 0xFFu, (code >> 8) & 0xFFu);
                        }
                        ++pos;
                    }
                }
                run += tot;
            }
        }
    }
    if (MODE == MG_MODE_COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) run += __shfl_xor_sync(0xFFFFFFFFu, run, o);
    } else {
        __syncwarp();
        if (lane == 0) sw.rowoff[k.nr] = run;
        __syncwarp();
    }
    return (unsigned)run;
}

// Constants of the find phase for structure s; stages the structure (positions, table when it
// fits).  Returns false if the structure emits nothing (empty, invalid lattice or positions).
__device__ __forceinline__ bool mg_struct_setup(WarpSmem &sw, double (*pd)[3], const CutoffArgs &A, const CutRec *R,
                                                int s, Task &k, FindCtx &F, int lane) {
    k.s = s;
    k.first = R->first;
    k.natoms = R->natoms;
    F.lat = A.lattice + 9 * (size_t)s;
    F.mloc = R->mloc;
    if (F.mloc <= 0) return false;
#pragma unroll
    for (int c = 0; c < 9; ++c) F.a[c] = __ldg(F.lat + c);
#pragma unroll
    for (int a = 0; a < 3; ++a) F.rho[a] = R->rho[a];
    F.m = R->m;
    F.nr2 = -__fmul_rn(A.r_c, A.r_c);
    // FP32 error bound of d2 - r_c^2 near the threshold (R23): the components of q', T
    // and q' + T are below 3 Q, about 13 roundings of 2^-24 relative size reach v (the wrapped
    // coordinates are below 1, their difference is rounded once), d2 = v . v adds 3 more
    F.win = 1.1920929e-7f * (2.f * A.r_c * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * A.r_c * A.r_c);
    if (!mg_warp_stage(sw, pd, A, k, lane)) {
        if (lane == 0) atomicOr(A.status, MGS_NONFINITE);
        F.mloc = 0;
        return false;
    }
    if (F.mloc <= MG_TLOC) mg_warp_table(sw, F.a, (F.m >> 8) & 0xFF, (F.m >> 16) & 0xFF, F.mloc, 0, lane);
    return true;
}

template <int MODE>
__device__ __forceinline__ unsigned mg_find_dispatch(WarpSmem &sw, unsigned *stash, const double (*pd)[3],
                                                     const CutoffArgs &A, const Task &k, const FindCtx &F,
                                                     long long goff, int lane) {
    if (F.mloc <= 32) return mg_warp_find<1, MODE>(sw, stash, pd, A, k, F, goff, lane);
    if (F.mloc <= 64) return mg_warp_find<2, MODE>(sw, stash, pd, A, k, F, goff, lane);
    return mg_warp_find<4, MODE>(sw, stash, pd, A, k, F, goff, lane);
}

// First (structure, row) of warp w's range: the first row whose cost prefix is >= c0 = w * chunk.
// The cost prefix of row r of structure s is bpre[s / MG_CP_BLOCK] + rec[s].lpre + r * rowcost.
__device__ inline void mg_range_start(const CutoffArgs &A, unsigned long long c0, int &s_out, int &r_out, int lane) {
    // level 1: last prep block b with bpre[b] <= c0 (32-ary search)
    int lo = 0, hi = A.n_blocks;                   // answer in [lo, hi)
    while (hi - lo > 1) {
        const int step = (hi - lo + 31) / 32;
        const int idx = lo + (lane + 1) * step;
        const bool ok = idx < hi && __ldg(A.bpre + idx) <= c0;
        lo += __popc(__ballot_sync(0xFFFFFFFFu, ok)) * step;
        hi = min(hi, lo + step);
    }
    const int b = lo;
    const unsigned long long bp = __ldg(A.bpre + b);
    // level 2: last structure of the block whose prefix is <= c0
    int cnt = 0;
#pragma unroll
    for (int q = 0; q < MG_CP_BLOCK / 32; ++q) {
        const int s = b * MG_CP_BLOCK + q * 32 + lane;
        const bool ok = s < A.n_struct && bp + A.rec[s].lpre <= c0;
        cnt += __popc(__ballot_sync(0xFFFFFFFFu, ok));
    }
    int s = b * MG_CP_BLOCK + max(cnt, 1) - 1;
    const CutRec *R = A.rec + s;
    const unsigned long long cs = bp + R->lpre;
    const unsigned rc = R->rowcost;
    int r = c0 > cs ? (int)((c0 - cs + rc - 1) / rc) : 0;
    if (r >= R->natoms) { s += 1; r = 0; }         // every later row starts at or after c0
    s_out = s;
    r_out = r;
}

// Cost range of warp w: [c0, c1); the last warp takes everything that is left.
__device__ __forceinline__ void mg_warp_range(const CutoffArgs &A, int w, unsigned long long &c0,
                                              unsigned long long &c1) {
    const unsigned long long total = __ldg(A.bpre + A.n_blocks);
    const unsigned long long chunk = (total + (unsigned)A.n_warps - 1) / (unsigned)A.n_warps;
    c0 = (unsigned long long)w * chunk;
    c1 = w == A.n_warps - 1 ? ~0ull : c0 + chunk;
}

// ---------------------------------------------------------------------------------------------
// Launch 1: count.
__global__ void __launch_bounds__(MG_BLOCK, 4)
mg_cutoff_count_kernel(const __grid_constant__ CutoffArgs A) {
    __shared__ WarpSmem s_w[MG_WARPS];
    __shared__ unsigned long long s_part[MG_BLOCK];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem &sw = s_w[warp];
    const int w = blockIdx.x * MG_WARPS + warp;
    unsigned long long c0, c1;
    mg_warp_range(A, w, c0, c1);
    int s, r;
    mg_range_start(A, c0, s, r, lane);
    if (lane == 0) A.wstart[w] = make_int2(s, r);
    unsigned total = 0u;
    for (; s < A.n_struct; ++s, r = 0) {
        const CutRec *R = A.rec + s;
        const unsigned long long cs = __ldg(A.bpre + s / MG_CP_BLOCK) + R->lpre;
        if (cs + (unsigned long long)r * R->rowcost >= c1 && R->natoms > 0) break;
        if (R->natoms == 0) continue;
        // rows r .. rb - 1 start before c1
        const unsigned long long room = (c1 - cs + R->rowcost - 1) / R->rowcost;
        const int rb = (int)min((unsigned long long)R->natoms, room);
        Task k;
        FindCtx F;
        if (mg_struct_setup(sw, nullptr, A, R, s, k, F, lane)) {
            k.i0 = r;
            k.nr = rb - r;
            total += mg_find_dispatch<MG_MODE_COUNT>(sw, nullptr, nullptr, A, k, F, 0, lane);
        }
        if (rb < R->natoms) break;
    }
    if (lane == 0) A.wtotal[w] = total;
    // ---- last CTA out: exclusive scan of the warp totals, grand total
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(A.ctl + 1, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int nw = A.n_warps, per = (nw + MG_BLOCK - 1) / MG_BLOCK;
    const int b = threadIdx.x * per, e = min(nw, b + per);
    unsigned long long sum = 0ull;
    for (int g = b; g < e; ++g) sum += __ldcg(A.wtotal + g);
    s_part[threadIdx.x] = sum;
    __syncthreads();
    unsigned long long off = 0ull;
    for (int x = 0; x < (int)threadIdx.x; ++x) off += s_part[x];
    for (int g = b; g < e; ++g) {
        const unsigned v = __ldcg(A.wtotal + g);
        A.wtotal[g] = (unsigned)off;
        off += v;
    }
    if (threadIdx.x == MG_BLOCK - 1) {
        *A.n_edges = (long long)off;
        A.row_ptr[A.n_atoms] = (int)off;
        if (off > 0x7FFFFFFFull || (!A.count_only && (long long)off > A.capacity)) atomicOr(A.status, MGS_CAPACITY);
        A.ctl[1] = 0u;
    }
}

// ---------------------------------------------------------------------------------------------
// Launch 2: emit.
__global__ void __launch_bounds__(MG_BLOCK, 4)
mg_cutoff_emit_kernel(const __grid_constant__ CutoffArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    EmitSmem &se = reinterpret_cast<EmitSmem *>(smem_raw)[warp];
    WarpSmem &sw = se.w;
    const int w = blockIdx.x * MG_WARPS + warp;
    unsigned long long c0, c1;
    mg_warp_range(A, w, c0, c1);
    const int2 st = A.wstart[w];
    int s = st.x, r = st.y;
    long long goff = (long long)__ldg(A.wtotal + w);
    for (; s < A.n_struct; ++s, r = 0) {
        const CutRec *R = A.rec + s;
        const unsigned long long cs = __ldg(A.bpre + s / MG_CP_BLOCK) + R->lpre;
        if (cs + (unsigned long long)r * R->rowcost >= c1 && R->natoms > 0) break;
        if (R->natoms == 0) continue;
        const unsigned long long room = (c1 - cs + R->rowcost - 1) / R->rowcost;
        const int rb = (int)min((unsigned long long)R->natoms, room);
        Task k;
        FindCtx F;
        if (!mg_struct_setup(sw, se.pd, A, R, s, k, F, lane)) {
            for (int i = r + lane; i < rb; i += 32) A.row_ptr[R->first + i] = (int)goff;   // no edges
        } else {
            double Ld[9];
#pragma unroll
            for (int c = 0; c < 9; ++c) Ld[c] = (double)F.a[c];
            const int rpt = R->rpt;
            for (int i0 = r; i0 < rb; i0 += rpt) {
                k.i0 = i0;
                k.nr = min(rpt, rb - i0);
                const unsigned total = mg_find_dispatch<MG_MODE_STASH>(sw, se.stash, se.pd, A, k, F, goff, lane);
                if (total > MG_STASH) {            // does not fit: search again, write directly
                    mg_find_dispatch<MG_MODE_DIRECT>(sw, nullptr, se.pd, A, k, F, goff, lane);
                } else {
                    int rr = 0;
                    for (int e0 = 0; e0 < (int)total; e0 += 32) {
                        const int e = e0 + lane;
                        if (e < (int)total) {
                            while (e >= sw.rowoff[rr + 1]) ++rr;
                            const unsigned code = se.stash[e];
                            const int j = (int)(code & 0xFFu);
                            if (goff + e < A.capacity)
                                mg_emit_edge(A, goff + e, k.first + i0 + rr, k.first + j, se.pd[i0 + rr], se.pd[j], Ld,
                                             code >> 24, (code >> 16) & 0xFFu, (code >> 8) & 0xFFu);
                        }
                    }
                }
                goff += total;
                __syncwarp();
            }
        }
        if (rb < R->natoms) break;
    }
}
