// cutoff_pairs.cuh — cutoff graph (K3 distance filter + K4 count -> device-wide scan -> emit + K6
// batching) in two launches of autonomous WARPS: no block barriers, no spin waits.
// mg_cut_prep_kernel gives every ordered pair (i, j) an estimated cost; warp w of the grid owns the
// contiguous range of pairs, in (structure, i, j) order, whose cost prefix falls in
// [w, w+1) * total / n_warps and walks it structure by structure (positions and the translation
// table are staged once per structure; a range may split a source row or a large structure).
//
//   mg_cutoff_count_kernel  find phase over the warp's pairs -> hit masks (kept in a per-warp
//                           scratch) and edges per warp; the last CTA out turns the totals into an
//                           exclusive scan (the device-wide scan of K4) and writes n_edges.
//   mg_cutoff_emit_kernel   same ranges: masks read back, hits compacted into a shared-memory stash
//                           in (row, j) order; the running offset gives row_ptr; emit.
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
#include "ranges.cuh"

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
    int n_warps;                   // warps of the grid
    int n_ranges;                  // MG_OVER * n_warps ranges (MG_OVER = 1: one per warp; more were slower)
    unsigned *wtotal;              // [n_ranges + 1] edges per range -> exclusive scan
    unsigned *gtotal;              // [64] edges per group of ceil(n_ranges / 64) ranges (zero between calls)
    int2 *wstart;                  // [n_ranges] first (structure, pair) of each range
    unsigned *wmask;               // [n_ranges, MG_MASK_WORDS] hit masks kept from count to emit
    int mask_words;                // words of a range's scratch that may be used (MG_MASK_WORDS; tests: less)
    unsigned *wclock;              // [2, n_warps] cycles each warp spent in count / emit (tuning aid)
    unsigned *ctl;                 // [1] count CTAs done (mg_cutoff_count), [9] emit CTAs done
    unsigned *status;
    int count_only;
};

#define MG_TLOC 256                // local translation table tile (cells) = 8 mask words
#define MG_MODE_COUNT 0
#define MG_MODE_STASH 1
#define MG_MODE_DIRECT 2

#define MG_OVER 1                  // ranges per warp (more, handed out by ticket, measured slower: DESIGN.md)
#define MG_MASK_WORDS 4096         // per-warp mask scratch (32-bit words, multiple of 128)

struct WarpSmem {
    float4 T[MG_TLOC];             // t . L: planes x | y | z of MG_TLOC floats (mg_tplane); the rest is unused
    unsigned tcode[MG_TLOC];       // (t0 << 24 | t1 << 16 | t2 << 8)
    float4 x[MG_SMALL_MAX_ATOMS];  // wrapped fractional coordinates, .w = packed integer parts
};

struct EmitSmem {
    WarpSmem w;
    double pd[MG_SMALL_MAX_ATOMS][3];   // cartesian positions x . L in FP64
    unsigned stash[MG_STASH];
};

struct Task {
    int s, first, natoms;
};

// FP64 cartesian position x . L of atom idx (from the staged copy, or evaluated on the fly).
__device__ __forceinline__ void mg_pd_big(const float *gx, const double Ld[9], int idx, double out[3]) {
    const double d0 = (double)gx[3 * idx], d1 = (double)gx[3 * idx + 1], d2 = (double)gx[3 * idx + 2];
    out[0] = fma(d2, Ld[6], fma(d1, Ld[3], d0 * Ld[0]));
    out[1] = fma(d2, Ld[7], fma(d1, Ld[4], d0 * Ld[1]));
    out[2] = fma(d2, Ld[8], fma(d1, Ld[5], d0 * Ld[2]));
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
__device__ __forceinline__ bool mg_warp_stage(WarpSmem &sw, double (*pd)[3], const float *pos, const float *lattice,
                                              const Task &k, int lane) {
    const float *L = lattice + 9 * (size_t)k.s;
    bool ok = true;
    __syncwarp();
    for (int j = lane; j < k.natoms; j += 32) {
        const float *xp = pos + 3 * (size_t)(k.first + j);
        const float x0 = xp[0], x1 = xp[1], x2 = xp[2];
        const float4 xw = mg_wrap_x(xp);
        ok = ok && __float_as_int(xw.w) != 0;
        sw.x[j] = xw;
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

// The table of translations is stored as three planes (x | y | z, MG_TLOC floats each) inside
// WarpSmem::T: four consecutive cells of one component are one LDS.128, and two cells go through
// one packed FP32 instruction (add / fma .f32x2 of sm_100: each half rounds like the scalar
// instruction, so the masks are those of the scalar filter).
__device__ __forceinline__ const float *mg_tplane(const WarpSmem &sw, int a) {
    return reinterpret_cast<const float *>(sw.T) + a * MG_TLOC;
}
__device__ __forceinline__ float4 mg_tcell(const WarpSmem &sw, int c) {
    return make_float4(mg_tplane(sw, 0)[c], mg_tplane(sw, 1)[c], mg_tplane(sw, 2)[c], 0.f);
}
// Local translations of cells [tile0, tile0 + MG_TLOC) of the per-pair sub-box m0 x m1 x m2:
// T = t . L in FP32, tcode = packed t; the tail is padded with a far-away sentinel.
__device__ __forceinline__ void mg_warp_table(WarpSmem &sw, const float a[9], int m1, int m2, int mloc,
                                              int tile0, int lane) {
    const int M12 = m1 * m2;
    const float inv12 = 1.f / (float)M12, inv2 = 1.f / (float)m2;
    __syncwarp();
#pragma unroll 1
    for (int cc = 0; cc < MG_TLOC && (cc == 0 || tile0 + cc < mloc); cc += 32) {
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
        float *tp = reinterpret_cast<float *>(sw.T);
        tp[c] = T.x; tp[MG_TLOC + c] = T.y; tp[2 * MG_TLOC + c] = T.z;
        sw.tcode[c] = code;
    }
    __syncwarp();
}

// Per-task constants of the find phase.
struct FindCtx {
    float a[9];            // lattice rows (FP32)
    const float *lat;      // the same, global
    const float *pos;      // positions of the batch (exact predicate)
    float rc;              // radius of the predicate d < rc
    const float *gx;       // positions of the structure's first atom
    bool big;              // more than MG_SMALL_MAX_ATOMS atoms: positions are read from global memory
    float rho[3];
    int m;                 // m_0 | m_1 << 8 | m_2 << 16
    int mloc;
    float nr2, win;        // -r_c^2, rounding window of d2
};

// One block of 32 ordered pairs against the cells [0, ncl) of the current table tile: hit masks in
// registers (W words = 32 W cells).  Lanes that saw a candidate inside the rounding window decide
// their window cells with the exact FP64 predicate.
template <int W>
__device__ __forceinline__ void mg_pair_masks(const WarpSmem &sw, const FindCtx &F,
                                              float qx, float qy, float qz, int gi, int gj,
                                              int l0, int l1, int l2, int ncl, unsigned (&mask)[W]) {
    bool near = false;
    const float nr2 = F.nr2, win = F.win;
    if (W == 1 && ncl == 1) {                     // one image per pair (cells wider than 2 r_c): T_0 = 0
        const float y = __fmaf_rn(qz, qz, __fmaf_rn(qy, qy, __fmaf_rn(qx, qx, nr2)));
        mask[0] = y < 0.f ? 0x80000000u : 0u;
        near = fabsf(y) < win;
    } else
#pragma unroll
    for (int w = 0; w < W; ++w) {
        // bit 31 - c <-> cell 32 w + c: the sign bits of y = |q' + T|^2 - r^2 are shifted in one by one, two
        // groups of four cells per trip (a group past the word's cells holds sentinels)
        unsigned m = 0u;
        const int n4 = min(8, max(0, (ncl - 32 * w + 3) >> 2)), n4r = (n4 + 1) & ~1;      // warp-uniform
        const float4 *Xp = reinterpret_cast<const float4 *>(mg_tplane(sw, 0) + 32 * w);
        const float4 *Yp = reinterpret_cast<const float4 *>(mg_tplane(sw, 1) + 32 * w);
        const float4 *Zp = reinterpret_cast<const float4 *>(mg_tplane(sw, 2) + 32 * w);
#pragma unroll 1                  // a loop, not 8 copies: the kernels are bound by instruction fetch
        for (int g = 0; g < n4r; g += 2) {
            float y[8];
            mg_filter4(Xp[g], Yp[g], Zp[g], make_float2(qx, qx), make_float2(qy, qy), make_float2(qz, qz),
                       make_float2(nr2, nr2), *reinterpret_cast<float (*)[4]>(&y[0]));
            mg_filter4(Xp[g + 1], Yp[g + 1], Zp[g + 1], make_float2(qx, qx), make_float2(qy, qy), make_float2(qz, qz),
                       make_float2(nr2, nr2), *reinterpret_cast<float (*)[4]>(&y[4]));
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                m = __funnelshift_l(__float_as_uint(y[c]), m, 1);
                near = near || fabsf(y[c]) < win;
            }
        }
        mask[w] = n4r == 0 ? 0u : (n4r < 8 ? m << (32 - 4 * n4r) : m);
    }
    if (near) {                                   // rare: decide the window cells in FP64
        const float *xi = F.pos + 3 * (size_t)gi, *xj = F.pos + 3 * (size_t)gj;
        for (int c = 0; c < ncl; ++c) {
            const float4 T = mg_tcell(sw, c);
            const float vx = __fadd_rn(qx, T.x), vy = __fadd_rn(qy, T.y), vz = __fadd_rn(qz, T.z);
            const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, nr2)));
            if (fabsf(y) < win) {
                const unsigned tc = sw.tcode[c];
                double v[3];
                const double d = mg_exact_vec(xi, xj, l0 + (int)(tc >> 24), l1 + (int)((tc >> 16) & 0xFFu),
                                              l2 + (int)((tc >> 8) & 0xFFu), F.lat, v);
                const unsigned bit = 0x80000000u >> (c & 31);
#pragma unroll
                for (int w = 0; w < W; ++w)
                    if (w == (c >> 5)) mask[w] = d < (double)F.rc ? (mask[w] | bit) : (mask[w] & ~bit);
            }
        }
    }
}


// One lane's ordered pair (i, j) of the staged structure: q' = (u + lo) . L with u = x_j - x_i
// (wrapped coordinates) and lo = floor(-rho - u) + 1 the first cell of the pair's sub-box; the cell
// offsets relative to the coordinates AS GIVEN start at l = lo + k_i - k_j.
struct PairLane {
    float qx, qy, qz;
    int l0, l1, l2;       // first cell (absolute)
    int self;             // index of the cell tau = 0 in the local table if i == j, else -1
    bool ok;              // valid lane and offsets inside int8
};

__device__ __forceinline__ PairLane mg_pair_setup(const WarpSmem &sw, const FindCtx &F, bool valid, int i, int j) {
    PairLane p;
    const int m0 = F.m & 0xFF, m1 = (F.m >> 8) & 0xFF, m2 = (F.m >> 16) & 0xFF;
    const float4 xi = F.big ? mg_wrap_x(F.gx + 3 * i) : sw.x[i], xj = F.big ? mg_wrap_x(F.gx + 3 * j) : sw.x[j];
    const float u0 = __fsub_rn(xj.x, xi.x), u1 = __fsub_rn(xj.y, xi.y), u2 = __fsub_rn(xj.z, xi.z);
    const float e0 = floorf(__fsub_rn(-F.rho[0], u0)) + 1.f, e1 = floorf(__fsub_rn(-F.rho[1], u1)) + 1.f,
                e2 = floorf(__fsub_rn(-F.rho[2], u2)) + 1.f;
    const float f0 = __fadd_rn(u0, e0), f1 = __fadd_rn(u1, e1), f2 = __fadd_rn(u2, e2);
    p.qx = __fmaf_rn(f2, F.a[6], __fmaf_rn(f1, F.a[3], __fmul_rn(f0, F.a[0])));
    p.qy = __fmaf_rn(f2, F.a[7], __fmaf_rn(f1, F.a[4], __fmul_rn(f0, F.a[1])));
    p.qz = __fmaf_rn(f2, F.a[8], __fmaf_rn(f1, F.a[5], __fmul_rn(f0, F.a[2])));
    const int ki = __float_as_int(xi.w), kj = __float_as_int(xj.w);
    p.l0 = (int)e0 + (ki & 1023) - (kj & 1023);
    p.l1 = (int)e1 + ((ki >> 10) & 1023) - ((kj >> 10) & 1023);
    p.l2 = (int)e2 + ((ki >> 20) & 1023) - ((kj >> 20) & 1023);
    p.ok = valid && ki != 0 && kj != 0 && p.l0 >= -127 && p.l1 >= -127 && p.l2 >= -127 && p.l0 + m0 <= 128 && p.l1 + m1 <= 128 &&
           p.l2 + m2 <= 128;
    if (!p.ok) { p.qx = 1e18f; p.qy = 1e18f; p.qz = 1e18f; }
    p.self = i == j ? (-(int)e0 * m1 - (int)e1) * m2 - (int)e2 : -1;   // (i,i,0) is not an edge (R3)
    return p;
}

template <int W>
__device__ __forceinline__ void mg_block_masks(const WarpSmem &sw, const FindCtx &F,
                                               const PairLane &p, int gi, int gj, int tile0, int ncl,
                                               unsigned (&mask)[W]) {
    mg_pair_masks<W>(sw, F, p.qx, p.qy, p.qz, gi, gj, p.l0, p.l1, p.l2, ncl, mask);
    const int cs = p.self - tile0;
#pragma unroll
    for (int w = 0; w < W; ++w)
        if (p.self >= 0 && cs >= 32 * w && cs < 32 * w + 32) mask[w] &= ~(0x80000000u >> (cs & 31));
}

// The same for ONE word of the mask — cells [32 w, 32 w + 32) of the table tile that starts at cell
// tile0 and holds ncl cells — with the word index a run-time value: the cutoff kernels have one copy
// of this code for tables of every size (they are bound by instruction fetch, profiles/).
__device__ __forceinline__ unsigned mg_word_mask(const WarpSmem &sw, const FindCtx &F, const PairLane &p, int gi,
                                                 int gj, int tile0, int w, int ncl) {
    const float nr2 = F.nr2, win = F.win;
    const int nw = min(32, ncl - 32 * w);                        // cells of the word (warp-uniform)
    const float4 *Xp = reinterpret_cast<const float4 *>(mg_tplane(sw, 0) + 32 * w);
    const float4 *Yp = reinterpret_cast<const float4 *>(mg_tplane(sw, 1) + 32 * w);
    const float4 *Zp = reinterpret_cast<const float4 *>(mg_tplane(sw, 2) + 32 * w);
    unsigned mask = 0u;
    bool near = false;
    if (ncl == 1 && tile0 == 0) {                                // one image per pair: T_0 = 0
        const float y = __fmaf_rn(p.qz, p.qz, __fmaf_rn(p.qy, p.qy, __fmaf_rn(p.qx, p.qx, nr2)));
        mask = y < 0.f ? 0x80000000u : 0u;
        near = fabsf(y) < win;
    } else {
        // bit 31 - c <-> cell c of the word: sign bits shifted in, two groups of four cells per trip
        const int n4r = (((nw + 3) >> 2) + 1) & ~1;
#pragma unroll 1
        for (int g = 0; g < n4r; g += 2) {
            float y[8];
            mg_filter4(Xp[g], Yp[g], Zp[g], make_float2(p.qx, p.qx), make_float2(p.qy, p.qy),
                       make_float2(p.qz, p.qz), make_float2(nr2, nr2), *reinterpret_cast<float (*)[4]>(&y[0]));
            mg_filter4(Xp[g + 1], Yp[g + 1], Zp[g + 1], make_float2(p.qx, p.qx), make_float2(p.qy, p.qy),
                       make_float2(p.qz, p.qz), make_float2(nr2, nr2), *reinterpret_cast<float (*)[4]>(&y[4]));
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                mask = __funnelshift_l(__float_as_uint(y[c]), mask, 1);
                near = near || fabsf(y[c]) < win;
            }
        }
        mask = n4r < 8 ? mask << (32 - 4 * n4r) : mask;
    }
    if (near) {                                   // rare: decide the window cells in FP64
        const float *xi = F.pos + 3 * (size_t)gi, *xj = F.pos + 3 * (size_t)gj;
        for (int c = 0; c < nw; ++c) {
            const float4 T = mg_tcell(sw, 32 * w + c);
            const float vx = __fadd_rn(p.qx, T.x), vy = __fadd_rn(p.qy, T.y), vz = __fadd_rn(p.qz, T.z);
            const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, nr2)));
            if (fabsf(y) < win) {
                const unsigned tc = sw.tcode[32 * w + c];
                double v[3];
                const double d = mg_exact_vec(xi, xj, p.l0 + (int)(tc >> 24), p.l1 + (int)((tc >> 16) & 0xFFu),
                                              p.l2 + (int)((tc >> 8) & 0xFFu), F.lat, v);
                mask = d < (double)F.rc ? (mask | (0x80000000u >> c)) : (mask & ~(0x80000000u >> c));
            }
        }
    }
    const int cs = p.self - tile0 - 32 * w;       // (i, i, 0) is not an edge
    if (p.self >= 0 && cs >= 0 && cs < 32) mask &= ~(0x80000000u >> cs);
    return mask;
}

// Constants of the find phase for structure s with radius rc; stages the structure (positions,
// table when it fits).  Returns false if the structure emits nothing (empty, invalid lattice or
// positions).
__device__ __forceinline__ bool mg_struct_setup(WarpSmem &sw, double (*pd)[3], const float *pos, const float *lattice,
                                                unsigned *status, float rc, const CutRec *R, int s, Task &k,
                                                FindCtx &F, int lane) {
    k.s = s;
    k.first = R->first;
    k.natoms = R->natoms;
    F.lat = lattice + 9 * (size_t)s;
    F.pos = pos;
    F.rc = rc;
    F.mloc = R->mloc;
    if (F.mloc <= 0) return false;
#pragma unroll
    for (int c = 0; c < 9; ++c) F.a[c] = __ldg(F.lat + c);
#pragma unroll
    for (int a = 0; a < 3; ++a) F.rho[a] = R->rho[a];
    F.m = R->m;
    F.nr2 = -__fmul_rn(rc, rc);
    // FP32 error bound of d2 - rc^2 near the threshold (R23): the components of q', T
    // and q' + T are below 3 Q, about 13 roundings of 2^-24 relative size reach v (the wrapped
    // coordinates are below 1, their difference is rounded once), d2 = v . v adds 3 more
    F.win = 1.1920929e-7f * (2.f * rc * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * rc * rc);
    F.gx = pos + 3 * (size_t)k.first;
    F.big = k.natoms > MG_SMALL_MAX_ATOMS;
    if (!F.big && !mg_warp_stage(sw, pd, pos, lattice, k, lane)) {
        if (lane == 0) atomicOr(status, MGS_NONFINITE);
        F.mloc = 0;
        return false;
    }
    if (F.mloc <= MG_TLOC) mg_warp_table(sw, F.a, (F.m >> 8) & 0xFF, (F.m >> 16) & 0xFF, F.mloc, 0, lane);
    return true;
}

// ---------------------------------------------------------------------------------------------
// Launch 1: count.  Pairs [qa, qb) of the staged structure: hit masks -> edge count (per lane);
// the masks go to the warp's scratch for the emit launch while they fit (ceil(mloc / 32) words per
// lane and block of 32 pairs).  Structures whose table does not fit (mloc > MG_TLOC) walk their
// pairs once per tile of the table and keep nothing.
__device__ __forceinline__ unsigned mg_count_struct(WarpSmem &sw, const CutoffArgs &A, const Task &k,
                                                    const FindCtx &F, int qa, int qb, unsigned *wmask, int &midx,
                                                    int lane) {
    const int N = k.natoms;
    const float inv_N = 1.f / (float)N;
    const bool tiled = F.mloc > MG_TLOC;
    unsigned acc = 0u;
    for (int tile0 = 0; tile0 < F.mloc; tile0 += MG_TLOC) {
        const int ncl = min(MG_TLOC, F.mloc - tile0), nW = (ncl + 31) >> 5;
        if (tiled) mg_warp_table(sw, F.a, (F.m >> 8) & 0xFF, (F.m >> 16) & 0xFF, F.mloc, tile0, lane);
        for (int q0 = qa; q0 < qb; q0 += 32) {
            const int q = q0 + lane;
            const bool valid = q < qb;
            int i = 0, j = 0;
            if (valid) mg_qsplit(q, N, inv_N, i, j);
            const PairLane p = mg_pair_setup(sw, F, valid, i, j);
            if (valid && !p.ok && tile0 == 0) atomicOr(A.status, MGS_OFFSET);
            const bool keep = !tiled && midx + 32 * nW <= A.mask_words;
#pragma unroll 1
            for (int w = 0; w < nW; ++w) {
                const unsigned m = mg_word_mask(sw, F, p, k.first + i, k.first + j, tile0, w, ncl);
                acc += __popc(m);
                if (keep) wmask[midx + 32 * w + lane] = m;
            }
            if (!tiled) midx += 32 * nW;
        }
    }
    return acc;
}

// Structures with ONE candidate image per pair (mloc == 1: every plane spacing above 2 r_c, e.g. the
// supercells of BASELINE configs[3] — the minimum-image limit): the hit mask of a block of 32 pairs
// is one ballot word.  Returns the block's hits on lane 0 only (the caller reduces over lanes).
__device__ __forceinline__ unsigned mg_single_word(const WarpSmem &sw, const CutoffArgs &A, const Task &k,
                                                   const FindCtx &F, int q0, int qb, float inv_N, bool report,
                                                   int lane) {
    const int q = q0 + lane;
    const bool valid = q < qb;
    int i = 0, j = 0;
    if (valid) mg_qsplit(q, k.natoms, inv_N, i, j);
    const PairLane p = mg_pair_setup(sw, F, valid, i, j);
    if (report && valid && !p.ok) atomicOr(A.status, MGS_OFFSET);
    const unsigned m = mg_word_mask(sw, F, p, k.first + i, k.first + j, 0, 0, 1);
    return __ballot_sync(0xFFFFFFFFu, (m >> 31) != 0u);
}

// (its own structure setup: no table, no FP64 positions in the count launch)
__device__ __forceinline__ unsigned mg_count_single(WarpSmem &sw, const CutoffArgs &A, const CutRec *R, int s, int qa,
                                                 int qb, unsigned *wmask, int midx, int lane) {
    Task k;
    FindCtx F;
    if (!mg_struct_setup(sw, nullptr, A.pos, A.lattice, A.status, A.r_c, R, s, k, F, lane)) return 0u;
    const float inv_N = 1.f / (float)k.natoms;
    unsigned acc = 0u;
    for (int q0 = qa; q0 < qb; q0 += 32) {
        const unsigned word = mg_single_word(sw, A, k, F, q0, qb, inv_N, true, lane);
        if (lane == 0) {
            acc += __popc(word);
            if (midx < A.mask_words) wmask[midx] = word;
        }
        midx += 1;
    }
    return acc;
}

// The ranges of one warp.
__device__ __forceinline__ void mg_count_ranges(WarpSmem &sw, const CutoffArgs &A, const RangeCtx &RC, int wid,
                                                int lane) {
    // one range per warp (n_ranges == n_warps): no ticket, nothing that counts calls
    for (int w = wid; w < A.n_ranges; w += A.n_warps) {
        unsigned long long c0, c1;
        mg_warp_range(RC, w, c0, c1);
        int s, qa;
        mg_range_start(RC, c0, s, qa, lane);
        if (lane == 0) A.wstart[w] = make_int2(s, qa);
        unsigned *wmask = A.wmask + (size_t)w * MG_MASK_WORDS;
        int midx = 0;
        unsigned total = 0u;
        for (; s < A.n_struct; ++s, qa = 0) {
            const CutRec *R = A.rec + s;
            int qb;
            if (!mg_segment(RC, R, s, qa, c1, qb)) break;
            Task k;
            FindCtx F;
            if (qb > qa && R->mloc == 1) {
                total += mg_count_single(sw, A, R, s, qa, qb, wmask, midx, lane);
                midx += (qb - qa + 31) >> 5;
            } else if (qb > qa && mg_struct_setup(sw, nullptr, A.pos, A.lattice, A.status, A.r_c, R, s, k, F, lane)) {
                total += mg_count_struct(sw, A, k, F, qa, qb, wmask, midx, lane);
            }
            if (qb < R->natoms * R->natoms) break;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xFFFFFFFFu, total, o);
        if (lane == 0) {
            A.wtotal[w] = total;
            atomicAdd(A.gtotal + w / ((A.n_ranges + 63) >> 6), total);
        }
    }
}

#ifndef MG_CUT_CTAS
#define MG_CUT_CTAS 4
#endif
__global__ void __launch_bounds__(MG_BLOCK, MG_CUT_CTAS)
mg_cutoff_count_kernel(const __grid_constant__ CutoffArgs A) {
    mg_grid_dependency_wait();
    __shared__ WarpSmem s_w[MG_WARPS];
    __shared__ unsigned long long s_part[MG_BLOCK];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem &sw = s_w[warp];
    // consecutive ranges (often parts of one expensive structure) go to different SMs
    const int wid = warp * gridDim.x + blockIdx.x;
#ifdef MG_PHASE_CLOCKS
    const long long t_begin = clock64();
#endif
    RangeCtx RC;
    mg_range_init(RC, A.rec, A.bpre, A.n_blocks, A.n_struct, A.n_ranges, lane);
    mg_count_ranges(sw, A, RC, wid, lane);
#ifdef MG_PHASE_CLOCKS
    if (lane == 0) A.wclock[wid] = (unsigned)(clock64() - t_begin);
#endif
    // The emit launch sums the totals of the ranges before its own itself (one coalesced pass per
    // warp, overlapped with the other warps' work): no tail in this launch.  mg_cutoff_count has no
    // emit launch: ---- last CTA out: exclusive scan of the warp totals, grand total
    if (!A.count_only) return;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(A.ctl + 1, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int nw = A.n_ranges, per = (nw + MG_BLOCK - 1) / MG_BLOCK;
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
    if (threadIdx.x < 64) A.gtotal[threadIdx.x] = 0u;
}

// ---------------------------------------------------------------------------------------------
// Launch 2: emit.
struct EmitCtx {
    double Ld[9];
    long long goff;        // global index of the first edge in the stash
    int run, qb0;          // stash fill, first pair of the stash's batch
    const float *gx;       // positions of the structure's first atom
    bool big;              // positions are not staged: FP64 cartesian positions on the fly
#ifdef MG_PHASE_CLOCKS
    long long tc[6];       // cycles: pair setup + masks + scan, extraction, flush, structure setup,
                           // range prologue, segment bounds
#endif
};
#ifdef MG_PHASE_CLOCKS
#define MG_TIC const long long tic_ = clock64();
#define MG_TOC(i) E.tc[i] += clock64() - tic_;
#else
#define MG_TIC
#define MG_TOC(i)
#endif

// Stash -> global: lanes over consecutive edges; the low byte of a code is the pair's index
// relative to qb0.  vec = (p_j - p_i) + tau . L in FP64, rounded once (R24).
__device__ __forceinline__ void mg_flush(const EmitSmem &se, const CutoffArgs &A, const Task &k, const EmitCtx &E,
                                         int run, int qb0, float inv_N, int lane) {
    if (run == 0) return;
    const int N = k.natoms;
    // edges that fit the caller's arrays (all of them unless the capacity is exceeded)
    const long long room = A.capacity - E.goff;
    const int lim = room >= run ? run : (room > 0 ? (int)room : 0);
    int32_t *psrc = A.src + E.goff, *pdst = A.dst + E.goff;
    int8_t *poff = A.offset + 3 * E.goff;
    float *pvec = A.vec + 3 * E.goff;
    float *pdist = A.dist ? A.dist + E.goff : nullptr;
    // two edges per lane and iteration: two independent load -> FP64 -> store chains in flight
    for (int e0 = lane; e0 < lim; e0 += 32) {
#pragma unroll
        for (int h = 0; h < 1; ++h) {
            const int e = e0 + 32 * h;
            if (e >= lim) break;
            const unsigned code = se.stash[e];
            const int q = qb0 + (int)(code & 0xFFu);
            int i, j;
            mg_qsplit(q, N, inv_N, i, j);
            double pib[3], pjb[3];
            const double *pi = se.pd[i], *pj = se.pd[j];
            if (E.big) {
                mg_pd_big(E.gx, E.Ld, i, pib);
                mg_pd_big(E.gx, E.Ld, j, pjb);
                pi = pib;
                pj = pjb;
            }
            // (double)(b - 128) without a conversion instruction: 2^52 + b has b in its low mantissa word
            const double t0 = __hiloint2double(0x43300000, (int)(code >> 24)) - 4503599627370624.0;
            const double t1 = __hiloint2double(0x43300000, (int)((code >> 16) & 0xFFu)) - 4503599627370624.0;
            const double t2 = __hiloint2double(0x43300000, (int)((code >> 8) & 0xFFu)) - 4503599627370624.0;
            const double v0 = fma(t2, E.Ld[6], fma(t1, E.Ld[3], fma(t0, E.Ld[0], pj[0] - pi[0])));
            const double v1 = fma(t2, E.Ld[7], fma(t1, E.Ld[4], fma(t0, E.Ld[1], pj[1] - pi[1])));
            const double v2 = fma(t2, E.Ld[8], fma(t1, E.Ld[5], fma(t0, E.Ld[2], pj[2] - pi[2])));
            const unsigned tb = code ^ 0x80808000u;              // tau bytes as int8
            psrc[e] = k.first + i;
            pdst[e] = k.first + j;
            int8_t *po = poff + 3 * e;
            po[0] = (int8_t)(tb >> 24); po[1] = (int8_t)(tb >> 16); po[2] = (int8_t)(tb >> 8);
            float *pv = pvec + 3 * e;
            pv[0] = (float)v0; pv[1] = (float)v1; pv[2] = (float)v2;
            if (pdist) pdist[e] = __fsqrt_rn((float)fma(v2, v2, fma(v1, v1, v0 * v0)));
        }
    }
}

// Pairs [qa, qb) of the staged structure -> edges.  The hit masks of a block of 32 pairs live in MW
// registers, of which the first nW = ceil(cells / 32) are used: three instances (MW = 1, 2: 98 % of
// the pairs of an MP-like batch; 8: everything else), not one per table size — the kernel is bound
// by instruction fetch (profiles/).
//   * the table fits (mloc <= MG_TLOC): one segment [qa, qb), the masks are read back from the
//     scratch of the count launch one block ahead (evaluated again once the scratch is exhausted);
//   * it does not: segments of at most 256 pairs of ONE source row (pair indices in the stash are
//     8 bit), each walked once per tile of the table; the edges of a row then come tile by tile,
//     the row stays contiguous (canonical order inside a row is not kept).
// Hits go to the stash (pair indices relative to E.qb0) and are written out when it is full, when
// the pair index would overflow, and at the end of a segment: the pass q0 >= rb of the block loop
// only flushes (one flush site).
template <int MW>
__device__ __forceinline__ void mg_emit_struct(EmitSmem &se, const CutoffArgs &A, const Task &k, const FindCtx &F,
                                               EmitCtx &E, int qa, int qb, const unsigned *wmask, int &midx,
                                               int lane) {
    WarpSmem &sw = se.w;
    const int N = k.natoms;
    const float inv_N = 1.f / (float)N;
    const bool tiled = F.mloc > MG_TLOC;
    for (int ra = qa; ra < qb;) {
        int rb = qb;
        if (tiled) rb = min(min(qb, (ra / N + 1) * N), ra + 256);
        E.qb0 = ra;
        for (int tile0 = 0; tile0 < F.mloc; tile0 += MG_TLOC) {
            const int ncl = min(MG_TLOC, F.mloc - tile0), nW = (ncl + 31) >> 5;
            const bool last_tile = tile0 + MG_TLOC >= F.mloc;
            if (tiled) mg_warp_table(sw, F.a, (F.m >> 8) & 0xFF, (F.m >> 16) & 0xFF, F.mloc, tile0, lane);
            unsigned nmask[MW];                   // masks of the next block, loaded one block ahead
            bool nhave = !tiled && midx + 32 * nW <= A.mask_words;
#pragma unroll
            for (int w = 0; w < MW; ++w) nmask[w] = nhave && w < nW ? __ldg(wmask + midx + 32 * w + lane) : 0u;
            for (int q0 = ra;; q0 += 32) {
                const bool last = q0 >= rb;      // flush-only pass
                const int q = q0 + lane;
                const bool valid = q < rb;
                int i = 0, j = 0, cnt = 0, tot = 0, incl = 0;
                unsigned mask[MW];
                PairLane p;
                if (!last) {
                    MG_TIC
                    if (valid) mg_qsplit(q, N, inv_N, i, j);
                    p = mg_pair_setup(sw, F, valid, i, j);
#pragma unroll
                    for (int w = 0; w < MW; ++w) mask[w] = nmask[w];
                    if (!nhave) {
#pragma unroll 1
                        for (int w = 0; w < nW; ++w) {
                            const unsigned m = mg_word_mask(sw, F, p, k.first + i, k.first + j, tile0, w, ncl);
#pragma unroll
                            for (int x = 0; x < MW; ++x)
                                if (x == w) mask[x] = m;
                        }
                    }
                    if (!tiled) {
                        midx += 32 * nW;
                        nhave = q0 + 32 < rb && midx + 32 * nW <= A.mask_words;
#pragma unroll
                        for (int w = 0; w < MW; ++w)
                            nmask[w] = nhave && w < nW ? __ldg(wmask + midx + 32 * w + lane) : 0u;
                    }
#pragma unroll
                    for (int w = 0; w < MW; ++w) {
                        if (w >= nW) break;
                        cnt += __popc(mask[w]);
                    }
                    incl = cnt;                  // inclusive scan of the lanes' hit counts
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                        if (lane >= o) incl += v;
                    }
                    tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
                    MG_TOC(0)
                }
                // a block with more hits than the stash holds goes in several passes of consecutive
                // lanes (a lane has at most 256 hits): done = hits of the lanes already written
                const bool split = tot > MG_STASH;
                for (int done = 0, l0 = 0;;) {
                    bool mine = true;
                    int c = cnt, t = tot;
                    if (split) {                 // rare
                        mine = lane >= l0 && incl - done <= MG_STASH;
                        const int nl = __popc(__ballot_sync(0xFFFFFFFFu, mine));
                        t = __shfl_sync(0xFFFFFFFFu, incl, l0 + nl - 1) - done;
                        c = mine ? cnt : 0;
                        l0 += nl;
                    }
                    const bool full = E.run + t > MG_STASH || (!tiled && q0 + 32 - E.qb0 > 256);
                    if (last ? (last_tile && E.run > 0) : full) {              // write the stash out
                        __syncwarp();
                        { MG_TIC mg_flush(se, A, k, E, E.run, E.qb0, inv_N, lane); MG_TOC(2) }
                        __syncwarp();
                        E.goff += E.run;
                        E.run = 0;
                        if (!tiled) E.qb0 = q0;
                    }
                    if (last) break;
                    int pos = E.run + incl - cnt - done;
                    if (valid && j == 0 && tile0 == 0 && mine)
                        A.row_ptr[k.first + i] = (int)(E.goff + pos);
                    const unsigned paircode = ((unsigned)(p.l0 + 128) << 24) | ((unsigned)(p.l1 + 128) << 16) |
                                              ((unsigned)(p.l2 + 128) << 8) | (unsigned)(q - E.qb0);
                    { MG_TIC
#pragma unroll
                    for (int w = 0; w < MW; ++w) {
                        if (w >= nW) break;
                        unsigned mk = mine ? mask[w] : 0u;
                        while (mk) {
                            const int b = __clz(mk);
                            mk &= ~(0x80000000u >> b);
                            se.stash[pos++] = paircode + sw.tcode[32 * w + b];
                        }
                    }
                    MG_TOC(1) }
                    E.run += t;
                    done += t;
                    if (done >= tot) break;
                }
                if (last) break;
            }
        }
        ra = rb;
    }
}

// Emit for structures with one candidate image per pair (mloc == 1): 32 blocks (1024 pairs) at a
// time, one ballot word per lane; the hits are expanded into a list and then LANES <-> HITS, so the
// per-pair work (cell offsets, FP64 vec) is done for the edges only and the stores are coalesced.
// Returns the edge offset after the segment; the caller advances midx by ceil((qb - qa) / 32).
__device__ __forceinline__ long long mg_emit_single(EmitSmem &se, const CutoffArgs &A, const CutRec *R, int s, int qa,
                                                 int qb, const unsigned *wmask, int midx, long long goff, int lane) {
    WarpSmem &sw = se.w;
    Task k;
    FindCtx F;
    if (!mg_struct_setup(sw, se.pd, A.pos, A.lattice, A.status, A.r_c, R, s, k, F, lane)) {
        const int N0 = R->natoms;                  // no edges: rows that start in [qa, qb)
        for (int i = (qa + N0 - 1) / N0 + lane; i * N0 < qb; i += 32) A.row_ptr[R->first + i] = (int)goff;
        return goff;
    }
    double Ld[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) Ld[c] = (double)F.a[c];
    const int N = k.natoms;
    const float inv_N = 1.f / (float)N;
    for (int g0 = qa; g0 < qb; g0 += 1024) {
        const int gend = min(qb, g0 + 1024), nb = (gend - g0 + 31) >> 5;
        unsigned word = 0u;
        if (midx + nb <= A.mask_words) {
            if (lane < nb) word = __ldg(wmask + midx + lane);
        } else {                                   // scratch exhausted in the count launch: evaluate again
            for (int b = 0; b < nb; ++b) {
                const unsigned wb = mg_single_word(sw, A, k, F, g0 + 32 * b, qb, inv_N, false, lane);
                if (lane == b) word = wb;
            }
        }
        midx += nb;
        const int cnt = __popc(word);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        const int excl = incl - cnt, T = __shfl_sync(0xFFFFFFFFu, incl, 31);
        // row_ptr of the source rows whose first pair lies in this group
        for (int r0 = (g0 + N - 1) / N; r0 * N < gend; r0 += 32) {
            const int r = r0 + lane;
            const bool act = (long long)r * N < gend;
            const int qr = act ? r * N - g0 : 0;
            const unsigned wv = __shfl_sync(0xFFFFFFFFu, word, qr >> 5);
            const int ev = __shfl_sync(0xFFFFFFFFu, excl, qr >> 5);
            if (act) A.row_ptr[k.first + r] = (int)(goff + ev + __popc(wv & ((1u << (qr & 31)) - 1u)));
        }
        // hit list: pair indices relative to g0, in (i, j) order
        __syncwarp();
        {
            unsigned mk = word;
            int pos = excl;
            while (mk) {
                const int b = __ffs(mk) - 1;
                mk &= mk - 1;
                se.stash[pos++] = (unsigned)(32 * lane + b);
            }
        }
        __syncwarp();
        const long long room = A.capacity - goff;
        const int lim = room >= T ? T : (room > 0 ? (int)room : 0);
        for (int h = lane; h < lim; h += 32) {
            const int q = g0 + (int)se.stash[h];
            int i, j;
            mg_qsplit(q, N, inv_N, i, j);
            const PairLane p = mg_pair_setup(sw, F, true, i, j);         // tau = first (only) cell of the pair
            double pib[3], pjb[3];
            const double *pi = se.pd[F.big ? 0 : i], *pj = se.pd[F.big ? 0 : j];
            if (F.big) {
                mg_pd_big(F.gx, Ld, i, pib);
                mg_pd_big(F.gx, Ld, j, pjb);
                pi = pib;
                pj = pjb;
            }
            mg_emit_edge(A, goff + h, k.first + i, k.first + j, pi, pj, Ld, (unsigned)(p.l0 + 128),
                         (unsigned)(p.l1 + 128), (unsigned)(p.l2 + 128));
        }
        __syncwarp();
        goff += T;
    }
    return goff;
}

__device__ __forceinline__ void mg_emit_ranges(EmitSmem &se, const CutoffArgs &A, const RangeCtx &RC, int wid,
                                               int lane) {
    WarpSmem &sw = se.w;
    for (int w = wid; w < A.n_ranges; w += A.n_warps) {
#ifdef MG_PHASE_CLOCKS
        const long long t_range = clock64();
#endif
        unsigned long long c0, c1;
        mg_warp_range(RC, w, c0, c1);
        const int2 st = A.wstart[w];
        int s = st.x, qa = st.y;
        const unsigned *wmask = A.wmask + (size_t)w * MG_MASK_WORDS;
        int midx = 0;
        EmitCtx E;
#ifdef MG_PHASE_CLOCKS
        E.tc[0] = E.tc[1] = E.tc[2] = E.tc[3] = E.tc[4] = E.tc[5] = 0;
#endif
        {   // device-wide scan of K4, consumer side: edges of the ranges before this one
            // (group totals + the ranges of the own group: 4 independent loads per lane)
            unsigned long long before = 0ull;
            const int gs = (A.n_ranges + 63) >> 6, g = w / gs;
            for (int x = lane; x < g; x += 32) before += __ldg(A.gtotal + x);
            for (int c = g * gs + lane; c < w; c += 32) before += __ldg(A.wtotal + c);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) before += __shfl_xor_sync(0xFFFFFFFFu, before, o);
            E.goff = (long long)before;
            if (w == A.n_ranges - 1 && lane == 0) {          // the last range also knows the grand total
                const unsigned long long tot = before + __ldg(A.wtotal + w);
                *A.n_edges = (long long)tot;
                A.row_ptr[A.n_atoms] = (int)tot;
                if (tot > 0x7FFFFFFFull || (long long)tot > A.capacity) atomicOr(A.status, MGS_CAPACITY);
            }
        }
#ifdef MG_PHASE_CLOCKS
        E.tc[4] = clock64() - t_range;
#endif
        for (; s < A.n_struct; ++s, qa = 0) {
            const CutRec *R = A.rec + s;
            int qb;
            bool more_;
            { MG_TIC more_ = mg_segment(RC, R, s, qa, c1, qb); MG_TOC(5) }
            if (!more_) break;
            Task k;
            FindCtx F;
            if (qb > qa && R->mloc == 1) {
                E.goff = mg_emit_single(se, A, R, s, qa, qb, wmask, midx, E.goff, lane);
                midx += (qb - qa + 31) >> 5;
            } else if (qb > qa) {
                bool live_;
                { MG_TIC live_ = mg_struct_setup(sw, se.pd, A.pos, A.lattice, A.status, A.r_c, R, s, k, F, lane); MG_TOC(3) }
                if (!live_) {
                    const int N = R->natoms;                       // no edges: rows that start in [qa, qb)
                    for (int i = (qa + N - 1) / N + lane; i * N < qb; i += 32) A.row_ptr[R->first + i] = (int)E.goff;
                } else {
#pragma unroll
                    for (int c = 0; c < 9; ++c) E.Ld[c] = (double)F.a[c];
                    E.run = 0;
                    E.qb0 = qa;
                    E.gx = F.gx;
                    E.big = F.big;
                    if (F.mloc <= 64) mg_emit_struct<2>(se, A, k, F, E, qa, qb, wmask, midx, lane);
                    else mg_emit_struct<8>(se, A, k, F, E, qa, qb, wmask, midx, lane);
                }
            }
            if (qb < R->natoms * R->natoms) break;
        }
#ifdef MG_PHASE_CLOCKS
        if (lane == 0) for (int x = 0; x < 6; ++x) A.wmask[(size_t)w * MG_MASK_WORDS + MG_MASK_WORDS - 6 + x] = (unsigned)E.tc[x];
#endif
    }
}

__global__ void __launch_bounds__(MG_BLOCK, MG_CUT_CTAS)
mg_cutoff_emit_kernel(const __grid_constant__ CutoffArgs A) {
    mg_grid_dependency_wait();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    EmitSmem &se = reinterpret_cast<EmitSmem *>(smem_raw)[warp];
    // consecutive ranges (often parts of one expensive structure) go to different SMs
    const int wid = warp * gridDim.x + blockIdx.x;
#ifdef MG_PHASE_CLOCKS
    const long long t_begin = clock64();
#endif
    RangeCtx RC;
    mg_range_init(RC, A.rec, A.bpre, A.n_blocks, A.n_struct, A.n_ranges, lane);
    mg_emit_ranges(se, A, RC, wid, lane);
#ifdef MG_PHASE_CLOCKS
    if (lane == 0) A.wclock[A.n_warps + wid] = (unsigned)(clock64() - t_begin);
#endif
    // last CTA out zeroes the group totals for the next call
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(A.ctl + 9, 1u) == gridDim.x - 1) {
            A.ctl[9] = 0u;
            for (int x = 0; x < 64; ++x) A.gtotal[x] = 0u;
        }
    }
}
