// cut_fused.cuh — cutoff graph (K3 distance filter, K4 count -> device-wide scan -> emit, K6 batching,
// SURVEY.md 8(a)) in ONE launch of co-resident CTAs whose warps work on their own.
//
// mg_cut_prep_kernel gives every ordered pair (i, j) an estimated cost; warp r of the grid (r = 4 *
// blockIdx.x + warp: the warps of a CTA own consecutive ranges) owns the source rows whose first pair
// lies in the r-th of n_ranges equally expensive, contiguous ranges of the batch's pairs in
// (structure, i, j) order — which is the CSR order of the output.  A warp walks its rows twice:
//
//   count   per structure: stage the wrapped positions and the table of local translations in the
//           warp's shared memory, then blocks of 32 ordered pairs: lane <-> pair, FP32 filter over
//           the pair's sub-box (cut_prep.cuh; FP64 decision inside the rounding window, R23).
//           The 32-bit hit masks go to the warp's scratch in global memory (L2 resident).
//   scan    warp totals -> CTA total, published in a slot tagged with the call's epoch; warp 0 sums
//           the slots of the CTAs before its own (all CTAs are resident: cooperative launch): the
//           device-wide exclusive scan of K4 without a second launch and without a look-back chain.
//   emit    the same walk: masks read back, the hits of a block compacted into the warp's stash in
//           (row, j, t) order, row_ptr from the running offset; then LANES <-> EDGES: vec = (x_j - x_i
//           + l) . L + t . L in FP64 (the pair's part once per pair, the table's part from an FP64
//           table), rounded once (R24).  src / dst leave as coalesced 4-byte stores; vec and offset
//           are staged in shared memory at the misalignment of their global address and leave as
//           aligned 16-byte stores (scalar stores only for a ragged first / last piece).
//
// Structures the pair-lane path does not take (more than MGW_NMAX atoms, a sub-box of more than MGW_TL
// cells) go row by row through mgw_rows_*: lanes over the candidates (j, t) of one source row, ballot
// compaction, no table — exact and general, not tuned.
#pragma once
#include "common.cuh"
#include "cut_prep.cuh"
#include "cutoff_pairs.cuh"

#define MGF_BLOCK 128
#define MGF_WARPS (MGF_BLOCK / 32)
#define MGW_TL MG_PAIR_TL          // cells of a warp's table
#define MGW_NMAX 64                // atoms of a staged structure
#define MGW_STASH 256              // edges per pass
#define MGW_RING 512               // units (floats of vec / bytes of offset) of the output rings
#define MGF_MASK_WORDS 16384       // 32-bit words of mask scratch per CTA
#define MGW_MASK_WORDS (MGF_MASK_WORDS / MGF_WARPS)

struct FusedArgs {
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
    const unsigned long long *bpre;
    int n_blocks;
    unsigned *wmask;               // [gridDim.x, MGF_MASK_WORDS]
    int mask_words;                // words of a warp's scratch that may be used (tests: less)
    unsigned long long *slots;     // [gridDim.x] (epoch + 1) << 32 | edges of the CTA
    unsigned *ctl;                 // [10] epoch of the last finished call, [11] CTAs done
    unsigned *status;
    int count_only;
    unsigned *dbg;                 // MG_PHASE_CLOCKS builds: [gridDim.x, 4] globaltimer at the phase boundaries
};

#ifdef MG_PHASE_CLOCKS
__device__ __forceinline__ unsigned mgf_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return (unsigned)t;
}
#define MGF_STAMP(i) if (threadIdx.x == 0 && A.dbg) A.dbg[4 * blockIdx.x + (i)] = mgf_now();
#else
#define MGF_STAMP(i)
#endif

struct __align__(16) PairRec {         // per pair of the block: (x_j - x_i + l) . L, (l + 128) bytes << 8, i | j << 16
    double bx, by, bz;
    unsigned plc, pij;
};
struct __align__(16) CellRec {         // per cell of the table: t . L in FP64, t0 << 24 | t1 << 16 | t2 << 8
    double tx, ty, tz;
    unsigned tcode, pad;
};

#define MGW_RE 128                     // edges of the output rings
#define MGW_BATCH 96                   // edges per flush batch (+ the carried ragged piece < MGW_RE)

struct WSmem {                         // one warp's shared memory
    float T[3][MGW_TL + 4];            // t . L: planes x | y | z (+ one group read ahead)
    unsigned tcode[MGW_TL];            // t0 << 24 | t1 << 16 | t2 << 8
    CellRec cr[MGW_TL];                // (emit)
    float4 x[MGW_NMAX];                // wrapped fractional coordinates, .w = packed integer parts
    unsigned stash[MGW_STASH];         // (pair of the block) << 8 | cell
    PairRec pr[32];
    // output rings: unit 3 e + a of the OUTPUT (global edge e, component a) lives at 3 (e % MGW_RE) + a, so
    // that aligned 16-byte pieces of the rings are aligned pieces of vec / offset
    float vr[3 * MGW_RE];
    unsigned char br[3 * MGW_RE];
};

// Output state of a warp (the same on every lane).  A unit is one float of vec = one byte of offset:
// unit 3 e + a belongs to edge e.  Whole 16-byte pieces leave as STG.128; the ragged first piece of the
// warp's range, its last piece and the piece cut by the capacity leave as scalar stores.
struct OutCtx {
    long long u0;          // first unit of the warp's range
    long long vdone;       // vec units written as pieces so far (multiple of 4); head = [u0, vhead)
    long long bdone;       // offset units written as pieces so far (multiple of 16); head = [u0, bhead)
    long long vhead, bhead;
    long long cap3;        // 3 * capacity
    int vpos, bpos;        // vdone, bdone modulo the ring size
    bool vec16, off16;     // the arrays are 16-byte aligned (else: scalar stores only)
};

__device__ __forceinline__ void mgw_out_init(OutCtx &O, const FusedArgs &A, unsigned long long goff0) {
    O.u0 = 3 * (long long)goff0;
    O.vhead = O.vdone = (O.u0 + 3) & ~3ll;
    O.bhead = O.bdone = (O.u0 + 15) & ~15ll;
    O.vpos = (int)(O.vdone % (3 * MGW_RE));
    O.bpos = (int)(O.bdone % (3 * MGW_RE));
    O.cap3 = 3 * A.capacity;
    O.vec16 = (reinterpret_cast<unsigned long long>(A.vec) & 15ull) == 0ull;
    O.off16 = (reinterpret_cast<unsigned long long>(A.offset) & 15ull) == 0ull;
}

// Units [lo, hi) from the rings, one by one (rare paths).
__device__ __forceinline__ void mgw_out_scalar_v(const WSmem &ws, const FusedArgs &A, long long lo, long long hi, int lane) {
    for (long long u = lo + lane; u < hi; u += 32) A.vec[u] = ws.vr[(int)(u % (3 * MGW_RE))];
}
__device__ __forceinline__ void mgw_out_scalar_b(const WSmem &ws, const FusedArgs &A, long long lo, long long hi, int lane) {
    for (long long u = lo + lane; u < hi; u += 32) A.offset[u] = (int8_t)ws.br[(int)(u % (3 * MGW_RE))];
}

// The rings hold the units [lo, up) that were produced last: write out what is complete.
__device__ __forceinline__ void mgw_out_pieces(const WSmem &ws, const FusedArgs &A, OutCtx &O, long long lo, long long up,
                                               int lane) {
    const long long hi = up < O.cap3 ? up : O.cap3;
    if (O.vec16) {
        if (lo < O.vhead) mgw_out_scalar_v(ws, A, lo > O.u0 ? lo : O.u0, hi < O.vhead ? hi : O.vhead, lane);
        const long long npl = ((hi & ~3ll) - O.vdone) >> 2;                  // whole pieces (< 3 MGW_RE / 4)
        const int np = npl > 0 ? (int)npl : 0;
        float4 *dst = reinterpret_cast<float4 *>(A.vec + O.vdone);
        for (int k = lane; k < np; k += 32) {
            int pos = O.vpos + 4 * k;
            if (pos >= 3 * MGW_RE) pos -= 3 * MGW_RE;
            dst[k] = *reinterpret_cast<const float4 *>(&ws.vr[pos]);
        }
        if (np > 0) { O.vdone += 4ll * np; O.vpos = (O.vpos + 4 * np) % (3 * MGW_RE); }
        if (hi < up) { mgw_out_scalar_v(ws, A, O.vdone, hi, lane); O.vdone = 1ll << 60; }     // cut by the capacity
    } else {
        mgw_out_scalar_v(ws, A, lo, hi, lane);
    }
    if (O.off16) {
        if (lo < O.bhead) mgw_out_scalar_b(ws, A, lo > O.u0 ? lo : O.u0, hi < O.bhead ? hi : O.bhead, lane);
        const long long npl = ((hi & ~15ll) - O.bdone) >> 4;
        const int np = npl > 0 ? (int)npl : 0;
        uint4 *dst = reinterpret_cast<uint4 *>(A.offset + O.bdone);
        for (int k = lane; k < np; k += 32) {
            int pos = O.bpos + 16 * k;
            if (pos >= 3 * MGW_RE) pos -= 3 * MGW_RE;
            dst[k] = *reinterpret_cast<const uint4 *>(&ws.br[pos]);
        }
        if (np > 0) { O.bdone += 16ll * np; O.bpos = (O.bpos + 16 * np) % (3 * MGW_RE); }
        if (hi < up) { mgw_out_scalar_b(ws, A, O.bdone, hi, lane); O.bdone = 1ll << 60; }
    } else {
        mgw_out_scalar_b(ws, A, lo, hi, lane);
    }
}

// End of the warp's range (uend = its last unit + 1): the ragged last pieces.
__device__ __forceinline__ void mgw_out_finish(const WSmem &ws, const FusedArgs &A, const OutCtx &O, long long uend, int lane) {
    const long long hi = uend < O.cap3 ? uend : O.cap3;
    __syncwarp();
    if (O.vec16 && O.vdone < hi) mgw_out_scalar_v(ws, A, O.vdone, hi, lane);
    if (O.off16 && O.bdone < hi) mgw_out_scalar_b(ws, A, O.bdone, hi, lane);
}

struct FusedSmem {
    WSmem w[MGF_WARPS];
    unsigned wsum[MGF_WARPS];
    unsigned long long prefix;
    int last;
};

// Per-structure constants of a warp.
struct WCtx {
    float a[9];            // lattice rows
    float rho[3];
    int m0, m1, m2, mloc;
    float nr2, win, rc;
    const float *gx;       // positions of the structure's first atom
    const float *lat;
    int first, N;
};

__device__ __forceinline__ void mgw_ctx(WCtx &C, const FusedArgs &A, const CutRec *R, int s) {
    C.lat = A.lattice + 9 * (size_t)s;
#pragma unroll
    for (int c = 0; c < 9; ++c) C.a[c] = __ldg(C.lat + c);
#pragma unroll
    for (int a = 0; a < 3; ++a) C.rho[a] = R->rho[a];
    C.m0 = R->m & 0xFF; C.m1 = (R->m >> 8) & 0xFF; C.m2 = (R->m >> 16) & 0xFF;
    C.mloc = R->mloc;
    C.rc = A.r_c;
    C.nr2 = -__fmul_rn(A.r_c, A.r_c);
    // FP32 error bound of d2 - rc^2 near the threshold (R23)
    C.win = 1.1920929e-7f * (2.f * A.r_c * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * A.r_c * A.r_c);
    C.first = R->first;
    C.N = R->natoms;
    C.gx = A.pos + 3 * (size_t)R->first;
}

// ---- staging of one structure in the warp's shared memory ---------------------------------------
// Returns false (on every lane) if a coordinate is non-finite or too far from the cell.
template <bool EMIT>
__device__ __forceinline__ bool mgw_stage(WSmem &ws, const WCtx &C, int lane) {
    __syncwarp();
    bool ok = true;
    for (int j = lane; j < C.N; j += 32) {
        const float4 xw = mg_wrap_x(C.gx + 3 * j);
        ok = ok && __float_as_int(xw.w) != 0;
        ws.x[j] = xw;
    }
    // table of local translations t . L, t in [0, m): cells [0, mloc), then a far-away sentinel up to
    // a multiple of 32 and one group beyond (the filter reads one group ahead)
    const int M12 = C.m1 * C.m2;
    const float inv12 = 1.f / (float)M12, inv2 = 1.f / (float)C.m2;
    const int pad = min(MGW_TL + 4, ((C.mloc + 31) & ~31) + 4);
    for (int c = lane; c < pad; c += 32) {
        float Tx = 1e18f, Ty = 1e18f, Tz = 1e18f;
        if (c < C.mloc) {
            const int t0 = mg_fdiv(c, inv12), r = c - t0 * M12;
            const int t1 = mg_fdiv(r, inv2), t2 = r - t1 * C.m2;
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            Tx = __fmaf_rn(f2, C.a[6], __fmaf_rn(f1, C.a[3], __fmul_rn(f0, C.a[0])));
            Ty = __fmaf_rn(f2, C.a[7], __fmaf_rn(f1, C.a[4], __fmul_rn(f0, C.a[1])));
            Tz = __fmaf_rn(f2, C.a[8], __fmaf_rn(f1, C.a[5], __fmul_rn(f0, C.a[2])));
            const unsigned tcode = ((unsigned)t0 << 24) | ((unsigned)t1 << 16) | ((unsigned)t2 << 8);
            ws.tcode[c] = tcode;
            if (EMIT) {                // exact: small integers times FP32 values, three terms
                const double g0 = (double)t0, g1 = (double)t1, g2 = (double)t2;
                CellRec r;
                r.tx = fma(g2, (double)C.a[6], fma(g1, (double)C.a[3], g0 * (double)C.a[0]));
                r.ty = fma(g2, (double)C.a[7], fma(g1, (double)C.a[4], g0 * (double)C.a[1]));
                r.tz = fma(g2, (double)C.a[8], fma(g1, (double)C.a[5], g0 * (double)C.a[2]));
                r.tcode = tcode; r.pad = 0u;
                ws.cr[c] = r;
            }
        }
        ws.T[0][c] = Tx; ws.T[1][c] = Ty; ws.T[2][c] = Tz;
    }
    ok = __all_sync(0xFFFFFFFFu, ok);
    __syncwarp();
    return ok;
}

// One lane's ordered pair (i, j) of the staged structure: q' = (u + lo) . L with u = x_j - x_i
// (wrapped coordinates) and lo = floor(-rho - u) + 1 the first cell of the pair's sub-box
// (cut_prep.cuh); the cell offsets relative to the coordinates AS GIVEN start at l = lo + k_i - k_j.
struct WPair {
    float qx, qy, qz;
    int l0, l1, l2;
    int self;              // index of the cell tau = 0 in the table if i == j, else -1
    bool ok;               // valid lane, offsets inside int8
};

__device__ __forceinline__ WPair mgw_pair(const WSmem &ws, const WCtx &C, bool valid, int i, int j) {
    WPair p;
    const float4 xi = ws.x[i], xj = ws.x[j];
    const float u0 = __fsub_rn(xj.x, xi.x), u1 = __fsub_rn(xj.y, xi.y), u2 = __fsub_rn(xj.z, xi.z);
    const float e0 = floorf(__fsub_rn(-C.rho[0], u0)) + 1.f, e1 = floorf(__fsub_rn(-C.rho[1], u1)) + 1.f,
                e2 = floorf(__fsub_rn(-C.rho[2], u2)) + 1.f;
    const float f0 = __fadd_rn(u0, e0), f1 = __fadd_rn(u1, e1), f2 = __fadd_rn(u2, e2);
    p.qx = __fmaf_rn(f2, C.a[6], __fmaf_rn(f1, C.a[3], __fmul_rn(f0, C.a[0])));
    p.qy = __fmaf_rn(f2, C.a[7], __fmaf_rn(f1, C.a[4], __fmul_rn(f0, C.a[1])));
    p.qz = __fmaf_rn(f2, C.a[8], __fmaf_rn(f1, C.a[5], __fmul_rn(f0, C.a[2])));
    const int ki = __float_as_int(xi.w), kj = __float_as_int(xj.w);
    p.l0 = (int)e0 + (ki & 1023) - (kj & 1023);
    p.l1 = (int)e1 + ((ki >> 10) & 1023) - ((kj >> 10) & 1023);
    p.l2 = (int)e2 + ((ki >> 20) & 1023) - ((kj >> 20) & 1023);
    p.ok = valid && p.l0 >= -127 && p.l1 >= -127 && p.l2 >= -127 && p.l0 + C.m0 <= 128 && p.l1 + C.m1 <= 128 &&
           p.l2 + C.m2 <= 128;
    if (!p.ok) { p.qx = 1e18f; p.qy = 1e18f; p.qz = 1e18f; }
    p.self = i == j ? (-(int)e0 * C.m1 - (int)e1) * C.m2 - (int)e2 : -1;   // (i,i,0) is not an edge (R3)
    return p;
}

// Hit mask of cells [32 w, 32 w + 32) of the pair's sub-box: bit 31 - c <-> cell 32 w + c (the sign
// bits of y = |q' + T|^2 - r_c^2 are shifted in one by one).  Two cells per packed FP32 instruction,
// table groups read one ahead.  A lane that saw |y| < win decides those cells again with the exact
// FP64 predicate, so the mask is Def. 3's in FP64.
__device__ __forceinline__ unsigned mgw_word_mask(const WSmem &ws, const WCtx &C, const WPair &p, int i, int j, int w) {
    const int nw = min(32, C.mloc - 32 * w), n4 = (nw + 3) >> 2;      // warp-uniform
    const float4 *Xp = reinterpret_cast<const float4 *>(&ws.T[0][32 * w]);
    const float4 *Yp = reinterpret_cast<const float4 *>(&ws.T[1][32 * w]);
    const float4 *Zp = reinterpret_cast<const float4 *>(&ws.T[2][32 * w]);
    const float2 qx = make_float2(p.qx, p.qx), qy = make_float2(p.qy, p.qy), qz = make_float2(p.qz, p.qz);
    const float2 nr2 = make_float2(C.nr2, C.nr2);
    const float win = C.win;
    unsigned mask = 0u;
    bool near = false;
    const int n4r = (n4 + 1) & ~1;                // two groups per trip; a group past the word's cells holds sentinels
#pragma unroll 1
    for (int g = 0; g < n4r; g += 2) {
        const float4 X0 = Xp[g], Y0 = Yp[g], Z0 = Zp[g], X1 = Xp[g + 1], Y1 = Yp[g + 1], Z1 = Zp[g + 1];
        float y[8];
        mg_filter4(X0, Y0, Z0, qx, qy, qz, nr2, *reinterpret_cast<float (*)[4]>(&y[0]));
        mg_filter4(X1, Y1, Z1, qx, qy, qz, nr2, *reinterpret_cast<float (*)[4]>(&y[4]));
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            mask = __funnelshift_l(__float_as_uint(y[c]), mask, 1);    // (mask << 1) | sign(y)
            near = near || fabsf(y[c]) < win;
        }
    }
    mask = n4r < 8 ? mask << (32 - 4 * n4r) : mask;
    if (near) {                                   // rare: decide the window cells in FP64
        const float *xi = C.gx + 3 * i, *xj = C.gx + 3 * j;
        for (int c = 0; c < nw; ++c) {
            const float Tx = ws.T[0][32 * w + c], Ty = ws.T[1][32 * w + c], Tz = ws.T[2][32 * w + c];
            const float vx = __fadd_rn(p.qx, Tx), vy = __fadd_rn(p.qy, Ty), vz = __fadd_rn(p.qz, Tz);
            const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, C.nr2)));
            if (fabsf(y) < win) {
                const unsigned tc = ws.tcode[32 * w + c];
                double v[3];
                const double d = mg_exact_vec(xi, xj, p.l0 + (int)(tc >> 24), p.l1 + (int)((tc >> 16) & 0xFFu),
                                              p.l2 + (int)((tc >> 8) & 0xFFu), C.lat, v);
                const unsigned bit = 0x80000000u >> c;
                mask = d < (double)C.rc ? (mask | bit) : (mask & ~bit);
            }
        }
    }
    const int cs = p.self - 32 * w;               // (i, i, 0) is not an edge
    if (p.self >= 0 && cs >= 0 && cs < 32) mask &= ~(0x80000000u >> cs);
    return mask;
}

// ---- generic rows: any structure size, any sub-box (not tuned) -----------------------------------
// One warp per source row, lanes over candidates (j, t) of the row.  For the pair (i, j): u = x_j - x_i
// (wrapped coordinates), the sub-box starts at lo_a = floor(-rho_a - u_a) + 1 (cut_prep.cuh);
// d2 = |(u + lo + t) . L|^2 in FP32, FP64 decision inside the rounding window (R23).
// Candidate (j, t) of row i: hit?  tau (relative to the coordinates as given) in tau[3].
__device__ __forceinline__ bool mgw_cand(const WCtx &C, const float4 xi, int i, int j, int t0, int t1, int t2,
                                         int tau[3], bool &bad) {
    const float4 xj = mg_wrap_x(C.gx + 3 * j);
    const int ki = __float_as_int(xi.w), kj = __float_as_int(xj.w);
    const float u0 = __fsub_rn(xj.x, xi.x), u1 = __fsub_rn(xj.y, xi.y), u2 = __fsub_rn(xj.z, xi.z);
    const float e0 = floorf(__fsub_rn(-C.rho[0], u0)) + 1.f, e1 = floorf(__fsub_rn(-C.rho[1], u1)) + 1.f,
                e2 = floorf(__fsub_rn(-C.rho[2], u2)) + 1.f;
    const float f0 = __fadd_rn(u0, e0 + (float)t0), f1 = __fadd_rn(u1, e1 + (float)t1), f2 = __fadd_rn(u2, e2 + (float)t2);
    const float vx = __fmaf_rn(f2, C.a[6], __fmaf_rn(f1, C.a[3], __fmul_rn(f0, C.a[0])));
    const float vy = __fmaf_rn(f2, C.a[7], __fmaf_rn(f1, C.a[4], __fmul_rn(f0, C.a[1])));
    const float vz = __fmaf_rn(f2, C.a[8], __fmaf_rn(f1, C.a[5], __fmul_rn(f0, C.a[2])));
    const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, C.nr2)));
    tau[0] = (int)e0 + t0 + (ki & 1023) - (kj & 1023);
    tau[1] = (int)e1 + t1 + ((ki >> 10) & 1023) - ((kj >> 10) & 1023);
    tau[2] = (int)e2 + t2 + ((ki >> 20) & 1023) - ((kj >> 20) & 1023);
    bad = ki == 0 || kj == 0 || tau[0] < -127 || tau[1] < -127 || tau[2] < -127 || tau[0] > 127 || tau[1] > 127 || tau[2] > 127;
    if (bad) return false;
    if (i == j && (tau[0] | tau[1] | tau[2]) == 0) return false;    // (i, i, 0) is not an edge (R3)
    bool hit = y < 0.f;
    if (fabsf(y) < C.win) {                                          // FP32 cannot decide: Def. 3 in FP64
        double v[3];
        hit = mg_exact_vec(C.gx + 3 * i, C.gx + 3 * j, tau[0], tau[1], tau[2], C.lat, v) < (double)C.rc;
    }
    return hit;
}

__device__ __forceinline__ void mgw_emit_one(const FusedArgs &A, long long e, int gi, int gj, const float *gx, int i,
                                             int j, const int t[3], const float *lat) {
    if (e >= A.capacity) return;
    double v[3];
    const double d = mg_exact_vec(gx + 3 * i, gx + 3 * j, t[0], t[1], t[2], lat, v);
    A.src[e] = gi;
    A.dst[e] = gj;
    A.offset[3 * e] = (int8_t)t[0]; A.offset[3 * e + 1] = (int8_t)t[1]; A.offset[3 * e + 2] = (int8_t)t[2];
    A.vec[3 * e] = (float)v[0]; A.vec[3 * e + 1] = (float)v[1]; A.vec[3 * e + 2] = (float)v[2];
    if (A.dist) A.dist[e] = (float)d;
}

// One source row: returns its edges; EMIT: writes them from goff on (any order inside the row).
// Tables of 32 cells and more: lane <-> cell (decoded once per 32 cells), loop over the targets j.
// Smaller tables: lane <-> (target, cell), floor(32 / mloc) targets per pass.
template <bool EMIT>
__device__ __forceinline__ unsigned mgw_row(const FusedArgs &A, const WCtx &C, int i, unsigned long long goff, int lane,
                                            bool &anybad) {
    const float4 xi = mg_wrap_x(C.gx + 3 * i);
    const int M12 = C.m1 * C.m2;
    unsigned cnt = 0u;
    const bool wide = C.mloc >= 32;
    const int J = wide ? 1 : 32 / C.mloc;                  // targets per pass
    const int jl = wide ? 0 : lane / C.mloc;
    const int npass = wide ? (C.mloc + 31) >> 5 : 1;
    for (int ps = 0; ps < npass; ++ps) {
        const int c = wide ? 32 * ps + lane : lane - jl * C.mloc;
        const bool cv = wide ? c < C.mloc : jl < J;
        const int t0 = c / M12, r = c - t0 * M12, t1 = r / C.m2, t2 = r - t1 * C.m2;
        for (int j0 = 0; j0 < C.N; j0 += J) {
            const int j = j0 + jl;
            int tau[3] = {0, 0, 0};
            bool bad = false;
            const bool hit = cv && j < C.N && mgw_cand(C, xi, i, j, t0, t1, t2, tau, bad);
            anybad = anybad || bad;
            const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
            if (EMIT && hit)
                mgw_emit_one(A, (long long)(goff + cnt) + __popc(bal & ((1u << lane) - 1u)), C.first + i, C.first + j, C.gx, i, j, tau, C.lat);
            cnt += __popc(bal);
        }
    }
    return cnt;
}

// Rows [ia, ib) of structure s, counted by one warp; row totals go to the scratch while they fit.
__device__ __forceinline__ unsigned mgw_rows_count(const FusedArgs &A, const WCtx &C, int ia, int ib, unsigned *wm,
                                                   int midx, int lane) {
    unsigned total = 0u;
    for (int i = ia; i < ib; ++i) {
        bool anybad = false;
        const unsigned cnt = mgw_row<false>(A, C, i, 0ull, lane, anybad);
        if (anybad) atomicOr(A.status, __float_as_int(mg_wrap_x(C.gx + 3 * i).w) == 0 ? MGS_NONFINITE : MGS_OFFSET);
        total += cnt;
    }
    return total;
}

// Emit rows [ia, ib) from goff; returns the offset after them.
__device__ __forceinline__ unsigned long long mgw_rows_emit(const FusedArgs &A, const WCtx &C, int ia, int ib,
                                                            unsigned long long goff, int lane) {
    for (int i = ia; i < ib; ++i) {
        if (lane == 0) A.row_ptr[C.first + i] = (int)goff;
        bool anybad = false;
        goff += mgw_row<true>(A, C, i, goff, lane, anybad);
    }
    return goff;
}

// ---- stash -> global ------------------------------------------------------------------------------
// Edges [0, n) of the warp's stash are the edges [goff, goff + n) of the output.  Batches of MGW_BATCH
// edges: lane <-> edge, src / dst / dist as coalesced 4-byte stores, vec and offset into the output
// rings; after every batch the complete 16-byte pieces of the rings are written out.
__device__ __forceinline__ void mgw_flush(WSmem &ws, const FusedArgs &A, OutCtx &O, int first, long long goff, int n,
                                          int lane) {
    for (int e0 = 0; e0 < n; e0 += MGW_BATCH) {
        const int nb = min(MGW_BATCH, n - e0);
        const long long E0 = goff + e0;                 // global index of the batch's first edge
        const long long room = A.capacity - E0;
        const int nst = room >= nb ? nb : (room > 0 ? (int)room : 0);       // edges that fit src / dst / dist
        int32_t *psrc = A.src + E0, *pdst = A.dst + E0;
        float *pdist = A.dist ? A.dist + E0 : nullptr;
        const int em = (int)(E0 & (MGW_RE - 1));
#pragma unroll 1
        for (int x = lane; x < nb; x += 32) {
            const unsigned code = ws.stash[e0 + x];
            const PairRec P = ws.pr[code >> 8];
            const CellRec Q = ws.cr[code & 0xFFu];
            const double v0 = P.bx + Q.tx, v1 = P.by + Q.ty, v2 = P.bz + Q.tz;
            const unsigned tb = (P.plc + Q.tcode) ^ 0x80808000u;             // tau bytes as int8
            if (x < nst) {
                psrc[x] = first + (int)(P.pij & 0xFFFFu);
                pdst[x] = first + (int)(P.pij >> 16);
                if (pdist) pdist[x] = __fsqrt_rn((float)fma(v2, v2, fma(v1, v1, v0 * v0)));
            }
            const int u = 3 * ((em + x) & (MGW_RE - 1));
            ws.vr[u] = (float)v0; ws.vr[u + 1] = (float)v1; ws.vr[u + 2] = (float)v2;
            ws.br[u] = (unsigned char)(tb >> 24); ws.br[u + 1] = (unsigned char)(tb >> 16); ws.br[u + 2] = (unsigned char)(tb >> 8);
        }
        __syncwarp();
        mgw_out_pieces(ws, A, O, 3 * E0, 3 * (E0 + nb), lane);
        __syncwarp();
    }
}

// ---- the walk of a warp over its rows -------------------------------------------------------------
// PHASE 0: count (returns the warp's edges, the same value on every lane); PHASE 1: emit from goff.
template <int PHASE>
__device__ __forceinline__ unsigned long long mgw_walk(WSmem &ws, const FusedArgs &A, const RangeCtx &RC, int rid,
                                                       unsigned *wm, unsigned long long goff, int lane) {
    OutCtx O;
    if (PHASE == 1) mgw_out_init(O, A, goff);
    unsigned long long c0, c1;
    mg_warp_range(RC, rid, c0, c1);
    int s, qa;
    mg_range_start(RC, c0, s, qa, lane);
    int midx = 0;
    unsigned total = 0u, lane_total = 0u;          // warp-uniform part (rows path), per-lane part (pair-lane path)
#ifdef MG_PHASE_CLOCKS
    const long long wt0 = clock64();
    const int dbg_s0 = s;
    int dbg_seg = 0, dbg_blk = 0, dbg_rows = 0;
#endif
    for (; s < A.n_struct; ++s, qa = 0) {
        const CutRec *R = A.rec + s;
        int qb;
        if (!mg_segment(RC, R, s, qa, c1, qb)) break;
        const int N = R->natoms;
        const bool more = qb >= N * N;
        // source rows whose first pair lies in [qa, qb)
        const int ia = N ? (qa + N - 1) / N : 0, ib = N ? (qb + N - 1) / N : 0;
        if (ib > ia) {
            const int mloc = R->mloc;
            if (mloc <= 0) {                       // invalid structure: empty rows
                if (PHASE == 1)
                    for (int i = ia + lane; i < ib; i += 32) A.row_ptr[R->first + i] = (int)goff;
            } else if (N > MGW_NMAX || mloc > MGW_TL) {
                WCtx C;
                mgw_ctx(C, A, R, s);
                if (PHASE == 0) total += mgw_rows_count(A, C, ia, ib, wm, midx, lane);
                else {                             // these rows bypass the output rings
                    mgw_out_finish(ws, A, O, 3 * (long long)goff, lane);
                    goff = mgw_rows_emit(A, C, ia, ib, goff, lane);
                    mgw_out_init(O, A, goff);
                }
                #ifdef MG_PHASE_CLOCKS
                dbg_rows += ib - ia; dbg_seg += 1;
#endif
            } else {
                WCtx C;
                mgw_ctx(C, A, R, s);
                const bool live = mgw_stage<PHASE == 1>(ws, C, lane);
                const int nW = (mloc + 31) >> 5, recw = 32 * nW;
                const int q0 = ia * N, q1 = ib * N, nblk = (q1 - q0 + 31) >> 5;
                const float inv_N = 1.f / (float)N;
                if (!live) {
                    if (lane == 0) atomicOr(A.status, MGS_NONFINITE);
                    if (PHASE == 1)
                        for (int i = ia + lane; i < ib; i += 32) A.row_ptr[C.first + i] = (int)goff;
                } else {
#pragma unroll 1
                    for (int b = 0; b < nblk; ++b) {
                        const int q = q0 + 32 * b + lane;
                        const bool valid = q < q1;
                        int i = 0, j = 0;
                        if (valid) { i = mg_fdiv(q, inv_N); j = q - i * N; }
                        const WPair p = mgw_pair(ws, C, valid, i, j);
                        const int base = midx + b * recw;
                        const bool have = base + recw <= A.mask_words;
                        unsigned *mp = wm + base + lane;
                        if (PHASE == 0) {
                            if (valid && !p.ok) atomicOr(A.status, MGS_OFFSET);
                            unsigned cnt = 0u;
#pragma unroll 1
                            for (int w = 0; w < nW; ++w) {
                                const unsigned m = mgw_word_mask(ws, C, p, i, j, w);
                                cnt += __popc(m);
                                if (have) mp[32 * w] = m;
                            }
                            lane_total += cnt;         // reduced over the lanes at the end
                        } else {
                            unsigned cnt = 0u;
#pragma unroll 1
                            for (int w = 0; w < nW; ++w)
                                cnt += __popc(have ? __ldcg(mp + 32 * w) : mgw_word_mask(ws, C, p, i, j, w));
                            unsigned incl = cnt;
#pragma unroll
                            for (int o = 1; o < 32; o <<= 1) {
                                const unsigned v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                                if (lane >= o) incl += v;
                            }
                            const unsigned tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
                            if (valid && j == 0) A.row_ptr[C.first + i] = (int)(goff + incl - cnt);
                            if (tot == 0u) continue;
                            // the pair's part of vec: (x_j - x_i + l) . L in FP64, coordinates as given
                            if (valid) {
                                const float *xi = C.gx + 3 * i, *xj = C.gx + 3 * j;
                                const double f0 = ((double)xj[0] - (double)xi[0]) + (double)p.l0;
                                const double f1 = ((double)xj[1] - (double)xi[1]) + (double)p.l1;
                                const double f2 = ((double)xj[2] - (double)xi[2]) + (double)p.l2;
                                PairRec P;
                                P.bx = fma(f2, (double)C.a[6], fma(f1, (double)C.a[3], f0 * (double)C.a[0]));
                                P.by = fma(f2, (double)C.a[7], fma(f1, (double)C.a[4], f0 * (double)C.a[1]));
                                P.bz = fma(f2, (double)C.a[8], fma(f1, (double)C.a[5], f0 * (double)C.a[2]));
                                P.plc = ((unsigned)(p.l0 + 128) << 24) | ((unsigned)(p.l1 + 128) << 16) |
                                        ((unsigned)(p.l2 + 128) << 8);
                                P.pij = (unsigned)i | ((unsigned)j << 16);
                                ws.pr[lane] = P;
                            }
                            // passes of consecutive lanes whose hits fit the stash (nearly always one)
                            unsigned done = 0u;
                            int l0 = 0;
                            while (done < tot) {
                                const bool mine = lane >= l0 && incl - done <= MGW_STASH;
                                const int nl = __popc(__ballot_sync(0xFFFFFFFFu, mine));   // >= 1: a lane has <= MGW_TL hits
                                const unsigned t = __shfl_sync(0xFFFFFFFFu, incl, l0 + nl - 1) - done;
                                if (mine) {
                                    unsigned pos = incl - cnt - done;
                                    const unsigned pc = (unsigned)lane << 8;
#pragma unroll 1
                                    for (int w = 0; w < nW; ++w) {
                                        unsigned mk = have ? __ldcg(mp + 32 * w) : mgw_word_mask(ws, C, p, i, j, w);
                                        while (mk) {
                                            const int bit = __clz(mk);
                                            mk &= ~(0x80000000u >> bit);
                                            ws.stash[pos++] = pc | (unsigned)(32 * w + bit);
                                        }
                                    }
                                }
                                __syncwarp();
                                mgw_flush(ws, A, O, C.first, (long long)goff, (int)t, lane);
                                goff += t;
                                done += t;
                                l0 += nl;
                            }
                        }
                    }
                }
                midx += nblk * recw;
#ifdef MG_PHASE_CLOCKS
                dbg_blk += nblk; dbg_seg += 1;
#endif
            }
        }
        if (!more) break;
    }
#ifdef MG_PHASE_CLOCKS
    if (lane == 0 && A.dbg) {
        unsigned *d = A.dbg + 4 * 2048 + 16 * rid + 8 * PHASE;
        d[0] = (unsigned)(clock64() - wt0); d[1] = dbg_s0; d[2] = dbg_seg; d[3] = dbg_blk; d[4] = dbg_rows; d[5] = midx;
    }
#endif
    if (PHASE == 1) mgw_out_finish(ws, A, O, 3 * (long long)goff, lane);
    if (PHASE == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) lane_total += __shfl_xor_sync(0xFFFFFFFFu, lane_total, o);
        goff = (unsigned long long)(total + lane_total);
    }
    return goff;
}

// ---- the kernel -------------------------------------------------------------------------------------
#ifndef MGF_MIN_CTAS
#define MGF_MIN_CTAS 5
#endif
__global__ void __launch_bounds__(MGF_BLOCK, MGF_MIN_CTAS)
mg_cutoff_fused_kernel(const __grid_constant__ FusedArgs A) {
    mg_grid_dependency_wait();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FusedSmem &sm = *reinterpret_cast<FusedSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    WSmem &ws = sm.w[warp];
    const unsigned epoch = *reinterpret_cast<volatile unsigned *>(A.ctl + 10) + 1u;   // tag of this call's slots
    RangeCtx RC;
    mg_range_init(RC, A.rec, A.bpre, A.n_blocks, A.n_struct, (int)gridDim.x * MGF_WARPS, lane);
    const int rid = (int)blockIdx.x * MGF_WARPS + warp;
    unsigned *wm = A.wmask + (size_t)rid * MGW_MASK_WORDS;
    MGF_STAMP(0)
    const unsigned long long wtotal = mgw_walk<0>(ws, A, RC, rid, wm, 0ull, lane);
    if (lane == 0) sm.wsum[warp] = (unsigned)wtotal;
    __syncthreads();
    MGF_STAMP(1)
    unsigned long long total = 0ull, mine = 0ull;
#pragma unroll
    for (int w = 0; w < MGF_WARPS; ++w) {
        if (w < warp) mine += sm.wsum[w];
        total += sm.wsum[w];
    }
    if (tid == 0) mg_st_release(A.slots + blockIdx.x, ((unsigned long long)epoch << 32) | (total & 0xFFFFFFFFull));
    if (!A.count_only) {
        // device-wide exclusive scan of K4: sum of the slots before this CTA's (all CTAs are resident)
        if (warp == 0) {
            unsigned long long before = 0ull;
            for (int c0 = 0; c0 < (int)blockIdx.x; c0 += 32) {
                const int c = c0 + lane;
                if (c < (int)blockIdx.x) {
                    unsigned long long v;
                    while ((unsigned)((v = mg_ld_acquire(A.slots + c)) >> 32) != epoch) __nanosleep(400);
                    before += v & 0xFFFFFFFFull;
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) before += __shfl_xor_sync(0xFFFFFFFFu, before, o);
            if (lane == 0) sm.prefix = before;
        }
        __syncthreads();
        const unsigned long long before = sm.prefix;
        MGF_STAMP(2)
        if (blockIdx.x == gridDim.x - 1 && tid == 0) {           // the last range knows the grand total
            const unsigned long long tot = before + total;
            *A.n_edges = (long long)tot;
            A.row_ptr[A.n_atoms] = (int)tot;
            if (tot > 0x7FFFFFFFull || (long long)tot > A.capacity) atomicOr(A.status, MGS_CAPACITY);
        }
        mgw_walk<1>(ws, A, RC, rid, wm, before + mine, lane);
        MGF_STAMP(3)
    }
    // last CTA out: the call is over (count_only: it also adds the totals up)
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        sm.last = atomicAdd(A.ctl + 11, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!sm.last) return;
    if (A.count_only && warp == 0) {
        unsigned long long sum = 0ull;
        for (int c = lane; c < (int)gridDim.x; c += 32) {
            unsigned long long v;
            do { v = mg_ld_acquire(A.slots + c); } while ((unsigned)(v >> 32) != epoch);
            sum += v & 0xFFFFFFFFull;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xFFFFFFFFu, sum, o);
        if (lane == 0) {
            *A.n_edges = (long long)sum;
            if (sum > 0x7FFFFFFFull) atomicOr(A.status, MGS_CAPACITY);
        }
    }
    if (tid == 0) {
        A.ctl[11] = 0u;
        __threadfence();
        *reinterpret_cast<volatile unsigned *>(A.ctl + 10) = epoch;
    }
}
