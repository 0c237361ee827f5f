// cut_scan.cuh — cutoff graph (K3 distance filter, K4 count -> device-wide scan -> emit, K6 batching,
// SURVEY.md 8(a)) in ONE cooperative launch; DESIGN.md 5.7.
//
//   mg_cutoff_scan_kernel.  Co-resident CTAs whose warps work on their own: warp r of the grid (r = 4 *
//     blockIdx.x + warp) owns the source rows whose first pair lies in the r-th of n_ranges equally expensive,
//     contiguous ranges of the batch's ordered pairs in (structure, i, j) order — the CSR order of the
//     output (cut_prep.cuh).
//       find    per structure: wrapped positions and the table of local translations staged in the warp's
//               shared memory; blocks of 32 ordered pairs, lane <-> pair: FP32 filter over the pair's sub-box
//               (FP64 decision inside the rounding window, R23), 32-bit hit masks in shared memory,
//               hits compacted in (row, j, t) order into 8-byte codes (dst, tau) that go to chunks of a pool
//               (the warp does not know yet where its edges start); row_ptr local to the warp;
//       scan    warp totals -> CTA total, published in a slot tagged with the call's epoch; warp 0 sums
//               the slots of the CTAs before its own (all CTAs are resident: cooperative launch): the
//               device-wide exclusive scan of K4 without a launch of its own;
//       write   the warp turns its codes into the caller's arrays: lane <-> four consecutive edges, src
//               from row_ptr, vec = ((x_dst - x_src) + tau) . L in FP64 in the oracle's operation order,
//               rounded once (R24); every array leaves in aligned 16-byte stores.
//     A warp whose codes did not fit the pool walks its rows a second time and writes edge by edge.
//   mg_cutoff_write_kernel (MATGRAPH_WRITE_KERNEL=1, an A/B variant): the write phase as a launch of its
//     own over one code stream, a warp per slice of 128 consecutive edges.
//
// Structures the pair-lane path does not take (more than MGS_NMAX atoms, a sub-box of more than MGS_TL
// cells) go row by row, lanes over the candidates of one source row: through the cell list of
// cut_bins.cuh when the sub-box is one cell (mgs_row_binned), else over all (j, t) (mgs_row).
#pragma once
#include "common.cuh"
#include "cut_prep.cuh"
#include "cut_bins.cuh"
#include "ranges.cuh"

#define MGS_BLOCK 128
#define MGS_WARPS (MGS_BLOCK / 32)
#define MGS_TL MG_PAIR_TL          // cells of a warp's table
#define MGS_NMAX MG_SMALL_MAX_ATOMS // atoms of a staged structure
#define MGS_STASH 256              // codes per pass
#define MGS_CHUNK 512              // codes per chunk of the pool
#define MGS_MAXCH 64               // chunks a range can hold (beyond: its rows are listed again in the second phase)
#ifndef MGS_WAVES
#define MGS_WAVES 1
#endif
//                // ranges per warp: wave w of the grid holds the ranges w * n_warps .. (w + 1) * n_warps - 1
#define MGS_SLICE 128              // edges per slice of the write kernel

struct ScanArgs {
    const float *pos;
    const float *lattice;
    const float4 *xw4;             // [n_atoms] wrapped coordinates + packed integer parts (cut_prep.cuh)
    const float4 *xs4;             // [n_atoms] ... in bin order, .w = atom index and integer parts (cut_bins.cuh)
    const int *bin_start;          // [n_atoms + 2 n_struct + 2] ... first entry of each bin
    int n_struct, n_atoms;
    const float *radii;            // [n_atoms] or NULL: cutoff of every SOURCE atom (Def. 3's c_i); NULL: the
                                   // same cutoff for all (the structure's radius in its CutRec)
    int32_t *row_ptr;
    long long capacity;
    long long *n_edges;
    const CutRec *rec;
    const unsigned long long *bpre;
    int n_blocks;
    uint2 *pool;                   // [n_pool, MGS_CHUNK] codes of the warps before their final place is known
    int n_pool;                    // chunks of the pool (tests: less)
    unsigned long long *slots;     // [MGS_WAVES, gridDim.x] epoch << 32 | edges of the CTA's ranges of a wave
    unsigned *ctl;                 // [10] epoch of the last finished call, [11] CTAs done, [12] pool chunks taken
    unsigned *status;
    int count_only;
    // the caller's edge arrays: written by this kernel itself when write_here
    int32_t *src, *dst;
    int8_t *offset;
    float *vec, *dist;
    int write_here;
    // products for the write kernel (write_here == 0)
    uint2 *codes;                  // [capacity] .x = dst, .y = (tau + 128) bytes << 8
    int4 *slice_row;               // [ceil(capacity / MGS_SLICE) + 1] for edge MGS_SLICE * k: its row, first atom and
                                   // end of the atoms of the row's structure, the structure
    int32_t *atom_struct;          // [n_atoms]
    double *pos64;                 // [n_atoms, 4] FP64 copies of the positions, one 32-byte sector per atom
    double *lat64;                 // [n_struct, 9]
    unsigned *dbg;                 // MG_PHASE_CLOCKS builds: globaltimer at the phase boundaries, per-warp cycles
};

#ifdef MG_PHASE_CLOCKS
__device__ __forceinline__ unsigned mgs_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return (unsigned)t;
}
#define MGS_STAMP(i) if (threadIdx.x == 0 && A.dbg) A.dbg[4 * blockIdx.x + (i)] = mgs_now();
#else
#define MGS_STAMP(i)
#endif

struct SSmem {                         // one warp's shared memory
    float T[3][MGS_TL + 4];            // t . L: planes x | y | z (+ one group read ahead)
    unsigned tcode[MGS_TL];            // t0 << 24 | t1 << 16 | t2 << 8
    float4 x[MGS_NMAX];                // wrapped fractional coordinates, .w = packed integer parts
    uint2 stash[MGS_STASH];            // codes of one pass
    unsigned mk[MGS_TL / 32][32];      // hit masks of the current block
    int chunks[MGS_WAVES][MGS_MAXCH];  // the chunks of the pool that hold the codes of the warp's ranges
    int wave[MGS_WAVES][8];            // per range: edges, chunks, pool ok, first row, end of rows, edges of the warps before (2 words)
    unsigned long long bar[2];         // mbarriers of the two candidate buffers (binned rows: TMA bulk copies)
    unsigned bphase;                   // ... their phase bits
};

// The candidate buffers of the binned rows: the staging area of the pair-lane path (T | tcode | x is one
// contiguous, 16-byte aligned piece of the warp's shared memory), two buffers of MGS_CH entries.
#define MGS_CH 192
static_assert(2 * MGS_CH * sizeof(float4) <= sizeof(float) * 3 * (MGS_TL + 4) + sizeof(unsigned) * MGS_TL + sizeof(float4) * MGS_NMAX,
              "two candidate buffers fit the staging area");
static_assert((sizeof(float) * 3 * (MGS_TL + 4)) % 16 == 0 && (sizeof(unsigned) * MGS_TL) % 16 == 0, "staging area is contiguous");

// ---- TMA bulk copies (global -> the warp's shared memory) that complete on an mbarrier
__device__ __forceinline__ unsigned mgs_saddr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mgs_bar_init(unsigned long long *bar) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(mgs_saddr(bar)) : "memory");
}
__device__ __forceinline__ void mgs_bar_expect(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(mgs_saddr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mgs_bar_wait(unsigned long long *bar, unsigned phase) {
    unsigned done = 0u;
    const unsigned a = mgs_saddr(bar);
    while (!done)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.b32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(a), "r"(phase) : "memory");
}
__device__ __forceinline__ void mgs_bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(mgs_saddr(dst)), "l"(src), "r"(bytes), "r"(mgs_saddr(bar)) : "memory");
}
// (generic-proxy accesses to shared memory before, async-proxy accesses after)
__device__ __forceinline__ void mgs_fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

struct ScanSmem {
    SSmem w[MGS_WARPS];
    unsigned wsum[MGS_WARPS];
    int wok[MGS_WARPS];
    unsigned long long prefix, wave_all;
    int last;
};

// Per-structure constants of a warp.
struct WCtx {
    float a[9];            // lattice rows
    float rho[3];
    int m0, m1, m2, mloc;
    float nr2, win, rc;
    const float *gx;       // positions of the structure's first atom
    const float4 *xw;      // ... and their wrapped copies
    const float *cr;       // ... and their cutoffs (NULL: rc for all)
    const float *lat;
    int first, N;
    int nb0, nb1, nb2;     // cell list (cut_bins.cuh): slabs per axis; nb0 == 0: none
    const float4 *xs;      // ... entries in bin order
    const int *bs;         // ... first entry of each bin
};

template <bool BINNED>
__device__ __forceinline__ void mgs_ctx(WCtx &C, const ScanArgs &A, const CutRec *R, int s) {
    C.lat = A.lattice + 9 * (size_t)s;
#pragma unroll
    for (int c = 0; c < 9; ++c) C.a[c] = __ldg(C.lat + c);
#pragma unroll
    for (int a = 0; a < 3; ++a) C.rho[a] = R->rho[a];
    C.m0 = R->m & 0xFF; C.m1 = (R->m >> 8) & 0xFF; C.m2 = (R->m >> 16) & 0xFF;
    C.mloc = R->mloc;
    // (with per-atom cutoffs the structure's radius is the largest of them: bounds and the rounding window hold
    // for every source, the threshold itself is the source's)
    const float rc = R->radius;
    C.rc = rc;
    C.nr2 = -__fmul_rn(rc, rc);
    // FP32 error bound of d2 - rc^2 near the threshold (R23)
    C.win = 1.1920929e-7f * (2.f * rc * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * rc * rc);
    C.first = R->first;
    C.N = R->natoms;
    C.gx = A.pos + 3 * (size_t)R->first;
    C.xw = A.xw4 + R->first;
    C.cr = A.radii ? A.radii + R->first : nullptr;
    const int bins = BINNED ? R->bins : 0;      // (the instance without cell lists: every large structure by the generic rows)
    C.nb0 = bins >> 24 ? bins & 0xFF : 0; C.nb1 = (bins >> 8) & 0xFF; C.nb2 = (bins >> 16) & 0xFF;
    C.xs = A.xs4 + R->first;
    C.bs = A.bin_start + R->first + 2 * s;
    // (an atom far from the origin or not finite: the generic rows, which check every offset)
    if (C.nb0 && C.bs[C.nb0 * C.nb1 * C.nb2 + 1] == 0) C.nb0 = 0;
}


// ---- staging of one structure in the warp's shared memory ---------------------------------------
// Returns false (on every lane) if a coordinate is non-finite or too far from the cell.
__device__ __forceinline__ bool mgs_stage(SSmem &ws, const WCtx &C, int lane) {
    __syncwarp();
    bool ok = true;
    for (int j = lane; j < C.N; j += 32) {
        const float4 xw = C.xw[j];
        ok = ok && __float_as_int(xw.w) != 0;
        ws.x[j] = xw;
    }
    // table of local translations t . L, t in [0, m): cells [0, mloc), then a far-away sentinel up to
    // a multiple of 32 and one group beyond (the filter reads one group ahead)
    const int M12 = C.m1 * C.m2;
    const float inv12 = 1.f / (float)M12, inv2 = 1.f / (float)C.m2;
    const int pad = min(MGS_TL + 4, ((C.mloc + 31) & ~31) + 4);
    for (int c = lane; c < pad; c += 32) {
        float Tx = 1e18f, Ty = 1e18f, Tz = 1e18f;
        if (c < C.mloc) {
            const int t0 = mg_fdiv(c, inv12), r = c - t0 * M12;
            const int t1 = mg_fdiv(r, inv2), t2 = r - t1 * C.m2;
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            Tx = __fmaf_rn(f2, C.a[6], __fmaf_rn(f1, C.a[3], __fmul_rn(f0, C.a[0])));
            Ty = __fmaf_rn(f2, C.a[7], __fmaf_rn(f1, C.a[4], __fmul_rn(f0, C.a[1])));
            Tz = __fmaf_rn(f2, C.a[8], __fmaf_rn(f1, C.a[5], __fmul_rn(f0, C.a[2])));
            ws.tcode[c] = ((unsigned)t0 << 24) | ((unsigned)t1 << 16) | ((unsigned)t2 << 8);
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
struct SPair {
    float qx, qy, qz;
    int l0, l1, l2;
    int self;              // index of the cell tau = 0 in the table if i == j, else -1
    float rc;              // cutoff of the source
    bool ok;               // valid lane, offsets inside int8
};

__device__ __forceinline__ SPair mgs_pair(const SSmem &ws, const WCtx &C, bool valid, int i, int j) {
    SPair p;
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
    p.rc = C.cr ? C.cr[i] : C.rc;
    return p;
}

// Hit mask of cells [32 w, 32 w + 32) of the pair's sub-box: bit 31 - c <-> cell 32 w + c (the sign
// bits of y = |q' + T|^2 - r_c^2 are shifted in one by one).  Two cells per packed FP32 instruction,
// table groups read one ahead.  A lane that saw |y| < win decides those cells again with the exact
// FP64 predicate, so the mask is Def. 3's in FP64.
__device__ __forceinline__ unsigned mgs_word_mask(const SSmem &ws, const WCtx &C, const SPair &p, int i, int j, int w) {
    const int nw = min(32, C.mloc - 32 * w), n4 = (nw + 3) >> 2;      // warp-uniform
    const float4 *Xp = reinterpret_cast<const float4 *>(&ws.T[0][32 * w]);
    const float4 *Yp = reinterpret_cast<const float4 *>(&ws.T[1][32 * w]);
    const float4 *Zp = reinterpret_cast<const float4 *>(&ws.T[2][32 * w]);
    const float2 qx = make_float2(p.qx, p.qx), qy = make_float2(p.qy, p.qy), qz = make_float2(p.qz, p.qz);
    const float nr2s = C.cr ? -__fmul_rn(p.rc, p.rc) : C.nr2;
    const float2 nr2 = make_float2(nr2s, nr2s);
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
            const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, nr2s)));
            if (fabsf(y) < win) {
                const unsigned tc = ws.tcode[32 * w + c];
                double v[3];
                const double d = mg_exact_vec(xi, xj, p.l0 + (int)(tc >> 24), p.l1 + (int)((tc >> 16) & 0xFFu),
                                              p.l2 + (int)((tc >> 8) & 0xFFu), C.lat, v);
                const unsigned bit = 0x80000000u >> c;
                mask = d < (double)p.rc ? (mask | bit) : (mask & ~bit);
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
__device__ __forceinline__ bool mgs_cand(const WCtx &C, const float4 xi, float rci, int i, int j, int t0, int t1, int t2,
                                         int tau[3], bool &bad) {
    const float4 xj = C.xw[j];
    const int ki = __float_as_int(xi.w), kj = __float_as_int(xj.w);
    const float u0 = __fsub_rn(xj.x, xi.x), u1 = __fsub_rn(xj.y, xi.y), u2 = __fsub_rn(xj.z, xi.z);
    const float e0 = floorf(__fsub_rn(-C.rho[0], u0)) + 1.f, e1 = floorf(__fsub_rn(-C.rho[1], u1)) + 1.f,
                e2 = floorf(__fsub_rn(-C.rho[2], u2)) + 1.f;
    const float f0 = __fadd_rn(u0, e0 + (float)t0), f1 = __fadd_rn(u1, e1 + (float)t1), f2 = __fadd_rn(u2, e2 + (float)t2);
    const float vx = __fmaf_rn(f2, C.a[6], __fmaf_rn(f1, C.a[3], __fmul_rn(f0, C.a[0])));
    const float vy = __fmaf_rn(f2, C.a[7], __fmaf_rn(f1, C.a[4], __fmul_rn(f0, C.a[1])));
    const float vz = __fmaf_rn(f2, C.a[8], __fmaf_rn(f1, C.a[5], __fmul_rn(f0, C.a[2])));
    const float y = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmaf_rn(vx, vx, -__fmul_rn(rci, rci))));
    tau[0] = (int)e0 + t0 + (ki & 1023) - (kj & 1023);
    tau[1] = (int)e1 + t1 + ((ki >> 10) & 1023) - ((kj >> 10) & 1023);
    tau[2] = (int)e2 + t2 + ((ki >> 20) & 1023) - ((kj >> 20) & 1023);
    bad = ki == 0 || kj == 0 || tau[0] < -127 || tau[1] < -127 || tau[2] < -127 || tau[0] > 127 || tau[1] > 127 || tau[2] > 127;
    if (bad) return false;
    if (i == j && (tau[0] | tau[1] | tau[2]) == 0) return false;    // (i, i, 0) is not an edge (R3)
    bool hit = y < 0.f;
    if (fabsf(y) < C.win) {                                          // FP32 cannot decide: Def. 3 in FP64
        double v[3];
        hit = mg_exact_vec(C.gx + 3 * i, C.gx + 3 * j, tau[0], tau[1], tau[2], C.lat, v) < (double)rci;
    }
    return hit;
}


// What the list phase leaves for the write kernel, per source row [first + ia, first + ib) of structure s.
__device__ __forceinline__ void mgs_row_products(const ScanArgs &A, const WCtx &C, int s, int ia, int ib, int lane) {
    for (int i = ia + lane; i < ib; i += 32) {
        const int g = C.first + i;
        A.atom_struct[g] = s;
        double2 *p = reinterpret_cast<double2 *>(A.pos64 + 4 * (size_t)g);
        p[0] = make_double2((double)C.gx[3 * i], (double)C.gx[3 * i + 1]);
        p[1] = make_double2((double)C.gx[3 * i + 2], 0.0);
    }
    if (ia == 0 && lane < 9) A.lat64[9 * (size_t)s + lane] = (double)C.lat[lane];
}

// The edges [g0, g0 + n) belong to rows in such a way that edge g0 + p is in the row `row` on the lane
// that holds p in [excl, excl + cnt): every MGS_SLICE-th edge records its row.
__device__ __forceinline__ void mgs_slice_rows(const ScanArgs &A, unsigned long long g0, unsigned n, unsigned excl,
                                               unsigned cnt, int row, int first, int natoms, int s) {
    const unsigned long long b0 = (g0 + MGS_SLICE - 1) & ~(unsigned long long)(MGS_SLICE - 1);
    for (unsigned long long b = b0; b < g0 + n && (long long)b < A.capacity; b += MGS_SLICE) {
        const unsigned p = (unsigned)(b - g0);
        if (p >= excl && p < excl + cnt) A.slice_row[b / MGS_SLICE] = make_int4(row, first, first + natoms, s);
    }
}

// One edge written directly (the rare second walk of a warp whose codes did not fit the pool, PHASE 2).
__device__ __forceinline__ void mgs_emit_one(const ScanArgs &A, long long e, int gi, int gj, const float *gx, int i,
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

// ---- the code pool ------------------------------------------------------------------------------------
// While a warp finds its edges it does not know where they go in the output, so their codes go to
// chunks of MGS_CHUNK codes taken from a pool (one atomic per chunk); the chunk list stays in the warp's
// shared memory.  Local position p of the warp's codes lives at chunk list[p / MGS_CHUNK], p % MGS_CHUNK.
struct PoolState {
    unsigned wcount;       // codes of the warp so far (the same on every lane)
    int nch;               // chunks taken
    int *list;             // the range's chunk list (shared memory)
    bool ok;               // false: the pool or the list ran out; the warp only counts from then on and
                           // lists its rows again in the second phase (mgs_walk<1>)
};

__device__ __forceinline__ uint2 *mgs_pool_addr(const ScanArgs &A, const int *list, unsigned p) {
    return A.pool + (size_t)list[p / MGS_CHUNK] * MGS_CHUNK + (p % MGS_CHUNK);
}

// Make sure the chunks for local positions < upto exist.
__device__ __forceinline__ void mgs_pool_reserve(const ScanArgs &A, SSmem &ws, PoolState &P, unsigned upto, int lane) {
    while (P.ok && (unsigned)P.nch * MGS_CHUNK < upto) {
        int c = 0;
        if (lane == 0) c = (int)atomicAdd(A.ctl + 12, 1u);
        c = __shfl_sync(0xFFFFFFFFu, c, 0);
        if (c >= A.n_pool || P.nch >= MGS_MAXCH) { P.ok = false; break; }
        if (lane == 0) P.list[P.nch] = c;
        P.nch += 1;
        __syncwarp();
    }
}

// One source row: returns its edges; their codes go to the pool (PHASE 0) or to their final place from
// goff on (PHASE 1), in any order inside the row.
// Tables of 32 cells and more: lane <-> cell (decoded once per 32 cells), loop over the targets j.
// Smaller tables: lane <-> (target, cell), floor(32 / mloc) targets per pass.
template <int PHASE>
__device__ __forceinline__ unsigned mgs_row(const ScanArgs &A, SSmem &ws, PoolState &P, const WCtx &C, int i,
                                            unsigned long long goff, int lane, bool &anybad) {
    const float4 xi = C.xw[i];
    const float rci = C.cr ? C.cr[i] : C.rc;
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
            const bool hit = cv && j < C.N && mgs_cand(C, xi, rci, i, j, t0, t1, t2, tau, bad);
            anybad = anybad || bad;
            const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
            if (PHASE == 0 && bal) mgs_pool_reserve(A, ws, P, P.wcount + cnt + 32u, lane);
            if (hit) {
                const uint2 code = make_uint2((unsigned)(C.first + j), ((unsigned)(tau[0] + 128) << 24) |
                                              ((unsigned)(tau[1] + 128) << 16) | ((unsigned)(tau[2] + 128) << 8));
                const unsigned k = cnt + __popc(bal & ((1u << lane) - 1u));
                if (PHASE == 0) {
                    if (P.ok) *mgs_pool_addr(A, P.list, P.wcount + k) = code;
                } else if (PHASE == 2) {
                    mgs_emit_one(A, (long long)(goff + k), C.first + i, C.first + j, C.gx, i, j, tau, C.lat);
                } else if ((long long)(goff + k) < A.capacity) A.codes[goff + k] = code;
            }
            cnt += __popc(bal);
        }
    }
    return cnt;
}

// tau of a hit of a binned row: codes = rint(u_a) mod 4 (2 bits per axis), ki = the source's packed integer
// parts (cut_prep.cuh), wj = .w of the target's sorted entry (cut_bins.cuh): tau = -rint(u) + k_i - k_j.
__device__ __forceinline__ void mgs_bin_tau(unsigned codes, int ki, int wj, int tau[3]) {
    tau[0] = 1 - (int)((codes + 1u) & 3u) + ((ki & 1023) - 512) - (((wj >> 16) & 31) - 16);
    tau[1] = 1 - (int)(((codes >> 2) + 1u) & 3u) + (((ki >> 10) & 1023) - 512) - (((wj >> 21) & 31) - 16);
    tau[2] = 1 - (int)(((codes >> 4) + 1u) & 3u) + (((ki >> 20) & 1023) - 512) - (((wj >> 26) & 31) - 16);
}

// One source row of a structure with a cell list (cut_bins.cuh; one-cell sub-box): the candidates are
// the atoms of the 5 x 5 columns of bins around the row's bin (5 consecutive slabs of the last axis each:
// one or, across the periodic wrap, two runs of entries), walked as ONE sequence, lane <-> candidate, so
// that every trip but the last is full.  (BASELINE.json north_star: "stages each structure's positions ...
// in shared memory (TMA bulk copy where the structure is large)": the runs reach shared memory by
// cp.async.bulk.)
template <int PHASE>
__device__ __forceinline__ unsigned mgs_row_binned(const ScanArgs &A, SSmem &ws, PoolState &P, const WCtx &C, int i,
                                                   unsigned long long goff, int lane) {
    const float4 xi = C.xw[i];
    const float rci = C.cr ? C.cr[i] : C.rc;
    // ---- the row's columns: exclusive prefix of their lengths, first run (start, length), start of the second
    int *tp = reinterpret_cast<int *>(&ws.mk[0][0]), *ta1 = tp + 32, *tn1 = tp + 64, *ta2 = tp + 96;
    const int s0 = C.nb0 > 1 ? 5 : 1, s1 = C.nb1 > 1 ? 5 : 1, ncol = s0 * s1;
    int a1 = 0, n1 = 0, a2 = 0, n2 = 0;
    if (lane < ncol) {
        const int q = s1 == 5 ? lane / 5 : lane;
        int c0 = mgb_axis(xi.x, C.nb0) + (s0 == 5 ? q - 2 : 0), c1 = mgb_axis(xi.y, C.nb1) + (s1 == 5 ? lane - 5 * q - 2 : 0);
        c0 += c0 < 0 ? C.nb0 : 0; c0 -= c0 >= C.nb0 ? C.nb0 : 0;
        c1 += c1 < 0 ? C.nb1 : 0; c1 -= c1 >= C.nb1 ? C.nb1 : 0;
        const int *col = C.bs + (c0 * C.nb1 + c1) * C.nb2;
        if (C.nb2 == 1) { a1 = col[0]; n1 = col[1] - a1; }
        else {
            const int lo = mgb_axis(xi.z, C.nb2) - 2, hi = lo + 4;          // nb2 >= 6: the five slabs are distinct
            if (lo < 0) { a1 = col[0]; n1 = col[hi + 1] - a1; a2 = col[C.nb2 + lo]; n2 = col[C.nb2] - a2; }
            else if (hi >= C.nb2) { a1 = col[lo]; n1 = col[C.nb2] - a1; a2 = col[0]; n2 = col[hi - C.nb2 + 1] - a2; }
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
    // ---- the candidates.  The runs of the row's columns are copied, in sequence order, into two buffers of
    // MGS_CH entries in the warp's shared memory by TMA bulk copies (every lane issues the pieces of its own
    // column; the copy of chunk k + 1 flies while chunk k is tested), so a trip reads candidate v at buf[v].
    // A hit is the image of j nearest to i in fractional coordinates (rho_a < 1/2: no other image can be inside
    // r_c): f = u - rint(u), u = x_j - x_i (wrapped), d2 in FP32, FP64 decision inside the rounding window.
    // A trip only TESTS its candidates (two per lane, v and v + 32, in packed FP32; rint(u) = (u + 1.5 * 2^23)
    // - 1.5 * 2^23, whose low mantissa bits are rint(u) mod 4); the hits go to the stash as (v, rint(u) mod 4)
    // words and become codes, lane <-> hit, when the stash leaves.
    uint2 *st = ws.stash;                                          // MGS_STASH hits: (rint(u) mod 4 codes, .w of the entry)
    float4 *buf = reinterpret_cast<float4 *>(&ws.T[0][0]);         // 2 x MGS_CH entries
    const int ki = __float_as_int(xi.w);
    const float nr2 = -__fmul_rn(rci, rci), win = C.win;
    // the pieces of this lane's column inside chunk [base, base + MGS_CH) -> buffer b
    const int myp = incl - (n1 + n2);
    auto issue = [&](int base, int b) {
        const int nchunk = min(MGS_CH, total - base);
        if (lane == 0) mgs_bar_expect(&ws.bar[b], 16u * (unsigned)nchunk);
        __syncwarp();
        const int r_lo = max(base - myp, 0), r_hi = min(base + MGS_CH - myp, n1 + n2);
        if (r_lo < r_hi) {
            float4 *dst = buf + b * MGS_CH + (myp - base);
            const int e1 = min(r_hi, n1);
            if (r_lo < e1) mgs_bulk_g2s(dst + r_lo, C.xs + a1 + r_lo, 16u * (unsigned)(e1 - r_lo), &ws.bar[b]);
            const int b2 = max(r_lo, n1);
            if (b2 < r_hi) mgs_bulk_g2s(dst + b2, C.xs + a2 + (b2 - n1), 16u * (unsigned)(r_hi - b2), &ws.bar[b]);
        }
    };
    unsigned cnt = 0u, ns = 0u, done = 0u;
    unsigned phase = ws.bphase;
    const unsigned lt = (1u << lane) - 1u;
    const float2 nx0 = make_float2(-xi.x, -xi.x), nx1 = make_float2(-xi.y, -xi.y), nx2 = make_float2(-xi.z, -xi.z);
    const float2 MAG = make_float2(12582912.f, 12582912.f), NMAG = make_float2(-12582912.f, -12582912.f);
    const float2 M1 = make_float2(-1.f, -1.f), Z2 = make_float2(0.f, 0.f), nr22 = make_float2(nr2, nr2);
    const float2 a0 = make_float2(C.a[0], C.a[0]), a1v = make_float2(C.a[1], C.a[1]), a2v = make_float2(C.a[2], C.a[2]),
                 a3 = make_float2(C.a[3], C.a[3]), a4 = make_float2(C.a[4], C.a[4]), a5 = make_float2(C.a[5], C.a[5]),
                 a6 = make_float2(C.a[6], C.a[6]), a7 = make_float2(C.a[7], C.a[7]), a8 = make_float2(C.a[8], C.a[8]);
    mgs_fence_async();                             // (the staging area may hold the pair-lane path's tables)
    __syncwarp();
    if (total > 0) issue(0, 0);
    for (int v0 = 0; v0 < total || ns; v0 += 64) {
        if (v0 < total) {
            const int k = v0 / MGS_CH, b = k & 1, t = v0 - k * MGS_CH;
            if (t == 0) {                          // a new chunk: wait for it, send for the next one
                mgs_bar_wait(&ws.bar[b], (phase >> b) & 1u);
                phase ^= 1u << b;
                if ((k + 1) * MGS_CH < total) issue((k + 1) * MGS_CH, b ^ 1);
            }
            const int vA = v0 + lane, vB = vA + 32;
            const bool okA = vA < total, okB = vB < total;
            const float4 xA = buf[b * MGS_CH + t + lane], xB = buf[b * MGS_CH + t + 32 + lane];
            const float2 u0 = mg_add2(make_float2(xA.x, xB.x), nx0), u1 = mg_add2(make_float2(xA.y, xB.y), nx1),
                         u2 = mg_add2(make_float2(xA.z, xB.z), nx2);
            const float2 m0 = mg_add2(u0, MAG), m1 = mg_add2(u1, MAG), m2 = mg_add2(u2, MAG);
            const float2 f0 = mg_fma2(mg_add2(m0, NMAG), M1, u0), f1 = mg_fma2(mg_add2(m1, NMAG), M1, u1),
                         f2 = mg_fma2(mg_add2(m2, NMAG), M1, u2);
            const float2 vx = mg_fma2(f2, a6, mg_fma2(f1, a3, mg_fma2(f0, a0, Z2)));
            const float2 vy = mg_fma2(f2, a7, mg_fma2(f1, a4, mg_fma2(f0, a1v, Z2)));
            const float2 vz = mg_fma2(f2, a8, mg_fma2(f1, a5, mg_fma2(f0, a2v, Z2)));
            const float2 y = mg_fma2(vz, vz, mg_fma2(vy, vy, mg_fma2(vx, vx, nr22)));
            bool hitA = okA && y.x < 0.f, hitB = okB && y.y < 0.f;
            const unsigned wordA = (__float_as_uint(m0.x) & 3u) | ((__float_as_uint(m1.x) & 3u) << 2) | ((__float_as_uint(m2.x) & 3u) << 4);
            const unsigned wordB = (__float_as_uint(m0.y) & 3u) | ((__float_as_uint(m1.y) & 3u) << 2) | ((__float_as_uint(m2.y) & 3u) << 4);
            if (fminf(fabsf(y.x), fabsf(y.y)) < win) {                        // FP32 cannot decide: Def. 3 in FP64
#pragma unroll 1
                for (int h = 0; h < 2; ++h) {
                    const float yh = h ? y.y : y.x;
                    if (!(h ? okB : okA) || !(fabsf(yh) < win)) continue;
                    int tau[3];
                    const int wj = __float_as_int((h ? xB : xA).w);
                    mgs_bin_tau(h ? wordB : wordA, ki, wj, tau);
                    const int j = wj & 0xFFFF, t0 = tau[0], t1 = tau[1], t2 = tau[2];
                    double w3[3];
                    const bool e = mg_exact_vec(C.gx + 3 * i, C.gx + 3 * j, t0, t1, t2, C.lat, w3) < (double)rci;
                    if (h) hitB = e; else hitA = e;
                }
            }
            hitA = hitA && (__float_as_int(xA.w) & 0xFFFF) != i;               // (i, i, 0) is not an edge (R3)
            hitB = hitB && (__float_as_int(xB.w) & 0xFFFF) != i;
            const unsigned balA = __ballot_sync(0xFFFFFFFFu, hitA), balB = __ballot_sync(0xFFFFFFFFu, hitB);
            const unsigned nA = __popc(balA);
            if (hitA) st[ns + __popc(balA & lt)] = make_uint2(wordA, __float_as_uint(xA.w));
            if (hitB) st[ns + nA + __popc(balB & lt)] = make_uint2(wordB, __float_as_uint(xB.w));
            ns += nA + __popc(balB);
            cnt += nA + __popc(balB);
            if (ns <= MGS_STASH - 64 && v0 + 64 < total) continue;
        }
        // ---- the stash leaves: entry -> (dst, tau) code, lane <-> hit
        __syncwarp();
        if (PHASE == 0) mgs_pool_reserve(A, ws, P, P.wcount + done + ns, lane);
        for (unsigned x = lane; x < ns; x += 32) {
            const uint2 w = st[x];
            const int j = (int)(w.y & 0xFFFFu);
            int tau[3];
            mgs_bin_tau(w.x, ki, (int)w.y, tau);
            // (cut_bins.cuh: the atoms are finite and within 15 cells of the origin, so |tau| <= 31)
            const uint2 code = make_uint2((unsigned)(C.first + j), ((unsigned)(tau[0] + 128) << 24) |
                                          ((unsigned)(tau[1] + 128) << 16) | ((unsigned)(tau[2] + 128) << 8));
            if (PHASE == 0) {
                if (P.ok) *mgs_pool_addr(A, P.list, P.wcount + done + x) = code;
            } else if (PHASE == 2) {
                mgs_emit_one(A, (long long)(goff + done + x), C.first + i, C.first + j, C.gx, i, j, tau, C.lat);
            } else if ((long long)(goff + done + x) < A.capacity) A.codes[goff + done + x] = code;
        }
        done += ns;
        ns = 0u;
        __syncwarp();
    }
    if (lane == 0) ws.bphase = phase;
    return cnt;
}

// ---- the walk of a warp over its rows -------------------------------------------------------------
// PHASE 0 (find): hits of every block -> codes in the pool, row_ptr = offsets LOCAL to the warp, the
//   products of the rows (atom_struct, pos64, lat64); returns the warp's edge count (on every lane).
// PHASE 1 (list again): for a warp whose codes did not fit the pool: the same walk with the final
//   offset goff known: row_ptr, slice records and codes go straight to their place.
template <int PHASE, bool BINNED>
__device__ __forceinline__ unsigned long long mgs_walk(SSmem &ws, const ScanArgs &A, const RangeCtx &RC, int rid,
                                                       PoolState &P, int &row_lo, int &row_hi,
                                                       unsigned long long goff, int lane) {
    unsigned long long c0, c1;
    mg_warp_range(RC, rid, c0, c1);
    int s, qa;
    mg_range_start(RC, c0, s, qa, lane);
#ifdef MG_PHASE_CLOCKS
    const long long wt0 = clock64();
    const int dbg_s0 = s;
    int dbg_seg = 0, dbg_blk = 0, dbg_rows = 0, dbg_grp = 0;
    const unsigned long long dbg_g0 = goff;
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
            WCtx C;
            mgs_ctx<BINNED>(C, A, R, s);
            if (PHASE == 0) {
                mgs_row_products(A, C, s, ia, ib, lane);
                if (row_lo < 0) row_lo = C.first + ia;
                row_hi = C.first + ib;
            }
            // where the next edge goes: local position (find) or final position (list again)
#define MGS_HERE (PHASE == 0 ? (unsigned long long)P.wcount : goff)
            if (mloc <= 0) {                       // invalid structure: empty rows
                for (int i = ia + lane; i < ib; i += 32) A.row_ptr[C.first + i] = (int)MGS_HERE;
            } else if (N > MGS_NMAX || mloc > MGS_TL) {
                for (int i = ia; i < ib; ++i) {
                    bool anybad = false;
                    if (lane == 0) A.row_ptr[C.first + i] = (int)MGS_HERE;
                    const unsigned cnt = BINNED && C.nb0 ? mgs_row_binned<PHASE>(A, ws, P, C, i, goff, lane)
                                               : mgs_row<PHASE>(A, ws, P, C, i, goff, lane, anybad);
                    if (PHASE == 0) {
                        if (anybad) atomicOr(A.status, __float_as_int(C.xw[i].w) == 0 ? MGS_NONFINITE : MGS_OFFSET);
                        P.wcount += cnt;
                    } else {
                        if (PHASE == 1 && lane == 0) mgs_slice_rows(A, goff, cnt, 0u, cnt, C.first + i, C.first, C.N, s);
                        goff += cnt;
                    }
                }
#ifdef MG_PHASE_CLOCKS
                dbg_rows += ib - ia; dbg_seg += 1;
#endif
            } else {
                const bool live = mgs_stage(ws, C, lane);
                const int nW = (mloc + 31) >> 5;
                const int q0 = ia * N, q1 = ib * N, nblk = (q1 - q0 + 31) >> 5;
                const float inv_N = 1.f / (float)N;
                if (!live) {
                    if (PHASE == 0 && lane == 0) atomicOr(A.status, MGS_NONFINITE);
                    for (int i = ia + lane; i < ib; i += 32) A.row_ptr[C.first + i] = (int)MGS_HERE;
                } else {
#pragma unroll 1
                    for (int b = 0; b < nblk; ++b) {
                        const int q = q0 + 32 * b + lane;
                        const bool valid = q < q1;
                        int i = 0, j = 0;
                        if (valid) { i = mg_fdiv(q, inv_N); j = q - i * N; }
                        const SPair p = mgs_pair(ws, C, valid, i, j);
                        if (PHASE == 0 && valid && !p.ok) atomicOr(A.status, MGS_OFFSET);
                        unsigned cnt = 0u;
#pragma unroll 1
                        for (int w = 0; w < nW; ++w) {
                            const unsigned m = mgs_word_mask(ws, C, p, i, j, w);
                            cnt += __popc(m);
                            ws.mk[w][lane] = m;
                        }
                        unsigned incl = cnt;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const unsigned v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                            if (lane >= o) incl += v;
                        }
                        const unsigned tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
                        if (valid && j == 0) A.row_ptr[C.first + i] = (int)(MGS_HERE + incl - cnt);
                        if (tot == 0u) continue;
                        if (PHASE == 1) mgs_slice_rows(A, goff, tot, incl - cnt, cnt, C.first + i, C.first, C.N, s);
                        if (PHASE == 0) mgs_pool_reserve(A, ws, P, P.wcount + tot, lane);
                        if (PHASE == 0 && !P.ok) { P.wcount += tot; continue; }       // count only from here on
                        // passes of consecutive lanes whose hits fit the stash (nearly always one)
                        const unsigned pc = ((unsigned)(p.l0 + 128) << 24) | ((unsigned)(p.l1 + 128) << 16) |
                                            ((unsigned)(p.l2 + 128) << 8);
                        const unsigned gj = (unsigned)(C.first + j);
                        unsigned done = 0u;
                        int l0 = 0;
                        while (done < tot) {
                            const bool mine = lane >= l0 && incl - done <= MGS_STASH;
                            const int nl = __popc(__ballot_sync(0xFFFFFFFFu, mine));   // >= 1: a lane has <= MGS_TL hits
                            const unsigned t = __shfl_sync(0xFFFFFFFFu, incl, l0 + nl - 1) - done;
                            if (mine) {
                                unsigned pos = incl - cnt - done;
#pragma unroll 1
                                for (int w = 0; w < nW; ++w) {
                                    unsigned mk = ws.mk[w][lane];
                                    while (mk) {
                                        const int bit = __clz(mk);
                                        mk &= ~(0x80000000u >> bit);
                                        const unsigned tbits = pc + ws.tcode[32 * w + bit];
                                        if (PHASE == 2) {
                                            const int tau[3] = {(int)(tbits >> 24) - 128, (int)((tbits >> 16) & 0xFFu) - 128,
                                                                (int)((tbits >> 8) & 0xFFu) - 128};
                                            mgs_emit_one(A, (long long)(goff + pos), C.first + i, (int)gj, C.gx, i, j, tau, C.lat);
                                            ++pos;
                                        } else ws.stash[pos++] = make_uint2(gj, tbits);
                                    }
                                }
                            }
                            __syncwarp();
                            if (PHASE == 0) {          // codes -> the pool, at the warp's local positions
                                for (unsigned x = lane; x < t; x += 32) *mgs_pool_addr(A, P.list, P.wcount + x) = ws.stash[x];
                                P.wcount += t;
                            } else if (PHASE == 2) {
                                goff += t;
                            } else {                   // codes -> their final place in the stream
                                const long long room = A.capacity - (long long)goff;
                                const int lim = room >= (long long)t ? (int)t : (room > 0 ? (int)room : 0);
                                uint2 *dst = A.codes + goff;
                                for (int x = lane; x < lim; x += 32) dst[x] = ws.stash[x];
                                goff += t;
                            }
                            __syncwarp();
                            done += t;
                            l0 += nl;
                        }
                    }
                }
#ifdef MG_PHASE_CLOCKS
                dbg_blk += nblk; dbg_seg += 1;
                for (int w = 0; w < nW; ++w) dbg_grp += nblk * ((((min(32, mloc - 32 * w) + 3) >> 2) + 1) & ~1);
#endif
            }
#undef MGS_HERE
        }
        if (!more) break;
    }
#ifdef MG_PHASE_CLOCKS
    if (lane == 0 && A.dbg) {
        unsigned *d = A.dbg + 4 * 2048 + 16 * rid + 8 * PHASE;
        d[0] = (unsigned)(clock64() - wt0); d[1] = dbg_s0; d[2] = dbg_seg; d[3] = dbg_blk; d[4] = dbg_rows; d[5] = P.nch;
        d[6] = dbg_grp; d[7] = PHASE == 1 ? (unsigned)(goff - dbg_g0) : P.wcount;
    }
#endif
    return PHASE == 0 ? (unsigned long long)P.wcount : goff;
}

// ((x_dst - x_src) + tau) . L evaluated like the oracle does (Def. 3, R15: no FMA contraction,
// sums left to right); tb = (tau + 128) bytes << 8.
__device__ __forceinline__ void mgs_vec(const double xi[3], const double xj[3], unsigned tb, const double L[9], double w3[3]) {
    // (double)(b - 128) without a conversion instruction: 2^52 + b has b in its low mantissa word
    const double f0 = __dadd_rn(__dsub_rn(xj[0], xi[0]), __hiloint2double(0x43300000, (int)(tb >> 24)) - 4503599627370624.0);
    const double f1 = __dadd_rn(__dsub_rn(xj[1], xi[1]), __hiloint2double(0x43300000, (int)((tb >> 16) & 0xFFu)) - 4503599627370624.0);
    const double f2 = __dadd_rn(__dsub_rn(xj[2], xi[2]), __hiloint2double(0x43300000, (int)((tb >> 8) & 0xFFu)) - 4503599627370624.0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
        w3[c] = __dadd_rn(__dadd_rn(__dmul_rn(f0, L[c]), __dmul_rn(f1, L[3 + c])), __dmul_rn(f2, L[6 + c]));
}

// What the caller's arrays look like to the writers.
struct OutArrays {
    int32_t *src, *dst;
    int8_t *offset;
    float *vec, *dist;
    bool al16;             // src, dst, vec (, dist) 16-byte aligned, offset 4-byte aligned
};

// Four consecutive edges e .. e + 3 of one lane (e a multiple of 4); ok[y]: edge y exists.
__device__ __forceinline__ void mgs_store4(const OutArrays &O, long long e, const bool ok[4], const int gi[4], const int gj[4],
                                           const unsigned tb[4], const float v[4][3], const float d[4]) {
    if (O.al16 && ok[0] && ok[3]) {
        *reinterpret_cast<int4 *>(O.src + e) = make_int4(gi[0], gi[1], gi[2], gi[3]);
        *reinterpret_cast<int4 *>(O.dst + e) = make_int4(gj[0], gj[1], gj[2], gj[3]);
        float4 *pv = reinterpret_cast<float4 *>(O.vec + 3 * e);
        pv[0] = make_float4(v[0][0], v[0][1], v[0][2], v[1][0]);
        pv[1] = make_float4(v[1][1], v[1][2], v[2][0], v[2][1]);
        pv[2] = make_float4(v[2][2], v[3][0], v[3][1], v[3][2]);
        // 12 offset bytes: tau of four edges (a code's .y = b0 b1 b2 0 from the top byte down), signed
        const unsigned t0 = tb[0] ^ 0x80808000u, t1 = tb[1] ^ 0x80808000u, t2 = tb[2] ^ 0x80808000u, t3 = tb[3] ^ 0x80808000u;
        unsigned *po = reinterpret_cast<unsigned *>(O.offset + 3 * e);
        po[0] = __byte_perm(t0, t1, 0x7123);       // bytes in memory: t0.b3 t0.b2 t0.b1 t1.b3
        po[1] = __byte_perm(t1, t2, 0x6712);       //                  t1.b2 t1.b1 t2.b3 t2.b2
        po[2] = __byte_perm(t2, t3, 0x5671);       //                  t2.b1 t3.b3 t3.b2 t3.b1
        if (O.dist) *reinterpret_cast<float4 *>(O.dist + e) = make_float4(d[0], d[1], d[2], d[3]);
    } else {
#pragma unroll
        for (int y = 0; y < 4; ++y)
            if (ok[y]) {
                O.src[e + y] = gi[y];
                O.dst[e + y] = gj[y];
                O.vec[3 * (e + y)] = v[y][0]; O.vec[3 * (e + y) + 1] = v[y][1]; O.vec[3 * (e + y) + 2] = v[y][2];
                const unsigned t = tb[y] ^ 0x80808000u;
                O.offset[3 * (e + y)] = (int8_t)(t >> 24); O.offset[3 * (e + y) + 1] = (int8_t)(t >> 16);
                O.offset[3 * (e + y) + 2] = (int8_t)(t >> 8);
                if (O.dist) O.dist[e + y] = d[y];
            }
    }
}

// Second phase of a warp whose codes are in the pool: codes -> their final place, row_ptr from local to
// final offsets, and for every MGS_SLICE-th edge of the output the record the write kernel starts from.
__device__ __forceinline__ void mgs_place(const ScanArgs &A, const int *list, unsigned total, int row_lo, int row_hi,
                                          unsigned long long base, int lane) {
    {
        const long long room = A.capacity - (long long)base;
        const unsigned lim = room >= (long long)total ? total : (room > 0 ? (unsigned)room : 0u);
        uint2 *dst = A.codes + base;
        unsigned x = lane;
        for (; x + 96 < lim; x += 128) {               // four loads in flight
            const uint2 c0 = *mgs_pool_addr(A, list, x), c1 = *mgs_pool_addr(A, list, x + 32),
                        c2 = *mgs_pool_addr(A, list, x + 64), c3 = *mgs_pool_addr(A, list, x + 96);
            dst[x] = c0; dst[x + 32] = c1; dst[x + 64] = c2; dst[x + 96] = c3;
        }
        for (; x < lim; x += 32) dst[x] = *mgs_pool_addr(A, list, x);
    }
    for (int r0 = row_lo; r0 < row_hi; r0 += 32) {
        const int r = r0 + lane;
        unsigned v = total, vn = total;
        if (r < row_hi) v = (unsigned)A.row_ptr[r];
        if (lane == 31 && r + 1 < row_hi) vn = (unsigned)A.row_ptr[r + 1];
        const unsigned down = __shfl_down_sync(0xFFFFFFFFu, v, 1);
        if (lane < 31) vn = down;                   // (rows past row_hi hold `total`)
        __syncwarp();
        if (r < row_hi) {
            A.row_ptr[r] = (int)(base + v);
            if (vn > v) {
                const unsigned long long b0 = (base + v + MGS_SLICE - 1) & ~(unsigned long long)(MGS_SLICE - 1);
                if (b0 < base + vn && (long long)b0 < A.capacity) {
                    const int s = A.atom_struct[r];
                    const int first = A.rec[s].first, nat = A.rec[s].natoms;
                    for (unsigned long long b = b0; b < base + vn && (long long)b < A.capacity; b += MGS_SLICE)
                        A.slice_row[b / MGS_SLICE] = make_int4(r, first, first + nat, s);
                }
            }
        }
    }
}

// Second phase of a warp whose codes are in the pool, writing the caller's arrays itself (no code stream,
// no write kernel): row_ptr from local to final offsets, then batches of 128 edges, lane <-> four
// consecutive edges whose global index starts at a multiple of 4, so that every array leaves in aligned
// 16-byte stores (scalar stores for the ragged first / last lanes of the warp's edges).  Uses the stash
// area of the warp's shared memory for the row counters and the staged FP64 positions.
__device__ __forceinline__ void mgs_place_write(const ScanArgs &A, const OutArrays &O, SSmem &ws, const int *list,
                                                unsigned total, int row_lo, int row_hi, unsigned long long base, int lane) {
    for (int r0 = row_lo; r0 < row_hi; r0 += 32) {          // my rows: local -> final offsets
        const int r = r0 + lane;
        if (r < row_hi) A.row_ptr[r] = (int)(base + (unsigned)A.row_ptr[r]);
    }
    __syncwarp();
    if (total == 0u) return;
    int *cnt = reinterpret_cast<int *>(ws.stash);
    double *xs = reinterpret_cast<double *>(ws.stash + 64);            // 3 * MGS_NMAX doubles
    const long long lim = (long long)total < A.capacity - (long long)base ? (long long)total : A.capacity - (long long)base;
    int r0 = row_lo, cur_s = -1, a_lo = 0, win = 0, nat = 0;
    double L[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) L[c] = 0.0;
    for (long long qb = -(long long)(base & 3ull); qb < lim; qb += 128) {
        const long long gb = (long long)base + qb;                     // global index of the batch's first slot
        // ---- the lane's codes
        int gj[4];
        unsigned tb[4];
        bool ok[4];
#pragma unroll
        for (int y = 0; y < 4; ++y) {
            const long long q = qb + 4 * lane + y;
            ok[y] = q >= 0 && q < lim;
            gj[y] = 0; tb[y] = 0x80808000u;
            if (ok[y]) { const uint2 c = *mgs_pool_addr(A, list, (unsigned)q); gj[y] = (int)c.x; tb[y] = c.y; }
        }
        // ---- rows: row of slot p = r0 + number of my rows r > r0 that start at or before it
        __syncwarp();
#pragma unroll
        for (int x = 0; x < 4; ++x) cnt[32 * x + lane] = 0;
        __syncwarp();
        for (int rb = r0 + 1;; rb += 32) {
            const int r = rb + lane;
            bool in = false;
            if (r < row_hi) {
                const long long start = (long long)A.row_ptr[r];
                in = start < gb + 128;
                if (in) atomicAdd(&cnt[start > gb ? (int)(start - gb) : 0], 1);
            }
            if (!__all_sync(0xFFFFFFFFu, in)) break;
        }
        __syncwarp();
        int c4[4];
#pragma unroll
        for (int y = 0; y < 4; ++y) c4[y] = cnt[4 * lane + y];
        int incl = c4[0] + c4[1] + c4[2] + c4[3];
        const int own = incl;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        int row = r0 + incl - own;
        int gi[4];
#pragma unroll
        for (int y = 0; y < 4; ++y) { row += c4[y]; gi[y] = row; }
        // ---- lattice and positions of the structure of the batch's first row
        const int rf = __shfl_sync(0xFFFFFFFFu, gi[0], 0);
        const int s0 = A.atom_struct[rf];
        if (s0 != cur_s) {
            cur_s = s0;
            a_lo = A.rec[s0].first;
            nat = A.rec[s0].natoms;
            win = min(MGS_NMAX, nat);
            const double *pl = A.lat64 + 9 * (size_t)s0;
#pragma unroll
            for (int c = 0; c < 9; ++c) L[c] = pl[c];
            __syncwarp();
            const double2 *px = reinterpret_cast<const double2 *>(A.pos64 + 4 * (size_t)a_lo);
            for (int a = lane; a < win; a += 32) {
                const double2 p0 = px[2 * a], p1 = px[2 * a + 1];
                xs[3 * a] = p0.x; xs[3 * a + 1] = p0.y; xs[3 * a + 2] = p1.x;
            }
            __syncwarp();
        }
        float v[4][3], d[4];
        double xi[3] = {0.0, 0.0, 0.0};                // position of the source of the lane's last edge outside the window
        int xi_of = -1;                                // (a lane's four edges are nearly always one row: loaded once)
#pragma unroll
        for (int y = 0; y < 4; ++y) {
            v[y][0] = v[y][1] = v[y][2] = 0.f; d[y] = 0.f;
            if (!ok[y]) continue;
            double w3[3];
            const unsigned wi = (unsigned)(gi[y] - a_lo), wj = (unsigned)(gj[y] - a_lo);
            if (wi < (unsigned)win && wj < (unsigned)win) {
                mgs_vec(xs + 3 * wi, xs + 3 * wj, tb[y], L, w3);
            } else {                                   // a structure above the window, or another structure
                double xj[3];
                {                                      // one sector per atom, two 16-byte loads
                    const double2 *pj = reinterpret_cast<const double2 *>(A.pos64 + 4 * (size_t)gj[y]);
                    const double2 j0 = pj[0], j1 = pj[1];
                    if (gi[y] != xi_of) {
                        const double2 *pi = reinterpret_cast<const double2 *>(A.pos64 + 4 * (size_t)gi[y]);
                        const double2 i0 = pi[0], i1 = pi[1];
                        xi[0] = i0.x; xi[1] = i0.y; xi[2] = i1.x;
                        xi_of = gi[y];
                    }
                    xj[0] = j0.x; xj[1] = j0.y; xj[2] = j1.x;
                }
                if (wi < (unsigned)nat) mgs_vec(xi, xj, tb[y], L, w3);
                else {
                    const int s = A.atom_struct[gi[y]];
                    double L2[9];
#pragma unroll
                    for (int c = 0; c < 9; ++c) L2[c] = A.lat64[9 * (size_t)s + c];
                    mgs_vec(xi, xj, tb[y], L2, w3);
                }
            }
            v[y][0] = (float)w3[0]; v[y][1] = (float)w3[1]; v[y][2] = (float)w3[2];
            if (O.dist)
                d[y] = __fsqrt_rn((float)__dadd_rn(__dadd_rn(__dmul_rn(w3[0], w3[0]), __dmul_rn(w3[1], w3[1])), __dmul_rn(w3[2], w3[2])));
        }
        mgs_store4(O, gb + 4 * lane, ok, gi, gj, tb, v, d);
        r0 = __shfl_sync(0xFFFFFFFFu, gi[3], 31);
    }
    __syncwarp();
}

// ---- launch 1 ---------------------------------------------------------------------------------------
#ifndef MGS_MIN_CTAS
#define MGS_MIN_CTAS 5
#endif
// BINNED: with the cell-list rows (batches of large structures).  The instance without them is the kernel for
// everything else that comes this way (per-atom cutoffs on small cells, MATGRAPH_FUSED): the cell-list code costs the
// pair-lane loops registers (90 against 82 us per call on BASELINE configs[2]).
template <bool BINNED>
__global__ void __launch_bounds__(MGS_BLOCK, MGS_MIN_CTAS)
mg_cutoff_scan_kernel(const __grid_constant__ ScanArgs A) {
    mg_grid_dependency_wait();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ScanSmem &sm = *reinterpret_cast<ScanSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    SSmem &ws = sm.w[warp];
    const unsigned epoch = *reinterpret_cast<volatile unsigned *>(A.ctl + 10) + 1u;   // tag of this call's slots
    if (lane == 0) { mgs_bar_init(&ws.bar[0]); mgs_bar_init(&ws.bar[1]); ws.bphase = 0u; }
    mgs_fence_async();
    __syncwarp();
    RangeCtx RC;
    const int n_warps = (int)gridDim.x * MGS_WARPS;
    mg_range_init(RC, A.rec, A.bpre, A.n_blocks, A.n_struct, MGS_WAVES * n_warps, lane);
    MGS_STAMP(0)
    // ---- find: the warp's range of every wave, one after the other; the CTA's total of a wave is published
    // as soon as its four warps are through, so that by the time a CTA wants the prefix of wave w the
    // other CTAs have long published theirs (they are busy with the waves after it)
#pragma unroll 1
    for (int wv = 0; wv < MGS_WAVES; ++wv) {
        PoolState P;
        P.wcount = 0u; P.nch = 0; P.ok = true; P.list = ws.chunks[wv];
        int row_lo = -1, row_hi = -1;
        const int rid = wv * n_warps + (int)blockIdx.x * MGS_WARPS + warp;
        const unsigned wtotal = (unsigned)mgs_walk<0, BINNED>(ws, A, RC, rid, P, row_lo, row_hi, 0ull, lane);
        __syncthreads();                               // (the previous wave's sums have been read)
        if (lane == 0) sm.wsum[warp] = wtotal;
        __syncthreads();
        unsigned long long total = 0ull, mine = 0ull;
#pragma unroll
        for (int w = 0; w < MGS_WARPS; ++w) {
            if (w < warp) mine += sm.wsum[w];
            total += sm.wsum[w];
        }
        if (lane == 0) {
            int *st = ws.wave[wv];
            st[0] = (int)wtotal; st[1] = P.nch; st[2] = P.ok ? 1 : 0; st[3] = row_lo; st[4] = row_hi;
            st[5] = (int)(unsigned)mine; st[6] = (int)(unsigned)total;
        }
        if (tid == 0)
            mg_st_release(A.slots + (size_t)wv * gridDim.x + blockIdx.x, ((unsigned long long)epoch << 32) | (total & 0xFFFFFFFFull));
    }
    __syncwarp();
    MGS_STAMP(1)
    if (!A.count_only) {
        OutArrays O;
        O.src = A.src; O.dst = A.dst; O.offset = A.offset; O.vec = A.vec; O.dist = A.dist;
        O.al16 = ((reinterpret_cast<unsigned long long>(A.src) | reinterpret_cast<unsigned long long>(A.dst) |
                   reinterpret_cast<unsigned long long>(A.vec) | reinterpret_cast<unsigned long long>(A.dist)) & 15ull) == 0ull &&
                 (reinterpret_cast<unsigned long long>(A.offset) & 3ull) == 0ull;
        unsigned long long waves_before = 0ull;        // edges of the waves before wv
#pragma unroll 1
        for (int wv = 0; wv < MGS_WAVES; ++wv) {
            // device-wide exclusive scan of K4: the slots of this wave before this CTA's, and the whole wave
            // (all CTAs are resident: cooperative launch)
            __syncthreads();
            if (warp == 0) {
                unsigned long long before = 0ull, all = 0ull;
                const unsigned long long *sl = A.slots + (size_t)wv * gridDim.x;
                // (a slot carries its own tag: relaxed loads, four in flight per lane, a lane spins only on a
                // slot that is not there yet)
                const int n_need = wv + 1 < MGS_WAVES ? (int)gridDim.x : (int)blockIdx.x;
                for (int c0 = 0; c0 < n_need; c0 += 128) {
                    unsigned long long v[4];
#pragma unroll
                    for (int x = 0; x < 4; ++x) {
                        const int c = c0 + 32 * x + lane;
                        v[x] = c < n_need ? mg_ld_relaxed(sl + c) : ((unsigned long long)epoch << 32);
                    }
#pragma unroll
                    for (int x = 0; x < 4; ++x) {
                        const int c = c0 + 32 * x + lane;
                        while ((unsigned)(v[x] >> 32) != epoch) { __nanosleep(100); v[x] = mg_ld_relaxed(sl + c); }
                        if (c < (int)blockIdx.x) before += v[x] & 0xFFFFFFFFull;
                        all += v[x] & 0xFFFFFFFFull;
                    }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    before += __shfl_xor_sync(0xFFFFFFFFu, before, o);
                    all += __shfl_xor_sync(0xFFFFFFFFu, all, o);
                }
                if (lane == 0) { sm.prefix = before; sm.wave_all = all; }
            }
            __syncthreads();
            const int *st = ws.wave[wv];
            const unsigned wtotal = (unsigned)st[0];
            PoolState P;
            P.wcount = wtotal; P.nch = st[1]; P.ok = st[2] != 0; P.list = ws.chunks[wv];
            int row_lo = st[3], row_hi = st[4];
            const unsigned long long base = waves_before + sm.prefix + (unsigned)st[5];
            if (wv == MGS_WAVES - 1 && blockIdx.x == gridDim.x - 1 && tid == 0) {    // the last range knows the grand total
                const unsigned long long tot = waves_before + sm.prefix + (unsigned)st[6];
                *A.n_edges = (long long)tot;
                A.row_ptr[A.n_atoms] = (int)tot;
                if (tot > 0x7FFFFFFFull || (long long)tot > A.capacity) atomicOr(A.status, MGS_CAPACITY);
            }
            waves_before += sm.wave_all;
            const int rid = wv * n_warps + (int)blockIdx.x * MGS_WARPS + warp;
            if (A.write_here) {
                if (P.ok) mgs_place_write(A, O, ws, P.list, wtotal, row_lo, row_hi, base, lane);
                else mgs_walk<2, BINNED>(ws, A, RC, rid, P, row_lo, row_hi, base, lane);
            } else if (P.ok) mgs_place(A, P.list, wtotal, row_lo, row_hi, base, lane);
            else mgs_walk<1, BINNED>(ws, A, RC, rid, P, row_lo, row_hi, base, lane);
        }
        MGS_STAMP(3)
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
        for (int c = lane; c < MGS_WAVES * (int)gridDim.x; c += 32) {
            unsigned long long v;
            while ((unsigned)((v = mg_ld_acquire(A.slots + c)) >> 32) != epoch) __nanosleep(100);
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
        A.ctl[12] = 0u;
        A.ctl[13] = 0u;                                // (the list of structures with a cell list: empty for the next call)
        __threadfence();
        *reinterpret_cast<volatile unsigned *>(A.ctl + 10) = epoch;
    }
}


// ---- launch 2 ---------------------------------------------------------------------------------------
struct WriteArgs {
    const uint2 *codes;
    const int4 *slice_row;
    const int32_t *atom_struct;
    const double *pos64, *lat64;
    const int32_t *row_ptr;
    const long long *n_edges;
    int n_atoms;
    long long capacity;
    int32_t *src, *dst;
    int8_t *offset;
    float *vec, *dist;
};

#define MGWR_BLOCK 256
#define MGWR_WARPS (MGWR_BLOCK / 32)
#define MGWR_WIN MGS_NMAX          // atoms of the position window a warp stages per slice
#ifndef MGWR_MIN_CTAS
#define MGWR_MIN_CTAS 3
#endif

// ((x_dst - x_src) + tau) . L evaluated like the oracle does (Def. 3, R15: no FMA contraction,
// sums left to right); tb = (tau + 128) bytes << 8.
__device__ __forceinline__ void mgwr_vec(const double xi[3], const double xj[3], unsigned tb, const double L[9], double w3[3]) {
    // (double)(b - 128) without a conversion instruction: 2^52 + b has b in its low mantissa word
    const double f0 = __dadd_rn(__dsub_rn(xj[0], xi[0]), __hiloint2double(0x43300000, (int)(tb >> 24)) - 4503599627370624.0);
    const double f1 = __dadd_rn(__dsub_rn(xj[1], xi[1]), __hiloint2double(0x43300000, (int)((tb >> 16) & 0xFFu)) - 4503599627370624.0);
    const double f2 = __dadd_rn(__dsub_rn(xj[2], xi[2]), __hiloint2double(0x43300000, (int)((tb >> 8) & 0xFFu)) - 4503599627370624.0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
        w3[c] = __dadd_rn(__dadd_rn(__dmul_rn(f0, L[c]), __dmul_rn(f1, L[3 + c])), __dmul_rn(f2, L[6 + c]));
}

// A warp takes slices of MGS_SLICE consecutive edges; lane <-> edges 4 lane .. 4 lane + 3 of the slice.
// Per slice, two rounds of loads: (1) its record (row of the first edge, the atoms of that row's
// structure, the structure) and the lane's four codes; (2) the row_ptr entries after that row, the
// structure's lattice and positions (FP64 copies of the scan kernel).  An edge of a later structure
// (the slice crosses a structure boundary) takes its operands from global memory instead.
__global__ void __launch_bounds__(MGWR_BLOCK, MGWR_MIN_CTAS)
mg_cutoff_write_kernel(const __grid_constant__ WriteArgs A) {
    mg_grid_dependency_wait();
    __shared__ int s_cnt[MGWR_WARPS][MGS_SLICE];
    __shared__ double s_x[MGWR_WARPS][3 * MGWR_WIN];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int *cnt = s_cnt[warp];
    double *xs = s_x[warp];
    const long long E = *A.n_edges < A.capacity ? *A.n_edges : A.capacity;       // edges to write
    const long long n_slices = (E + MGS_SLICE - 1) / MGS_SLICE;
    const bool al16 = ((reinterpret_cast<unsigned long long>(A.src) | reinterpret_cast<unsigned long long>(A.dst) |
                        reinterpret_cast<unsigned long long>(A.vec)) & 15ull) == 0ull &&
                      (reinterpret_cast<unsigned long long>(A.offset) & 3ull) == 0ull;
    const long long stride = (long long)gridDim.x * MGWR_WARPS;
    long long sl = (long long)blockIdx.x * MGWR_WARPS + warp;
    int4 info = make_int4(0, 0, 0, 0);
    if (sl < n_slices) info = __ldg(A.slice_row + sl);
    for (; sl < n_slices; sl += stride) {
        const long long g0 = sl * MGS_SLICE;
        const int n = (int)(E - g0 < MGS_SLICE ? E - g0 : MGS_SLICE);
        const int r0 = info.x, a_lo = info.y, a_hi = info.z, s0 = info.w;
        if (sl + stride < n_slices) info = __ldg(A.slice_row + sl + stride);     // the next slice's record
        // ---- round of loads: codes (the stream is padded beyond the last edge), row_ptr, lattice, positions
        const uint4 *cp = reinterpret_cast<const uint4 *>(A.codes + g0 + 4 * lane);
        const uint4 ca = __ldg(cp), cb = __ldg(cp + 1);
        double L[9];
        {
            const double *pl = A.lat64 + 9 * (size_t)s0;
#pragma unroll
            for (int c = 0; c < 9; ++c) L[c] = __ldg(pl + c);
        }
        // (the first 32 row_ptr entries after r0 in the same round of loads)
        long long start0 = 1ll << 62;
        if (r0 + 1 + lane <= A.n_atoms) start0 = (long long)__ldg(A.row_ptr + r0 + 1 + lane);
        __syncwarp();
        {
            const int na = min(MGWR_WIN, a_hi - a_lo);
            const double2 *px = reinterpret_cast<const double2 *>(A.pos64 + 4 * (size_t)a_lo);
            for (int a = lane; a < na; a += 32) {
                const double2 p0 = __ldg(px + 2 * a), p1 = __ldg(px + 2 * a + 1);
                xs[3 * a] = p0.x; xs[3 * a + 1] = p0.y; xs[3 * a + 2] = p1.x;
            }
        }
#pragma unroll
        for (int x = 0; x < MGS_SLICE / 32; ++x) cnt[32 * x + lane] = 0;
        __syncwarp();
        // ---- rows: row of edge p = r0 + number of rows r > r0 with row_ptr[r] <= g0 + p
        for (int rb = r0 + 1;; rb += 32) {
            const int r = rb + lane;
            long long start = start0;
            if (rb != r0 + 1) {
                start = 1ll << 62;
                if (r <= A.n_atoms) start = (long long)__ldg(A.row_ptr + r);
            }
            const bool in = start < g0 + n;
            if (in) atomicAdd(&cnt[(int)(start - g0)], 1);        // start > g0: row r0 holds g0 and r > r0
            if (!__all_sync(0xFFFFFFFFu, in)) break;
        }
        __syncwarp();
        int c4[4];
#pragma unroll
        for (int y = 0; y < 4; ++y) c4[y] = cnt[4 * lane + y];
        int incl = c4[0] + c4[1] + c4[2] + c4[3];
        const int own = incl;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        int row = r0 + incl - own;
        int gi[4], gj[4];
        unsigned tb[4];
        gj[0] = (int)ca.x; tb[0] = ca.y; gj[1] = (int)ca.z; tb[1] = ca.w;
        gj[2] = (int)cb.x; tb[2] = cb.y; gj[3] = (int)cb.z; tb[3] = cb.w;
        float v[4][3], d[4];
        const int win = min(MGWR_WIN, a_hi - a_lo);
#pragma unroll
        for (int y = 0; y < 4; ++y) {
            row += c4[y];
            gi[y] = row;
            v[y][0] = v[y][1] = v[y][2] = 0.f; d[y] = 0.f;
            if (4 * lane + y >= n) { gj[y] = row; tb[y] = 0x80808000u; continue; }
            double w3[3];
            const unsigned wi = (unsigned)(row - a_lo), wj = (unsigned)(gj[y] - a_lo);
            if (wi < (unsigned)win && wj < (unsigned)win) {
                mgwr_vec(xs + 3 * wi, xs + 3 * wj, tb[y], L, w3);
            } else {                                   // another structure, or a structure above the window
                const int s = __ldg(A.atom_struct + row);
                double L2[9], xi[3], xj[3];
#pragma unroll
                for (int c = 0; c < 9; ++c) L2[c] = __ldg(A.lat64 + 9 * (size_t)s + c);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    xi[c] = __ldg(A.pos64 + 4 * (size_t)row + c);
                    xj[c] = __ldg(A.pos64 + 4 * (size_t)gj[y] + c);
                }
                mgwr_vec(xi, xj, tb[y], L2, w3);
            }
            v[y][0] = (float)w3[0]; v[y][1] = (float)w3[1]; v[y][2] = (float)w3[2];
            if (A.dist)
                d[y] = __fsqrt_rn((float)__dadd_rn(__dadd_rn(__dmul_rn(w3[0], w3[0]), __dmul_rn(w3[1], w3[1])), __dmul_rn(w3[2], w3[2])));
        }
        // ---- stores: four edges per lane, every array in aligned 16-byte (offset: 4-byte) pieces
        const long long e = g0 + 4 * lane;
        if (al16 && 4 * lane + 4 <= n) {
            *reinterpret_cast<int4 *>(A.src + e) = make_int4(gi[0], gi[1], gi[2], gi[3]);
            *reinterpret_cast<int4 *>(A.dst + e) = make_int4(gj[0], gj[1], gj[2], gj[3]);
            float4 *pv = reinterpret_cast<float4 *>(A.vec + 3 * e);
            pv[0] = make_float4(v[0][0], v[0][1], v[0][2], v[1][0]);
            pv[1] = make_float4(v[1][1], v[1][2], v[2][0], v[2][1]);
            pv[2] = make_float4(v[2][2], v[3][0], v[3][1], v[3][2]);
            // 12 offset bytes: tau of four edges (a code's .y = b0 b1 b2 0 from the top byte down), signed
            const unsigned t0 = tb[0] ^ 0x80808000u, t1 = tb[1] ^ 0x80808000u, t2 = tb[2] ^ 0x80808000u, t3 = tb[3] ^ 0x80808000u;
            unsigned *po = reinterpret_cast<unsigned *>(A.offset + 3 * e);
            po[0] = __byte_perm(t0, t1, 0x7123);       // bytes in memory: t0.b3 t0.b2 t0.b1 t1.b3
            po[1] = __byte_perm(t1, t2, 0x6712);       //                  t1.b2 t1.b1 t2.b3 t2.b2
            po[2] = __byte_perm(t2, t3, 0x5671);       //                  t2.b1 t3.b3 t3.b2 t3.b1
            if (A.dist) *reinterpret_cast<float4 *>(A.dist + e) = make_float4(d[0], d[1], d[2], d[3]);
        } else {
#pragma unroll
            for (int y = 0; y < 4; ++y)
                if (4 * lane + y < n) {
                    A.src[e + y] = gi[y];
                    A.dst[e + y] = gj[y];
                    A.vec[3 * (e + y)] = v[y][0]; A.vec[3 * (e + y) + 1] = v[y][1]; A.vec[3 * (e + y) + 2] = v[y][2];
                    const unsigned t = tb[y] ^ 0x80808000u;
                    A.offset[3 * (e + y)] = (int8_t)(t >> 24); A.offset[3 * (e + y) + 1] = (int8_t)(t >> 16);
                    A.offset[3 * (e + y) + 2] = (int8_t)(t >> 8);
                    if (A.dist) A.dist[e + y] = d[y];
                }
        }
    }
}
