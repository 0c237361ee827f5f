// cut_fused.cuh — cutoff graph (K3 distance filter, K4 count -> device-wide scan -> emit, K6 batching,
// SURVEY.md 8(a)) in ONE launch of co-resident CTAs.
//
// mg_cut_prep_kernel gives every ordered pair (i, j) an estimated cost; CTA b owns the source rows
// whose first pair lies in the b-th of gridDim.x equally expensive, contiguous ranges of the batch's
// pairs in (structure, i, j) order — which is the CSR order of the output.  A CTA walks its rows
// twice:
//
//   count   per structure: stage the wrapped positions and the table of local translations in shared
//           memory (once per CTA, not once per warp), then blocks of 32 ordered pairs, one block per
//           warp: lane <-> pair, FP32 filter over the pair's sub-box (cut_prep.cuh; FP64 decision
//           inside the rounding window, R23).  The 32-bit hit masks and the hits of every
//           block go to the CTA's scratch in global memory (L2 resident).
//   scan    the CTA publishes its edge total in a slot tagged with the call's epoch and sums the
//           slots of the CTAs before it (all CTAs are resident: cooperative launch): the device-wide
//           exclusive scan of K4 without a second launch, without re-staging and without a look-back
//           chain — every lane polls its own slots.
//   emit    the same walk: masks read back, hits compacted into a shared-memory stash in (row, j, t)
//           order, chunk by chunk (<= 4 blocks, <= MGF_STASH edges), row_ptr from the running offset;
//           then LANES <-> EDGES: vec = (p_j - p_i + l . L) + t . L in FP64 (the pair's part once per
//           pair, the table's part from an FP64 table), rounded once (R24).  src / dst leave as
//           coalesced 4-byte stores; vec and offset are staged per warp in shared memory with the
//           misalignment of their global address and leave as aligned 16-byte stores (scalar stores
//           only for the ragged head / tail of a warp's 128 edges).
//
// Structures the pair-lane path does not take (more than MG_SMALL_MAX_ATOMS atoms, a sub-box of more
// than MGF_TLOC cells) go row by row through mg_rows_* below: lanes over the candidates (j, t) of one
// source row, ballot compaction, no table — exact and general, not tuned.
#pragma once
#include "common.cuh"
#include "cut_prep.cuh"
#include "cutoff_pairs.cuh"

#define MGF_BLOCK 128
#define MGF_WARPS (MGF_BLOCK / 32)
#define MGF_TLOC MG_TLOC           // cells of the shared-memory table (= WarpSmem)
#define MGF_STASH 1024             // edges per chunk
#define MGF_CHUNK 4                // blocks of 32 pairs per chunk: one per warp
#define MGF_MASK_WORDS 16384       // 32-bit words of scratch per CTA (hit masks + block totals)

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
    int mask_words;                // words of a CTA's scratch that may be used (tests: less)
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

struct FusedSmem {
    WarpSmem w;                        // table planes, tcode, wrapped positions (one structure)
    double Td[3][MGF_TLOC];            // t . L in FP64 (emit)
    double pd[3][MG_SMALL_MAX_ATOMS];  // x . L in FP64, coordinates as given (emit)
    unsigned stash[MGF_STASH];         // (pair of the chunk) << 8 | cell
    double pb[3][32 * MGF_CHUNK];      // per pair of the chunk: p_j - p_i + l . L
    unsigned plc[32 * MGF_CHUNK];      // (l + 128) bytes << 8
    unsigned pij[32 * MGF_CHUNK];      // i | j << 16
    float sv[MGF_WARPS][128 * 3 + 4];  // per warp: vec of 128 edges, shifted by the global misalignment
    unsigned char sb[MGF_WARPS][128 * 3 + 16];
    unsigned wsum[MGF_WARPS];
    unsigned long long prefix;
    int last;
};

// ---- staging of one structure (all threads of the CTA) -------------------------------------------
// Returns false (for every thread) if a coordinate is non-finite or too far from the cell.
template <bool EMIT>
__device__ __forceinline__ bool mgf_stage(FusedSmem &sm, const FusedArgs &A, const CutRec *R, int s, Task &k,
                                          FindCtx &F) {
    const int tid = threadIdx.x;
    k.s = s;
    k.first = R->first;
    k.natoms = R->natoms;
    F.lat = A.lattice + 9 * (size_t)s;
    F.pos = A.pos;
    F.rc = A.r_c;
    F.mloc = R->mloc;
    F.m = R->m;
#pragma unroll
    for (int c = 0; c < 9; ++c) F.a[c] = __ldg(F.lat + c);
#pragma unroll
    for (int a = 0; a < 3; ++a) F.rho[a] = R->rho[a];
    F.nr2 = -__fmul_rn(A.r_c, A.r_c);
    F.win = 1.1920929e-7f * (2.f * A.r_c * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * A.r_c * A.r_c);
    F.gx = A.pos + 3 * (size_t)k.first;
    F.big = false;
    __syncthreads();                               // the previous structure's readers are done
    bool ok = true;
    for (int j = tid; j < k.natoms; j += MGF_BLOCK) {
        const float *xp = F.gx + 3 * j;
        const float4 xw = mg_wrap_x(xp);
        ok = ok && __float_as_int(xw.w) != 0;
        sm.w.x[j] = xw;
        if (EMIT) {
            const double d0 = (double)xp[0], d1 = (double)xp[1], d2 = (double)xp[2];
            sm.pd[0][j] = fma(d2, (double)F.a[6], fma(d1, (double)F.a[3], d0 * (double)F.a[0]));
            sm.pd[1][j] = fma(d2, (double)F.a[7], fma(d1, (double)F.a[4], d0 * (double)F.a[1]));
            sm.pd[2][j] = fma(d2, (double)F.a[8], fma(d1, (double)F.a[5], d0 * (double)F.a[2]));
        }
    }
    {   // table of local translations t . L, t in [0, m): cells [0, mloc), sentinel up to a multiple of 32
        const int m1 = (F.m >> 8) & 0xFF, m2 = (F.m >> 16) & 0xFF, M12 = m1 * m2;
        const float inv12 = 1.f / (float)M12, inv2 = 1.f / (float)m2;
        float *tp = reinterpret_cast<float *>(sm.w.T);
        const int pad = (F.mloc + 31) & ~31;
        for (int c = tid; c < pad; c += MGF_BLOCK) {
            float Tx = 1e18f, Ty = 1e18f, Tz = 1e18f;
            unsigned code = 0u;
            if (c < F.mloc) {
                const int t0 = mg_fdiv(c, inv12), r = c - t0 * M12;
                const int t1 = mg_fdiv(r, inv2), t2 = r - t1 * m2;
                const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
                Tx = __fmaf_rn(f2, F.a[6], __fmaf_rn(f1, F.a[3], __fmul_rn(f0, F.a[0])));
                Ty = __fmaf_rn(f2, F.a[7], __fmaf_rn(f1, F.a[4], __fmul_rn(f0, F.a[1])));
                Tz = __fmaf_rn(f2, F.a[8], __fmaf_rn(f1, F.a[5], __fmul_rn(f0, F.a[2])));
                code = ((unsigned)t0 << 24) | ((unsigned)t1 << 16) | ((unsigned)t2 << 8);
                if (EMIT) {            // exact: small integers times FP32 values, three terms
                    const double g0 = (double)t0, g1 = (double)t1, g2 = (double)t2;
                    sm.Td[0][c] = fma(g2, (double)F.a[6], fma(g1, (double)F.a[3], g0 * (double)F.a[0]));
                    sm.Td[1][c] = fma(g2, (double)F.a[7], fma(g1, (double)F.a[4], g0 * (double)F.a[1]));
                    sm.Td[2][c] = fma(g2, (double)F.a[8], fma(g1, (double)F.a[5], g0 * (double)F.a[2]));
                }
            }
            tp[c] = Tx; tp[MG_TLOC + c] = Ty; tp[2 * MG_TLOC + c] = Tz;
            sm.w.tcode[c] = code;
        }
    }
    ok = __syncthreads_and(ok) != 0;
    if (!ok && tid == 0) atomicOr(A.status, MGS_NONFINITE);
    return ok;
}

// ---- generic rows: any structure size, any sub-box (not tuned) -----------------------------------
// One warp per source row, lanes over the candidates f = j * mloc + c of the row.  For the pair
// (i, j): u = x_j - x_i (wrapped coordinates), the sub-box starts at lo_a = floor(-rho_a - u_a) + 1;
// cell c = (t0 m1 + t1) m2 + t2; d2 = |(u + lo + t) . L|^2 in FP32, FP64 decision inside the window.
struct RowsCtx {
    float a[9];
    float rho[3];
    int m0, m1, m2, mloc;
    float nr2, win, rc;
    const float *gx;       // positions of the structure's first atom
    const float *lat;
    int first, N;
};

__device__ __forceinline__ void mgf_rows_setup(RowsCtx &C, const FusedArgs &A, const CutRec *R, int s) {
    C.lat = A.lattice + 9 * (size_t)s;
#pragma unroll
    for (int c = 0; c < 9; ++c) C.a[c] = __ldg(C.lat + c);
#pragma unroll
    for (int a = 0; a < 3; ++a) C.rho[a] = R->rho[a];
    C.m0 = R->m & 0xFF; C.m1 = (R->m >> 8) & 0xFF; C.m2 = (R->m >> 16) & 0xFF;
    C.mloc = R->mloc;
    C.rc = A.r_c;
    C.nr2 = -__fmul_rn(A.r_c, A.r_c);
    C.win = 1.1920929e-7f * (2.f * A.r_c * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * A.r_c * A.r_c);
    C.first = R->first;
    C.N = R->natoms;
    C.gx = A.pos + 3 * (size_t)R->first;
}

// Candidate f of row i: hit?  tau (absolute, relative to the coordinates as given) in t[3].
__device__ __forceinline__ bool mgf_rows_eval(const RowsCtx &C, const FusedArgs &A, const float4 xi, int i,
                                              long long f, int &j, int t[3], bool &bad) {
    j = C.mloc == 1 ? (int)f : (int)(f / C.mloc);
    const int c = (int)(f - (long long)j * C.mloc);
    const int M12 = C.m1 * C.m2;
    const int t0 = c / M12, r = c - t0 * M12, t1 = r / C.m2, t2 = r - t1 * C.m2;
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
    t[0] = (int)e0 + t0 + (ki & 1023) - (kj & 1023);
    t[1] = (int)e1 + t1 + ((ki >> 10) & 1023) - ((kj >> 10) & 1023);
    t[2] = (int)e2 + t2 + ((ki >> 20) & 1023) - ((kj >> 20) & 1023);
    bad = ki == 0 || kj == 0 || t[0] < -127 || t[1] < -127 || t[2] < -127 || t[0] > 127 || t[1] > 127 || t[2] > 127;
    if (bad) return false;
    if (i == j && (t[0] | t[1] | t[2]) == 0) return false;          // (i, i, 0) is not an edge (R3)
    bool hit = y < C.win;
    if (fabsf(y) < C.win) {                                          // FP32 cannot decide: Def. 3 in FP64
        double v[3];
        hit = mg_exact_vec(C.gx + 3 * i, C.gx + 3 * j, t[0], t[1], t[2], C.lat, v) < (double)C.rc;
    }
    return hit;
}

// Count the edges of rows [ia, ib) of structure s: warp w of the CTA takes rows ia + w, ia + w + 4, ...
// Row totals go to the scratch (one word per row) when keep.
__device__ __forceinline__ unsigned mgf_rows_count(const FusedArgs &A, const CutRec *R, int s, int ia, int ib,
                                                   unsigned *wm, int midx, int mask_words) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    RowsCtx C;
    mgf_rows_setup(C, A, R, s);
    unsigned total = 0u;
    for (int i = ia + warp; i < ib; i += MGF_WARPS) {
        const float4 xi = mg_wrap_x(C.gx + 3 * i);
        const long long nf = (long long)C.N * C.mloc;
        unsigned cnt = 0u;
        bool anybad = false;
        for (long long f0 = 0; f0 < nf; f0 += 32) {
            const long long f = f0 + lane;
            int j, t[3];
            bool bad = false;
            const bool hit = f < nf && mgf_rows_eval(C, A, xi, i, f, j, t, bad);
            anybad = anybad || (f < nf && bad);
            cnt += __popc(__ballot_sync(0xFFFFFFFFu, hit));
        }
        if (anybad) atomicOr(A.status, __float_as_int(xi.w) == 0 ? MGS_NONFINITE : MGS_OFFSET);
        if (lane == 0 && midx + (i - ia) < mask_words) wm[midx + (i - ia)] = cnt;
        total += cnt;
    }
    return total;                                  // the same on every lane of the warp
}

__device__ __forceinline__ void mgf_emit_one(const FusedArgs &A, long long e, int gi, int gj, const float *gx, int i,
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

// Emit rows [ia, ib): goff = global index of the first edge of row ia.  Returns the edges written.
// Row totals come from the scratch (or are counted again when it was exhausted).
__device__ __forceinline__ unsigned mgf_rows_emit(FusedSmem &sm, const FusedArgs &A, const CutRec *R, int s, int ia,
                                                  int ib, const unsigned *wm, int midx, int mask_words,
                                                  long long goff) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    RowsCtx C;
    mgf_rows_setup(C, A, R, s);
    const long long nf = (long long)C.N * C.mloc;
    unsigned done = 0u;
    // groups of MGF_WARPS rows: warp w emits row i0 + w after the rows before it in the group
    for (int i0 = ia; i0 < ib; i0 += MGF_WARPS) {
        const int i = i0 + warp;
        unsigned cnt = 0u;
        float4 xi = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i < ib) {
            xi = mg_wrap_x(C.gx + 3 * i);
            if (midx + (i - ia) < mask_words) cnt = __ldcg(wm + midx + (i - ia));
            else
                for (long long f0 = 0; f0 < nf; f0 += 32) {
                    int j, t[3];
                    bool bad;
                    const bool hit = f0 + lane < nf && mgf_rows_eval(C, A, xi, i, f0 + lane, j, t, bad);
                    cnt += __popc(__ballot_sync(0xFFFFFFFFu, hit));
                }
        }
        __syncthreads();
        if (lane == 0) sm.wsum[warp] = cnt;
        __syncthreads();
        unsigned before = 0u, group = 0u;
#pragma unroll
        for (int w = 0; w < MGF_WARPS; ++w) {
            if (w < warp) before += sm.wsum[w];
            group += sm.wsum[w];
        }
        if (i < ib) {
            long long e = goff + done + before;
            if (lane == 0) A.row_ptr[C.first + i] = (int)e;
            for (long long f0 = 0; f0 < nf; f0 += 32) {
                int j = 0, t[3] = {0, 0, 0};
                bool bad;
                const bool hit = f0 + lane < nf && mgf_rows_eval(C, A, xi, i, f0 + lane, j, t, bad);
                const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
                if (hit) mgf_emit_one(A, e + __popc(bal & ((1u << lane) - 1u)), C.first + i, C.first + j, C.gx, i, j, t, C.lat);
                e += __popc(bal);
            }
        }
        done += group;
    }
    return done;
}

// ---- stash -> global ----------------------------------------------------------------------------------
// Edges [0, n) of the stash are the edges [goff, goff + n) of the output.  Warp w takes the batches
// w, w + 4, ... of 128 edges: lane <-> edge (four rounds), src / dst / dist as coalesced 4-byte
// stores, vec and offset staged in the warp's shared memory at the misalignment of their global
// address and written as aligned 16-byte pieces (scalar stores for a ragged first / last piece).
__device__ __forceinline__ void mgf_flush(FusedSmem &sm, const FusedArgs &A, int first, long long goff, int n) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long room = A.capacity - goff;
    const int lim = room >= n ? n : (room > 0 ? (int)room : 0);    // edges that fit the caller's arrays
    float *sv = sm.sv[warp];
    unsigned char *sb = sm.sb[warp];
    const bool vec16 = (reinterpret_cast<unsigned long long>(A.vec) & 15ull) == 0ull;
    const bool off16 = (reinterpret_cast<unsigned long long>(A.offset) & 15ull) == 0ull;
    for (int e0 = 128 * warp; e0 < lim; e0 += 128 * MGF_WARPS) {
        const int nb = min(128, lim - e0);
        const long long E0 = goff + e0;                 // global index of the batch's first edge
        const long long F0 = 3 * E0, F1 = F0 + 3 * nb;  // floats of vec = bytes of offset
        const int shv = (int)(F0 & 3), shb = (int)(F0 & 15);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int x = 32 * r + lane;
            if (x < nb) {
                const unsigned code = sm.stash[e0 + x];
                const int pidx = (int)(code >> 8), t = (int)(code & 0xFFu);
                const double v0 = sm.pb[0][pidx] + sm.Td[0][t];
                const double v1 = sm.pb[1][pidx] + sm.Td[1][t];
                const double v2 = sm.pb[2][pidx] + sm.Td[2][t];
                const unsigned tb = (sm.plc[pidx] + sm.w.tcode[t]) ^ 0x80808000u;   // tau bytes as int8
                const unsigned ij = sm.pij[pidx];
                A.src[E0 + x] = first + (int)(ij & 0xFFFFu);
                A.dst[E0 + x] = first + (int)(ij >> 16);
                if (A.dist) A.dist[E0 + x] = __fsqrt_rn((float)fma(v2, v2, fma(v1, v1, v0 * v0)));
                sv[3 * x + shv] = (float)v0; sv[3 * x + shv + 1] = (float)v1; sv[3 * x + shv + 2] = (float)v2;
                sb[3 * x + shb] = (unsigned char)(tb >> 24); sb[3 * x + shb + 1] = (unsigned char)(tb >> 16);
                sb[3 * x + shb + 2] = (unsigned char)(tb >> 8);
            }
        }
        __syncwarp();
        {   // vec: 16-byte pieces of [F0, F1); piece c holds the floats Fb + 4 c .. + 3
            const long long Fb = F0 - shv;
            const int np = (shv + 3 * nb + 3) >> 2;
            for (int c = lane; c < np; c += 32) {
                const long long g = Fb + 4 * c;
                if (vec16 && g >= F0 && g + 4 <= F1) {
                    *reinterpret_cast<float4 *>(A.vec + g) = *reinterpret_cast<const float4 *>(sv + 4 * c);
                } else {
#pragma unroll
                    for (int y = 0; y < 4; ++y)
                        if (g + y >= F0 && g + y < F1) A.vec[g + y] = sv[4 * c + y];
                }
            }
        }
        {   // offset: 16-byte pieces of the bytes [F0, F1)
            const long long Bb = F0 - shb;
            const int np = (shb + 3 * nb + 15) >> 4;
            for (int c = lane; c < np; c += 32) {
                const long long g = Bb + 16 * c;
                if (off16 && g >= F0 && g + 16 <= F1) {
                    *reinterpret_cast<uint4 *>(A.offset + g) = *reinterpret_cast<const uint4 *>(sb + 16 * c);
                } else {
#pragma unroll
                    for (int y = 0; y < 16; ++y)
                        if (g + y >= F0 && g + y < F1) A.offset[g + y] = (int8_t)sb[16 * c + y];
                }
            }
        }
        __syncwarp();
    }
}

// ---- the walk of a CTA over its rows ---------------------------------------------------------------
// PHASE 0: count (returns the CTA's edges, the same value on every thread); PHASE 1: emit from goff.
template <int PHASE>
__device__ __forceinline__ unsigned long long mgf_walk(FusedSmem &sm, const FusedArgs &A, const RangeCtx &RC,
                                                       unsigned *wm, unsigned long long goff) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long c0, c1;
    mg_warp_range(RC, blockIdx.x, c0, c1);
    int s, qa;
    mg_range_start(RC, c0, s, qa, lane);
    int midx = 0;
    unsigned wtotal = 0u;                          // PHASE 0: hits of this warp's blocks (lane 0 meaningful... all lanes equal)
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
                    for (int i = ia + tid; i < ib; i += MGF_BLOCK) A.row_ptr[R->first + i] = (int)goff;
            } else if (N > MG_SMALL_MAX_ATOMS || mloc > MGF_TLOC) {
                bool ok = true;                    // a structure with a non-finite coordinate emits nothing (R26)
                for (int j = tid; j < N; j += MGF_BLOCK)
                    ok = ok && __float_as_int(mg_wrap_x(A.pos + 3 * (size_t)(R->first + j)).w) != 0;
                ok = __syncthreads_and(ok) != 0;
                if (!ok) {
                    if (tid == 0) atomicOr(A.status, MGS_NONFINITE);
                    if (PHASE == 1)
                        for (int i = ia + tid; i < ib; i += MGF_BLOCK) A.row_ptr[R->first + i] = (int)goff;
                } else if (PHASE == 0) {
                    wtotal += mgf_rows_count(A, R, s, ia, ib, wm, midx, A.mask_words);
                } else {
                    goff += mgf_rows_emit(sm, A, R, s, ia, ib, wm, midx, A.mask_words, (long long)goff);
                }
                midx += ib - ia;
            } else {
                Task k;
                FindCtx F;
                const bool live = mgf_stage<PHASE == 1>(sm, A, R, s, k, F);
                const int nW = (mloc + 31) >> 5, recw = 32 * nW + 32;
                const int q0 = ia * N, q1 = ib * N, nblk = (q1 - q0 + 31) >> 5;
                const float inv_N = 1.f / (float)N;
                if (!live) {
                    if (PHASE == 1)
                        for (int i = ia + tid; i < ib; i += MGF_BLOCK) A.row_ptr[k.first + i] = (int)goff;
                } else if (PHASE == 0) {
                    for (int b = warp; b < nblk; b += MGF_WARPS) {
                        const int q = q0 + 32 * b + lane;
                        const bool valid = q < q1;
                        int i = 0, j = 0;
                        if (valid) mg_qsplit(q, N, inv_N, i, j);
                        const PairLane p = mg_pair_setup(sm.w, F, valid, i, j);
                        if (valid && !p.ok) atomicOr(A.status, MGS_OFFSET);
                        const int base = midx + b * recw;
                        const bool keep = base + recw <= A.mask_words;
                        unsigned cnt = 0u;
#pragma unroll 1
                        for (int w = 0; w < nW; ++w) {
                            const unsigned m = mg_word_mask(sm.w, F, p, k.first + i, k.first + j, 0, w, mloc);
                            cnt += __popc(m);
                            if (keep) wm[base + 32 * w + lane] = m;
                        }
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xFFFFFFFFu, cnt, o);
                        if (keep && lane == 0) wm[base + 32 * nW] = cnt;
                        wtotal += cnt;
                    }
                } else {
                    double Ld[9];
#pragma unroll
                    for (int c = 0; c < 9; ++c) Ld[c] = (double)F.a[c];
                    // chunks: runs of <= MGF_CHUNK blocks with <= MGF_STASH hits; a block with more hits (or
                    // whose masks did not fit the scratch) goes alone, in passes of consecutive lanes
                    for (int b0 = 0; b0 < nblk;) {
                        // block totals of the next MGF_CHUNK blocks (lane x: block b0 + x)
                        unsigned bt = 0u;
                        bool have = false;
                        if (lane < MGF_CHUNK && b0 + lane < nblk) {
                            const int base = midx + (b0 + lane) * recw;
                            have = base + recw <= A.mask_words;
                            if (have) bt = __ldcg(wm + base + 32 * nW);
                        }
                        const unsigned havem = __ballot_sync(0xFFFFFFFFu, have);
                        int nb = 0;
                        unsigned boff[MGF_CHUNK + 1];
                        boff[0] = 0u;
#pragma unroll
                        for (int x = 0; x < MGF_CHUNK; ++x) {
                            const unsigned v = __shfl_sync(0xFFFFFFFFu, bt, x);
                            boff[x + 1] = boff[x] + v;
                            if (nb == x && ((havem >> x) & 1u) && boff[x + 1] <= MGF_STASH) nb = x + 1;
                        }
                        if (nb > 0) {
                            // ---- fast chunk: warp x extracts block b0 + x
                            unsigned chunk_total = 0u;
#pragma unroll
                            for (int x = 0; x < MGF_CHUNK; ++x)
                                if (x < nb) chunk_total = boff[x + 1];
                            __syncthreads();                   // stash / pair records of the previous chunk are flushed
                            if (warp < nb) {
                                const int b = b0 + warp;
                                const int q = q0 + 32 * b + lane;
                                const bool valid = q < q1;
                                int i = 0, j = 0;
                                if (valid) mg_qsplit(q, N, inv_N, i, j);
                                const PairLane p = mg_pair_setup(sm.w, F, valid, i, j);
                                const unsigned *mp = wm + midx + b * recw + lane;
                                unsigned cnt = 0u;
#pragma unroll 1
                                for (int w = 0; w < nW; ++w) cnt += __popc(__ldcg(mp + 32 * w));
                                unsigned incl = cnt;
#pragma unroll
                                for (int o = 1; o < 32; o <<= 1) {
                                    const unsigned v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                                    if (lane >= o) incl += v;
                                }
                                unsigned mybase = 0u;
#pragma unroll
                                for (int x = 0; x < MGF_CHUNK; ++x)
                                    if (x == warp) mybase = boff[x];
                                unsigned pos = mybase + incl - cnt;
                                if (valid && j == 0) A.row_ptr[k.first + i] = (int)(goff + pos);
                                const int pidx = 32 * warp + lane;
                                if (valid) {
                                    const double l0 = (double)p.l0, l1 = (double)p.l1, l2 = (double)p.l2;
                                    sm.pb[0][pidx] = fma(l2, Ld[6], fma(l1, Ld[3], fma(l0, Ld[0], sm.pd[0][j] - sm.pd[0][i])));
                                    sm.pb[1][pidx] = fma(l2, Ld[7], fma(l1, Ld[4], fma(l0, Ld[1], sm.pd[1][j] - sm.pd[1][i])));
                                    sm.pb[2][pidx] = fma(l2, Ld[8], fma(l1, Ld[5], fma(l0, Ld[2], sm.pd[2][j] - sm.pd[2][i])));
                                    sm.plc[pidx] = ((unsigned)(p.l0 + 128) << 24) | ((unsigned)(p.l1 + 128) << 16) |
                                                   ((unsigned)(p.l2 + 128) << 8);
                                    sm.pij[pidx] = (unsigned)i | ((unsigned)j << 16);
                                }
                                const unsigned pc = (unsigned)pidx << 8;
#pragma unroll 1
                                for (int w = 0; w < nW; ++w) {
                                    unsigned mk = __ldcg(mp + 32 * w);
                                    while (mk) {
                                        const int bit = __ffs(mk) - 1;
                                        mk &= mk - 1;
                                        sm.stash[pos++] = pc | (unsigned)(32 * w + bit);
                                    }
                                }
                            }
                            __syncthreads();
                            mgf_flush(sm, A, k.first, (long long)goff, (int)chunk_total);
                            goff += chunk_total;
                            b0 += nb;
                        } else {
                            // ---- slow block: every warp evaluates / loads the masks of block b0, warp 0 extracts
                            // passes of consecutive lanes that fit the stash
                            const int b = b0;
                            const int q = q0 + 32 * b + lane;
                            const bool valid = q < q1;
                            int i = 0, j = 0;
                            if (valid) mg_qsplit(q, N, inv_N, i, j);
                            const PairLane p = mg_pair_setup(sm.w, F, valid, i, j);
                            const bool haveb = (havem & 1u) != 0u;
                            const unsigned *mp = wm + midx + b * recw + lane;
                            unsigned cnt = 0u;
#pragma unroll 1
                            for (int w = 0; w < nW; ++w)
                                cnt += __popc(haveb ? __ldcg(mp + 32 * w)
                                                    : mg_word_mask(sm.w, F, p, k.first + i, k.first + j, 0, w, mloc));
                            unsigned incl = cnt;
#pragma unroll
                            for (int o = 1; o < 32; o <<= 1) {
                                const unsigned v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
                                if (lane >= o) incl += v;
                            }
                            const unsigned tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
                            if (warp == 0 && valid && j == 0) A.row_ptr[k.first + i] = (int)(goff + incl - cnt);
                            unsigned done = 0u;
                            int l0 = 0;
                            while (l0 < 32) {
                                const bool mine = lane >= l0 && incl - done <= MGF_STASH;
                                const int nl = __popc(__ballot_sync(0xFFFFFFFFu, mine));   // >= 1: a lane has <= 256 hits
                                const unsigned t = __shfl_sync(0xFFFFFFFFu, incl, l0 + nl - 1) - done;
                                __syncthreads();
                                if (warp == 0 && mine) {
                                    unsigned pos = incl - cnt - done;
                                    const int pidx = lane;
                                    if (valid) {
                                        const double d0 = (double)p.l0, d1 = (double)p.l1, d2 = (double)p.l2;
                                        sm.pb[0][pidx] = fma(d2, Ld[6], fma(d1, Ld[3], fma(d0, Ld[0], sm.pd[0][j] - sm.pd[0][i])));
                                        sm.pb[1][pidx] = fma(d2, Ld[7], fma(d1, Ld[4], fma(d0, Ld[1], sm.pd[1][j] - sm.pd[1][i])));
                                        sm.pb[2][pidx] = fma(d2, Ld[8], fma(d1, Ld[5], fma(d0, Ld[2], sm.pd[2][j] - sm.pd[2][i])));
                                        sm.plc[pidx] = ((unsigned)(p.l0 + 128) << 24) | ((unsigned)(p.l1 + 128) << 16) |
                                                       ((unsigned)(p.l2 + 128) << 8);
                                        sm.pij[pidx] = (unsigned)i | ((unsigned)j << 16);
                                    }
#pragma unroll 1
                                    for (int w = 0; w < nW; ++w) {
                                        unsigned mk = haveb ? __ldcg(mp + 32 * w)
                                                            : mg_word_mask(sm.w, F, p, k.first + i, k.first + j, 0, w, mloc);
                                        while (mk) {
                                            const int bit = __ffs(mk) - 1;
                                            mk &= mk - 1;
                                            sm.stash[pos++] = ((unsigned)pidx << 8) | (unsigned)(32 * w + bit);
                                        }
                                    }
                                }
                                __syncthreads();
                                mgf_flush(sm, A, k.first, (long long)goff, (int)t);
                                goff += t;
                                done += t;
                                l0 += nl;
                            }
                            (void)tot;
                            b0 += 1;
                        }
                    }
                }
                midx += nblk * recw;
            }
        }
        if (!more) break;
    }
    if (PHASE == 1) return goff;
    // CTA total: every warp counted its own blocks (all lanes hold the warp's sum)
    __syncthreads();
    if (lane == 0) sm.wsum[warp] = wtotal;
    __syncthreads();
    unsigned long long total = 0ull;
#pragma unroll
    for (int w = 0; w < MGF_WARPS; ++w) total += sm.wsum[w];
    return total;
}

// ---- the kernel ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(MGF_BLOCK)
mg_cutoff_fused_kernel(const __grid_constant__ FusedArgs A) {
    mg_grid_dependency_wait();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    FusedSmem &sm = *reinterpret_cast<FusedSmem *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned epoch = *reinterpret_cast<volatile unsigned *>(A.ctl + 10) + 1u;   // tag of this call's slots
    RangeCtx RC;
    mg_range_init(RC, A.rec, A.bpre, A.n_blocks, A.n_struct, (int)gridDim.x, lane);
    unsigned *wm = A.wmask + (size_t)blockIdx.x * MGF_MASK_WORDS;
    MGF_STAMP(0)
    const unsigned long long total = mgf_walk<0>(sm, A, RC, wm, 0ull);
    MGF_STAMP(1)
    if (tid == 0) mg_st_release(A.slots + blockIdx.x, ((unsigned long long)epoch << 32) | (total & 0xFFFFFFFFull));
    unsigned long long before = 0ull;
    if (!A.count_only) {
        // device-wide exclusive scan of K4: sum of the slots before this CTA's (all CTAs are resident)
        if (warp == 0) {
            for (int c0 = 0; c0 < (int)blockIdx.x; c0 += 32) {
                const int c = c0 + lane;
                if (c < (int)blockIdx.x) {
                    unsigned long long v;
                    do { v = mg_ld_acquire(A.slots + c); } while ((unsigned)(v >> 32) != epoch);
                    before += v & 0xFFFFFFFFull;
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) before += __shfl_xor_sync(0xFFFFFFFFu, before, o);
            if (lane == 0) sm.prefix = before;
        }
        __syncthreads();
        before = sm.prefix;
        MGF_STAMP(2)
        if (blockIdx.x == gridDim.x - 1 && tid == 0) {           // the last range knows the grand total
            const unsigned long long tot = before + total;
            *A.n_edges = (long long)tot;
            A.row_ptr[A.n_atoms] = (int)tot;
            if (tot > 0x7FFFFFFFull || (long long)tot > A.capacity) atomicOr(A.status, MGS_CAPACITY);
        }
        mgf_walk<1>(sm, A, RC, wm, before);
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
