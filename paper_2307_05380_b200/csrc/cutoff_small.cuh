// cutoff_small.cuh — fused cutoff-graph kernel for structures of <= MG_SMALL_MAX_ATOMS atoms.
//
// One launch does distance filter (K3) -> count -> device-wide scan -> emit (K4) with batching by
// ticket (K6); SURVEY.md 8(a).  The per-structure bounds (K1) come from mg_prep_kernel (prep.cuh).
// Unit of scheduling ("chunk") = a contiguous range of source rows (atoms) holding about
// MG_CHUNK_COST candidates; it may split a heavy structure by rows and may span several light ones
// ("segments").  Chunks are taken in index order through an atomic ticket so that the decoupled
// look-back scan over the per-chunk edge totals always makes progress.
//
//  per segment  stage FP32 cartesian positions p_j; build the table of lattice translations T_tau
//           in shared memory; find: lane <-> ordered pair (i,j), the warp walks the table 32 cells
//           at a time (broadcast float4 loads) keeping a 32-bit hit mask in a register
//           (d2 < hi2: 3 FADD, 1 FMUL, 2 FFMA, 1 FSETP, 1 LOP per candidate), then appends the
//           hits as 4-byte codes (tau<<6 | j) to the row's segment of the shared-memory stash.
//           Candidates inside the FP32 rounding window are decided by the exact FP64 predicate, so
//           the edge set equals Def. 3 evaluated in FP64.
//  per chunk    row counts -> exclusive scan -> chunk total -> decoupled look-back -> base; row_ptr;
//           expand: one warp per row turns codes into (src, dst, tau, vec, dist); vec is the FP64
//           value rounded once.  Rows that did not fit their stash segment are searched again.
#pragma once
#include "common.cuh"

#define MG_TCAP 1024          // translation-table tile (cells)
#define MG_SCAP 4096          // stash entries per CTA
#define MG_HOLE 0xFFFFFFFFu

struct CutoffArgs {
    const float *pos;
    const float *lattice;
    const int32_t *struct_ptr;
    int n_struct, n_atoms;
    float r_c;
    int32_t *row_ptr, *src, *dst;
    int8_t *offset;
    float *vec, *dist;
    long long capacity;
    long long *n_edges;
    const StructRec *rec;
    const unsigned long long *cost_prefix;   // [n_struct + 1]
    unsigned long long *desc;   // [max chunks] look-back descriptors
    unsigned *ctl;              // [0] next chunk, [1] CTAs done, [6] number of chunks
    unsigned *status;
    unsigned epoch;
    int count_only;
};

struct CutoffSmem {
    float4 T[MG_TCAP];
    unsigned stash[MG_SCAP];
    float4 p[MG_SMALL_MAX_ATOMS];
    StructRec rec;                       // current segment
    float lat[9];
    int rowcnt[MG_MAX_ROWS], rowhole[MG_MAX_ROWS], rowoff[MG_MAX_ROWS + 1], rowcur[MG_MAX_ROWS];
    int rowseg[MG_MAX_ROWS], rowcap[MG_MAX_ROWS];
    int seg_s[MG_MAX_SEGS], seg_i0[MG_MAX_SEGS], seg_i1[MG_MAX_SEGS], seg_row0[MG_MAX_SEGS];
    int nseg, nrows, chunk, first_atom, any_over;
    unsigned base, total;
};

__device__ __forceinline__ void mg_unpack_tau(unsigned u, int &t0, int &t1, int &t2) {
    t0 = (int)(signed char)((u >> 16) & 0xFFu);
    t1 = (int)(signed char)((u >> 8) & 0xFFu);
    t2 = (int)(signed char)(u & 0xFFu);
}

// q / n for 0 <= q < 2^20, 1 <= n (exact: (q + 0.5) / n is never within rounding of an integer)
__device__ __forceinline__ int mg_fdiv(int q, float inv_n) {
    return __float2int_rz(__fmul_rn((float)q + 0.5f, inv_n));
}

// Warp 0: which rows does chunk k own?  Rows are laid out on a cost axis: row i of structure s
// starts at P[s] + i * rowcost_s; chunk k owns the starts in [k B, (k+1) B).
__device__ inline void mg_cutoff_segments(CutoffSmem &sm, const CutoffArgs &A, int k) {
    const int lane = threadIdx.x;
    const unsigned long long w0 = (unsigned long long)k * MG_CHUNK_COST, w1 = w0 + MG_CHUNK_COST;
    const unsigned long long *P = A.cost_prefix;
    int lo = 0, hi = A.n_struct + 1;              // largest s with P[s] <= w0
    while (hi - lo > 1) {
        const int step = (hi - lo + 31) / 32;
        const int idx = lo + (lane + 1) * step;
        const bool ok = idx < hi && __ldg(P + idx) <= w0;
        const int cnt = __popc(__ballot_sync(0xFFFFFFFFu, ok));
        lo += cnt * step;
        hi = min(hi, lo + step);
    }
    int nseg = 0, nrows = 0, first_atom = 0;
    for (int s0 = lo; s0 < A.n_struct; s0 += 32) {
        const int s = s0 + lane;
        unsigned long long Ps = ~0ull;
        int i0 = 0, i1 = 0, fa = 0;
        if (s < A.n_struct) {
            Ps = __ldg(P + s);
            const unsigned rc = A.rec[s].rowcost;
            const int N = A.rec[s].natoms;
            if (N > 0 && Ps < w1) {
                const unsigned long long span = (unsigned long long)N * rc;
                i0 = N;
                if (Ps >= w0) i0 = 0;
                else if (w0 - Ps < span) i0 = (int)(((unsigned)(w0 - Ps) + rc - 1u) / rc);
                i1 = N;
                if (w1 - Ps < span) i1 = (int)(((unsigned)(w1 - Ps) + rc - 1u) / rc);
                fa = A.rec[s].first + i0;
            }
        }
        const bool has = i0 < i1;
        const unsigned m = __ballot_sync(0xFFFFFFFFu, has);
        const int cnt = has ? i1 - i0 : 0;
        int incl = cnt;                                // inclusive scan of the row counts
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += t;
        }
        if (has) {
            const int slot = nseg + __popc(m & ((1u << lane) - 1u));
            if (slot < MG_MAX_SEGS) {
                sm.seg_s[slot] = s; sm.seg_i0[slot] = i0; sm.seg_i1[slot] = i1;
                sm.seg_row0[slot] = nrows + incl - cnt;
            }
        }
        if (nseg == 0 && m) first_atom = __shfl_sync(0xFFFFFFFFu, fa, __ffs(m) - 1);
        nseg += __popc(m);
        nrows += __shfl_sync(0xFFFFFFFFu, incl, 31);
        const unsigned long long Plast = __shfl_sync(0xFFFFFFFFu, Ps, 31);
        if (Plast >= w1) break;                       // also ends the loop past the last structure
    }
    if (lane == 0) {
        sm.nseg = min(nseg, MG_MAX_SEGS);
        sm.nrows = min(nrows, MG_MAX_ROWS);
        sm.first_atom = first_atom;
        sm.any_over = 0;
    }
}

// Stage segment g: record, lattice, FP32 cartesian positions; carve the rows' stash segments.
// `top` (next free stash entry) is carried in a register, identical in every thread.
__device__ inline void mg_cutoff_stage(CutoffSmem &sm, const CutoffArgs &A, int g, int &top, bool carve) {
    const int tid = threadIdx.x;
    const int s = sm.seg_s[g];
    if (tid < 32) reinterpret_cast<int *>(&sm.rec)[tid] = reinterpret_cast<const int *>(A.rec + s)[tid];
    if (tid >= 32 && tid < 41) sm.lat[tid - 32] = A.lattice[9 * (size_t)s + (tid - 32)];
    const StructRec *R = A.rec + s;
    const int N = R->natoms, first = R->first;
    if (tid >= 64 && tid - 64 < N) {
        const int j = tid - 64;
        const float *L = A.lattice + 9 * (size_t)s;
        const float x0 = A.pos[3 * (size_t)(first + j)], x1 = A.pos[3 * (size_t)(first + j) + 1],
                    x2 = A.pos[3 * (size_t)(first + j) + 2];
        float4 p;
        p.x = __fmaf_rn(x2, L[6], __fmaf_rn(x1, L[3], __fmul_rn(x0, L[0])));
        p.y = __fmaf_rn(x2, L[7], __fmaf_rn(x1, L[4], __fmul_rn(x0, L[1])));
        p.z = __fmaf_rn(x2, L[8], __fmaf_rn(x1, L[5], __fmul_rn(x0, L[2])));
        p.w = 0.f;
        sm.p[j] = p;
    }
    // expected row length lambda = N (4/3) pi r_c^3 / V, plus slack; whatever is left if short
    const int nr = sm.seg_i1[g] - sm.seg_i0[g], row0 = sm.seg_row0[g];
    int cap = 0;
    if (!A.count_only && R->ncell > 0) {
        const float lam = (float)N * 4.18879f * A.r_c * A.r_c * A.r_c / R->volume;
        cap = (int)(1.25f * lam) + 32;
        if (cap * nr > MG_SCAP - top) cap = (MG_SCAP - top) / nr;
    }
    if (carve && tid < nr && row0 + tid < MG_MAX_ROWS) {
        sm.rowseg[row0 + tid] = top + tid * cap;
        sm.rowcap[row0 + tid] = cap;
    }
    top += nr * cap;
}

// Table of translations for cells [cell0, cell0 + MG_TCAP) of the staged segment: T = tau . L in
// FP32, .w = packed tau; the padding up to a multiple of 32 is a far-away sentinel.
__device__ inline void mg_build_table(CutoffSmem &sm, int cell0) {
    const StructRec &g = sm.rec;
    const int D1 = 2 * g.n[1] + 1, D2 = 2 * g.n[2] + 1;
    const float inv12 = 1.f / (float)(D1 * D2), inv2 = 1.f / (float)D2;
    int ncl = g.ncell - cell0;
    if (ncl > MG_TCAP) ncl = MG_TCAP;
    const int padded = (ncl + 31) & ~31;
    for (int c = threadIdx.x; c < padded; c += MG_BLOCK) {
        float4 T = make_float4(1e18f, 1e18f, 1e18f, 0.f);
        if (c < ncl) {
            const int cell = cell0 + c;
            const bool big = g.ncell >= (1 << 20);          // float reciprocal is exact below 2^20 only
            const int u0 = big ? cell / (D1 * D2) : mg_fdiv(cell, inv12), r = cell - u0 * D1 * D2;
            const int u1 = big ? r / D2 : mg_fdiv(r, inv2);
            const int t0 = u0 - g.n[0], t1 = u1 - g.n[1], t2 = r - u1 * D2 - g.n[2];
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            T.x = __fmaf_rn(f2, sm.lat[6], __fmaf_rn(f1, sm.lat[3], __fmul_rn(f0, sm.lat[0])));
            T.y = __fmaf_rn(f2, sm.lat[7], __fmaf_rn(f1, sm.lat[4], __fmul_rn(f0, sm.lat[1])));
            T.z = __fmaf_rn(f2, sm.lat[8], __fmaf_rn(f1, sm.lat[5], __fmul_rn(f0, sm.lat[2])));
            T.w = __int_as_float(((t0 & 0xFF) << 16) | ((t1 & 0xFF) << 8) | (t2 & 0xFF));
        }
        sm.T[c] = T;
    }
}

// Find for the table tile starting at cell0 (already built, block-synchronised), segment g.
__device__ inline void mg_cutoff_find(CutoffSmem &sm, const CutoffArgs &A, int g, int cell0) {
    const StructRec &R = sm.rec;
    const int N = R.natoms, i0 = sm.seg_i0[g], row0 = sm.seg_row0[g];
    const int NP = (sm.seg_i1[g] - i0) * N;            // ordered pairs (row, j) of this segment
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int ncl = R.ncell - cell0;
    if (ncl > MG_TCAP) ncl = MG_TCAP;
    const int ncg = (ncl + 31) >> 5;
    const int npb = (NP + 31) >> 5;
    const int items = npb * ncg;
    const float inv_ncg = 1.f / (float)ncg, inv_N = 1.f / (float)N;
    const int center = (R.n[0] * (2 * R.n[1] + 1) + R.n[1]) * (2 * R.n[2] + 1) + R.n[2];   // tau = 0
    const float hi2 = R.hi2, lo2 = R.lo2;
    const float *xs = A.pos + 3 * (size_t)R.first;
    for (int item = warp; item < items; item += MG_WARPS) {
        const int pb = mg_fdiv(item, inv_ncg), cg = item - pb * ncg;
        const int q = pb * 32 + lane;
        const bool valid = q < NP;
        const int ri = valid ? mg_fdiv(q, inv_N) : 0;
        const int j = valid ? q - ri * N : 0;
        const int i = i0 + ri;
        float qx = 1e18f, qy = 1e18f, qz = 1e18f;
        if (valid) {
            const float4 pi = sm.p[i], pj = sm.p[j];
            qx = __fsub_rn(pj.x, pi.x); qy = __fsub_rn(pj.y, pi.y); qz = __fsub_rn(pj.z, pi.z);
        }
        const float4 *Tg = sm.T + cg * 32;
        unsigned mask = 0u;
#pragma unroll
        for (int c = 0; c < 32; ++c) {
            const float4 T = Tg[c];
            if (mg_d2(qx, qy, qz, T.x, T.y, T.z) < hi2) mask |= (1u << c);
        }
        if (i == j) {                       // (i,i,0) is not an edge (R3)
            const int rel = center - (cell0 + cg * 32);
            if (rel >= 0 && rel < 32) mask &= ~(1u << rel);
        }
        if (mask) {
            const int row = row0 + ri;
            int rank = atomicAdd(&sm.rowcnt[row], __popc(mask));
            const int cap = sm.rowcap[row];
            unsigned *seg = sm.stash + sm.rowseg[row];
            while (mask) {
                const int b = __ffs(mask) - 1;
                mask &= mask - 1;
                const float4 T = Tg[b];
                unsigned code = ((unsigned)__float_as_int(T.w) << 6) | (unsigned)j;
                if (mg_d2(qx, qy, qz, T.x, T.y, T.z) >= lo2) {     // inside the rounding window
                    int t0, t1, t2;
                    double v[3];
                    mg_unpack_tau((unsigned)__float_as_int(T.w), t0, t1, t2);
                    const double d = mg_exact_vec(xs + 3 * i, xs + 3 * j, t0, t1, t2, sm.lat, v);
                    if (!(d < (double)A.r_c)) { code = MG_HOLE; atomicAdd(&sm.rowhole[row], 1); }
                }
                if (rank < cap) seg[rank] = code;
                ++rank;
            }
        }
    }
}

// Remove the (rare) window rejects from the stash rows and correct the counts.
__device__ inline void mg_cutoff_fix_holes(CutoffSmem &sm) {
    const int r = threadIdx.x;
    if (r < sm.nrows) {
        const int holes = sm.rowhole[r], cnt = sm.rowcnt[r], cap = sm.rowcap[r];
        if (holes) {
            if (cnt <= cap) {
                unsigned *seg = sm.stash + sm.rowseg[r];
                int w = 0;
                for (int e = 0; e < cnt; ++e) {
                    const unsigned c = seg[e];
                    if (c != MG_HOLE) seg[w++] = c;
                }
            }
            sm.rowcnt[r] = cnt - holes;
        }
        if (cnt - holes > cap) sm.any_over = 1;   // benign race: all writers store 1
    }
}

// Exclusive scan of the <= 64 row counts (warp 0), look-back over the chunk totals.
__device__ inline void mg_cutoff_scan_lookback(CutoffSmem &sm, const CutoffArgs &A) {
    const int lane = threadIdx.x;     // called by warp 0 only
    const int nr = sm.nrows, k = sm.chunk;
    const int v0 = lane < nr ? sm.rowcnt[lane] : 0;
    const int v1 = lane + 32 < nr ? sm.rowcnt[lane + 32] : 0;
    int s0 = v0, s1 = v1;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t0 = __shfl_up_sync(0xFFFFFFFFu, s0, o), t1 = __shfl_up_sync(0xFFFFFFFFu, s1, o);
        if (lane >= o) { s0 += t0; s1 += t1; }
    }
    const int tot0 = __shfl_sync(0xFFFFFFFFu, s0, 31);
    const unsigned total = (unsigned)(tot0 + __shfl_sync(0xFFFFFFFFu, s1, 31));
    sm.rowoff[lane] = s0 - v0;
    sm.rowoff[lane + 32] = tot0 + s1 - v1;
    if (lane == 0) sm.rowoff[MG_MAX_ROWS] = (int)total;
    unsigned base = 0u;
    const unsigned ep = A.epoch & 0x3FFFFFFFu;
    if (k > 0) {
        if (lane == 0) *(volatile unsigned long long *)(A.desc + k) = mg_desc(MG_FLAG_AGG, ep, total);
        int idx = k - 1;
        for (;;) {
            const int t = idx - lane;
            unsigned long long d = mg_desc(MG_FLAG_PFX, ep, 0u);   // before chunk 0: prefix 0
            for (;;) {
                if (t >= 0) d = *(volatile const unsigned long long *)(A.desc + t);
                const bool ok = ((unsigned)(d >> 32) & 0x3FFFFFFFu) == ep && (d >> 62) != 0ull;
                if (__all_sync(0xFFFFFFFFu, ok)) break;
                __nanosleep(64);
            }
            const unsigned pfx = __ballot_sync(0xFFFFFFFFu, (d >> 62) == MG_FLAG_PFX);
            const int stop = pfx ? __ffs(pfx) - 1 : 31;       // nearest predecessor holding a prefix
            unsigned val = lane <= stop ? (unsigned)d : 0u;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xFFFFFFFFu, val, o);
            base += val;
            if (pfx) break;
            idx -= 32;
        }
    }
    if (lane == 0) {
        *(volatile unsigned long long *)(A.desc + k) = mg_desc(MG_FLAG_PFX, ep, base + total);
        sm.base = base;
        sm.total = total;
        if ((unsigned long long)base + total > 0x7FFFFFFFull) atomicOr(A.status, MGS_CAPACITY);
    }
}

// Write one edge.  vec / dist are the FP64 values of Def. 3 rounded once to FP32.
__device__ __forceinline__ void mg_emit_edge(const CutoffArgs &A, long long e, int gi, int gj,
                                             const float *lat9, int t0, int t1, int t2) {
    if (e >= A.capacity) return;
    double v[3];
    const double d = mg_exact_vec(A.pos + 3 * (size_t)gi, A.pos + 3 * (size_t)gj, t0, t1, t2, lat9, v);
    A.src[e] = gi;
    A.dst[e] = gj;
    A.offset[3 * e] = (int8_t)t0; A.offset[3 * e + 1] = (int8_t)t1; A.offset[3 * e + 2] = (int8_t)t2;
    A.vec[3 * e] = (float)v[0]; A.vec[3 * e + 1] = (float)v[1]; A.vec[3 * e + 2] = (float)v[2];
    if (A.dist) A.dist[e] = (float)d;
}

__device__ __forceinline__ int mg_row_segment(const CutoffSmem &sm, int r) {
    int g = 0;
    for (int t = 1; t < sm.nseg; ++t) g = (r >= sm.seg_row0[t]) ? t : g;
    return g;
}

// Expand the rows that fit their stash segment: one warp per row, lanes over consecutive edges.
__device__ inline void mg_cutoff_expand(CutoffSmem &sm, const CutoffArgs &A) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int r = warp; r < sm.nrows; r += MG_WARPS) {
        const int cnt = sm.rowcnt[r];
        if (cnt > sm.rowcap[r]) continue;
        const int s = sm.seg_s[mg_row_segment(sm, r)];
        const int first = A.rec[s].first;
        const float *lat9 = A.lattice + 9 * (size_t)s;
        const long long g0 = (long long)sm.base + sm.rowoff[r];
        const unsigned *seg = sm.stash + sm.rowseg[r];
        for (int e = lane; e < cnt; e += 32) {
            const unsigned code = seg[e];
            int t0, t1, t2;
            mg_unpack_tau(code >> 6, t0, t1, t2);
            mg_emit_edge(A, g0 + e, sm.first_atom + r, first + (int)(code & 63u), lat9, t0, t1, t2);
        }
    }
}

// Rows of the staged segment g whose stash segment overflowed: search again, warp per row, lanes
// over the cells of the current table tile, writing straight to global memory (rare path).
__device__ inline void mg_cutoff_research(CutoffSmem &sm, const CutoffArgs &A, int g, int cell0) {
    const StructRec &R = sm.rec;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int N = R.natoms, i0 = sm.seg_i0[g], row0 = sm.seg_row0[g], nr = sm.seg_i1[g] - i0;
    int ncl = R.ncell - cell0;
    if (ncl > MG_TCAP) ncl = MG_TCAP;
    const int center = (R.n[0] * (2 * R.n[1] + 1) + R.n[1]) * (2 * R.n[2] + 1) + R.n[2];
    const float *xs = A.pos + 3 * (size_t)R.first;
    for (int ri = warp; ri < nr; ri += MG_WARPS) {
        const int row = row0 + ri, i = i0 + ri;
        if (sm.rowcnt[row] <= sm.rowcap[row]) continue;
        const float4 pi = sm.p[i];
        int cur = sm.rowcur[row];
        const long long g0 = (long long)sm.base + sm.rowoff[row];
        for (int c = lane; c < ((ncl + 31) & ~31); c += 32) {
            const float4 T = sm.T[c];
            int t0, t1, t2;
            mg_unpack_tau((unsigned)__float_as_int(T.w), t0, t1, t2);
            for (int j = 0; j < N; ++j) {
                const float4 pj = sm.p[j];
                const float d2 = mg_d2(__fsub_rn(pj.x, pi.x), __fsub_rn(pj.y, pi.y),
                                       __fsub_rn(pj.z, pi.z), T.x, T.y, T.z);
                bool hit = d2 < R.hi2 && !(i == j && cell0 + c == center);
                if (hit && d2 >= R.lo2) {
                    double v[3];
                    hit = mg_exact_vec(xs + 3 * i, xs + 3 * j, t0, t1, t2, sm.lat, v) < (double)A.r_c;
                }
                const unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
                if (hit) mg_emit_edge(A, g0 + cur + __popc(m & ((1u << lane) - 1u)), R.first + i,
                                      R.first + j, sm.lat, t0, t1, t2);
                cur += __popc(m);
            }
        }
        if (lane == 0) sm.rowcur[row] = cur;
    }
}

__global__ void __launch_bounds__(MG_BLOCK)
mg_cutoff_small_kernel(const CutoffArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CutoffSmem &sm = *reinterpret_cast<CutoffSmem *>(smem_raw);
    const int tid = threadIdx.x;
    const int n_chunks = (int)*(volatile unsigned *)(A.ctl + 6);
    for (;;) {
        __syncthreads();                               // previous chunk fully retired
        if (tid == 0) sm.chunk = (int)atomicAdd(A.ctl, 1u);
        if (tid < MG_MAX_ROWS) { sm.rowcnt[tid] = 0; sm.rowhole[tid] = 0; sm.rowcur[tid] = 0; sm.rowcap[tid] = 0; }
        __syncthreads();
        const int k = sm.chunk;
        if (k >= n_chunks) break;
        if (tid < 32) mg_cutoff_segments(sm, A, k);
        __syncthreads();
        const int nseg = sm.nseg;
        int top = 0;
        // ---- find, segment by segment
        for (int g = 0; g < nseg; ++g) {
            if (g) __syncthreads();
            mg_cutoff_stage(sm, A, g, top, true);
            __syncthreads();
            const int ncell = sm.rec.ncell;
            for (int cell0 = 0; cell0 < ncell; cell0 += MG_TCAP) {
                if (cell0) __syncthreads();
                mg_build_table(sm, cell0);
                __syncthreads();
                mg_cutoff_find(sm, A, g, cell0);
            }
        }
        __syncthreads();
        mg_cutoff_fix_holes(sm);
        __syncthreads();
        // ---- scan + look-back, row_ptr
        if (tid < 32) mg_cutoff_scan_lookback(sm, A);
        __syncthreads();
        const long long base = sm.base;
        if (tid < sm.nrows) A.row_ptr[sm.first_atom + tid] = (int)(base + sm.rowoff[tid]);
        if (k == n_chunks - 1 && tid == 0) {
            const long long tot = base + sm.total;
            A.row_ptr[A.n_atoms] = (int)tot;
            *A.n_edges = tot;
            if (!A.count_only && tot > A.capacity) atomicOr(A.status, MGS_CAPACITY);
        }
        if (A.count_only) continue;
        // ---- expand
        mg_cutoff_expand(sm, A);
        if (sm.any_over) {
            for (int g = 0; g < nseg; ++g) {
                bool over = false;
                for (int r = sm.seg_row0[g]; r < sm.seg_row0[g] + sm.seg_i1[g] - sm.seg_i0[g]; ++r)
                    over = over || sm.rowcnt[r] > sm.rowcap[r];
                if (!over) continue;
                int dummy = 0;
                __syncthreads();
                mg_cutoff_stage(sm, A, g, dummy, false);
                __syncthreads();
                const int ncell = sm.rec.ncell;
                for (int cell0 = 0; cell0 < ncell; cell0 += MG_TCAP) {
                    if (cell0) __syncthreads();
                    mg_build_table(sm, cell0);
                    __syncthreads();
                    mg_cutoff_research(sm, A, g, cell0);
                }
            }
        }
    }
    // last CTA out resets the ticket for the next launch
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(A.ctl + 1, 1u) == gridDim.x - 1) { A.ctl[0] = 0u; A.ctl[1] = 0u; }
    }
}
