// cutoff_warp.cuh — fused cutoff-graph kernel, one autonomous WARP per task, no block barriers.
//
// One launch does distance filter (K3) -> count -> device-wide scan -> emit (K4) with batching by
// ticket (K6); SURVEY.md 8(a).  Per-structure bounds (K1) and the task split come from
// mg_prep_kernel (prep.cuh).  A task = up to 32 consecutive source rows of ONE structure, about
// MG_TASK_BUDGET candidates.  Warps take tasks in index order through an atomic ticket, so the
// decoupled look-back scan over the per-task edge totals always makes progress.  Each warp is
// software-pipelined over two stash buffers: it publishes the edge total of task A, runs the find
// phase of its next task B, and only then resolves A's output offset (by then its predecessors
// have published) and expands A — the look-back wait is hidden behind useful work.
//
//  find    stage FP32 cartesian positions p_j and the table of lattice translations T_tau in the
//          warp's shared memory; lane <-> ordered pair (row i, j); walk the table 8 cells at a
//          time (broadcast float4 loads) keeping a 32-bit hit mask in a register (d2 < hi2:
//          3 FADD, 1 FMUL, 2 FFMA, 1 FSETP, 1 LOP per candidate); append the hits as 4-byte codes
//          (tau<<6 | j) to the row's segment of the stash.  Candidates inside the FP32 rounding
//          window are decided by the exact FP64 predicate, so the edge set equals Def. 3
//           evaluated in FP64.
//  expand  one row at a time, lanes over consecutive edges: (src, dst, tau, vec, dist); vec is
//          evaluated in FP64 and rounded once.  Rows that did not fit their stash segment are
//          searched again, writing straight to global memory (rare).
#pragma once
#include "common.cuh"

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
    const unsigned *task_prefix;   // [n_struct + 1]
    unsigned long long *desc;      // [n_tasks] look-back descriptors
    unsigned *ctl;                 // [0] next task, [1] CTAs done, [6] number of tasks
    unsigned *status;
    unsigned epoch;
    int count_only;
};

struct WarpSmem {
    float4 T[MG_WT];
    float4 p[MG_SMALL_MAX_ATOMS];
    float x[MG_SMALL_MAX_ATOMS * 3];
    unsigned stash[2][MG_WS];
    int rowcnt[2][MG_TASK_ROWS];
    int rowhole[2][MG_TASK_ROWS];
    float lat[12];
};

struct Task {
    int t, s, first, natoms, i0, nr, cap, buf;
    int cnt, off;          // lane r: edges of row r, exclusive offset inside the task
    unsigned total;
    bool over;             // some row did not fit its stash segment
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

// Largest s with task_prefix[s] <= t (32-way search: three dependent loads for 32k structures).
__device__ __forceinline__ int mg_task_structure(const CutoffArgs &A, unsigned t, int lane) {
    int lo = 0, hi = A.n_struct + 1;
    while (hi - lo > 1) {
        const int step = (hi - lo + 31) / 32;
        const int idx = lo + (lane + 1) * step;
        const bool ok = idx < hi && __ldg(A.task_prefix + idx) <= t;
        lo += __popc(__ballot_sync(0xFFFFFFFFu, ok)) * step;
        hi = min(hi, lo + step);
    }
    return lo;
}

// Stage the structure of `k` in the warp's shared memory: lattice, fractional and cartesian
// positions.
__device__ __forceinline__ void mg_warp_stage(WarpSmem &sw, const CutoffArgs &A, const Task &k, int lane) {
    const float *L = A.lattice + 9 * (size_t)k.s;
    __syncwarp();
    if (lane < 9) sw.lat[lane] = L[lane];
    for (int j = lane; j < k.natoms; j += 32) {
        const float *xp = A.pos + 3 * (size_t)(k.first + j);
        const float x0 = xp[0], x1 = xp[1], x2 = xp[2];
        sw.x[3 * j] = x0; sw.x[3 * j + 1] = x1; sw.x[3 * j + 2] = x2;
        float4 p;
        p.x = __fmaf_rn(x2, L[6], __fmaf_rn(x1, L[3], __fmul_rn(x0, L[0])));
        p.y = __fmaf_rn(x2, L[7], __fmaf_rn(x1, L[4], __fmul_rn(x0, L[1])));
        p.z = __fmaf_rn(x2, L[8], __fmaf_rn(x1, L[5], __fmul_rn(x0, L[2])));
        p.w = 0.f;
        sw.p[j] = p;
    }
    __syncwarp();
}

// Translations of cells [cell0, cell0 + ncl): T = tau . L in FP32, .w = packed tau; padded to a
// `pad` entries with a far-away sentinel.
__device__ __forceinline__ void mg_warp_table(WarpSmem &sw, const int n[3], int ncell, int cell0,
                                              int ncl, int pad, int lane) {
    const int D1 = 2 * n[1] + 1, D2 = 2 * n[2] + 1;
    const float inv12 = 1.f / (float)(D1 * D2), inv2 = 1.f / (float)D2;
    const bool big = ncell >= (1 << 20);          // float reciprocal is exact below 2^20 only
    __syncwarp();
    for (int c = lane; c < pad; c += 32) {
        float4 T = make_float4(1e18f, 1e18f, 1e18f, 0.f);
        if (c < ncl) {
            const int cell = cell0 + c;
            const int u0 = big ? cell / (D1 * D2) : mg_fdiv(cell, inv12), r = cell - u0 * D1 * D2;
            const int u1 = big ? r / D2 : mg_fdiv(r, inv2);
            const int t0 = u0 - n[0], t1 = u1 - n[1], t2 = r - u1 * D2 - n[2];
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            T.x = __fmaf_rn(f2, sw.lat[6], __fmaf_rn(f1, sw.lat[3], __fmul_rn(f0, sw.lat[0])));
            T.y = __fmaf_rn(f2, sw.lat[7], __fmaf_rn(f1, sw.lat[4], __fmul_rn(f0, sw.lat[1])));
            T.z = __fmaf_rn(f2, sw.lat[8], __fmaf_rn(f1, sw.lat[5], __fmul_rn(f0, sw.lat[2])));
            T.w = __int_as_float(((t0 & 0xFF) << 16) | ((t1 & 0xFF) << 8) | (t2 & 0xFF));
        }
        sw.T[c] = T;
    }
    __syncwarp();
}

// Find phase of task t into stash buffer `buf`.  Returns the task with per-row counts scanned.
__device__ inline Task mg_warp_find(WarpSmem &sw, const CutoffArgs &A, unsigned t, int buf, int lane) {
    Task k;
    k.t = (int)t;
    k.buf = buf;
    k.s = mg_task_structure(A, t, lane);
    const StructRec *R = A.rec + k.s;
    k.first = R->first;
    k.natoms = R->natoms;
    const int rpt = R->rpt, ncell = R->ncell;
    k.cap = A.count_only ? 0 : R->cap;
    k.i0 = (int)(t - __ldg(A.task_prefix + k.s)) * rpt;
    k.nr = min(rpt, k.natoms - k.i0);
    const int n[3] = {R->n[0], R->n[1], R->n[2]};
    const float hi2 = R->hi2, lo2 = R->lo2;
    if (lane < MG_TASK_ROWS) { sw.rowcnt[buf][lane] = 0; sw.rowhole[buf][lane] = 0; }
    if (ncell > 0) {
        mg_warp_stage(sw, A, k, lane);
        const int N = k.natoms, NP = k.nr * N;
        const float inv_N = 1.f / (float)N;
        const int center = (n[0] * (2 * n[1] + 1) + n[1]) * (2 * n[2] + 1) + n[2];   // tau = 0
        unsigned *stash = sw.stash[buf];
        // lanes = P pair slots x C cell slots (P C = 32), chosen for the best lane utilisation:
        // few pairs (small N) -> more lanes along the cells.  C <= 8 keeps the table loads within
        // one shared-memory wavefront; C = 16, 32 cost 2 and 4.
        int logC = 0;
        {
            const int nc0 = min(ncell, MG_WT);
            float best = -1.f;
#pragma unroll
            for (int lc = 0; lc <= 5; ++lc) {
                const int C = 1 << lc, P = 32 >> lc;
                const int slots_p = ((NP + P - 1) / P) * P, slots_c = ((nc0 + 4 * C - 1) / (4 * C)) * (4 * C);
                float u = (float)NP * (float)nc0 / ((float)slots_p * (float)slots_c);
                if (lc == 5) u *= 0.6f;
                if (u > best) { best = u; logC = lc; }
            }
        }
        const int C = 1 << logC, P = 32 >> logC;
        const int ps = lane >> logC, cs = lane & (C - 1);
        const int npb = (NP + P - 1) / P;
        for (int cell0 = 0; cell0 < ncell; cell0 += MG_WT) {
            const int ncl = min(MG_WT, ncell - cell0);
            const int pad = ((ncl + 4 * C - 1) / (4 * C)) * (4 * C);
            mg_warp_table(sw, n, ncell, cell0, ncl, pad, lane);
            for (int pb = 0; pb < npb; ++pb) {
                const int q = pb * P + ps;
                const bool valid = q < NP;
                const int ri = valid ? mg_fdiv(q, inv_N) : 0;
                const int j = valid ? q - ri * N : 0;
                const int i = k.i0 + ri;
                float qx = 1e18f, qy = 1e18f, qz = 1e18f;
                if (valid) {
                    const float4 pi = sw.p[i], pj = sw.p[j];
                    qx = __fsub_rn(pj.x, pi.x); qy = __fsub_rn(pj.y, pi.y); qz = __fsub_rn(pj.z, pi.z);
                }
                for (int g0 = 0; g0 < pad; g0 += 32 * C) {      // this lane: cells g0 + m C + cs, m < 32
                    const float4 *Tg = sw.T + g0 + cs;
                    const int nb4 = min(32, (pad - g0) >> logC) >> 2;
                    unsigned mask = 0u;
                    for (int b4 = 0; b4 < nb4; ++b4) {
                        unsigned sub = 0u;
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const float4 T = Tg[(4 * b4 + c) << logC];
                            if (mg_d2(qx, qy, qz, T.x, T.y, T.z) < hi2) sub |= (1u << c);
                        }
                        mask |= sub << (4 * b4);
                    }
                    if (i == j) {                       // (i,i,0) is not an edge (R3)
                        const int rel = center - (cell0 + g0) - cs;
                        if (rel >= 0 && (rel & (C - 1)) == 0 && (rel >> logC) < 32) mask &= ~(1u << (rel >> logC));
                    }
                    if (mask) {
                        int rank = atomicAdd(&sw.rowcnt[buf][ri], __popc(mask));
                        unsigned *seg = stash + ri * k.cap;
                        while (mask) {
                            const int b = __ffs(mask) - 1;
                            mask &= mask - 1;
                            const float4 T = Tg[b << logC];
                            unsigned code = ((unsigned)__float_as_int(T.w) << 6) | (unsigned)j;
                            if (mg_d2(qx, qy, qz, T.x, T.y, T.z) >= lo2) {     // inside the rounding window
                                int t0, t1, t2;
                                double v[3];
                                mg_unpack_tau((unsigned)__float_as_int(T.w), t0, t1, t2);
                                const double d = mg_exact_vec(sw.x + 3 * i, sw.x + 3 * j, t0, t1, t2, sw.lat, v);
                                if (!(d < (double)A.r_c)) { code = MG_HOLE; atomicAdd(&sw.rowhole[buf][ri], 1); }
                            }
                            if (rank < k.cap) seg[rank] = code;
                            ++rank;
                        }
                    }
                }
            }
        }
    }
    __syncwarp();
    // ---- lane r: final count of row r (window rejects squeezed out), exclusive scan
    int cnt = 0;
    if (lane < k.nr) {
        const int raw = sw.rowcnt[buf][lane], holes = sw.rowhole[buf][lane];
        if (holes && raw <= k.cap) {
            unsigned *seg = sw.stash[buf] + lane * k.cap;
            int w = 0;
            for (int e = 0; e < raw; ++e) {
                const unsigned c = seg[e];
                if (c != MG_HOLE) seg[w++] = c;
            }
        }
        cnt = raw - holes;
    }
    k.cnt = cnt;
    k.over = __any_sync(0xFFFFFFFFu, cnt > k.cap);
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
    }
    k.off = incl - cnt;
    k.total = (unsigned)__shfl_sync(0xFFFFFFFFu, incl, 31);
    __syncwarp();
    return k;
}

// Decoupled look-back, resumable.  Walks back from task idx, adding the totals of predecessors
// that have published, until it meets one that holds an inclusive prefix (then done = true).  A
// predecessor that has not published yet stops the walk: blocking = false returns at once with
// the partial sum kept in (idx, sum) — the caller overlaps the wait with its next find phase —
// blocking = true spins (the predecessor is running: tickets are handed out in order).
struct LookBack { int idx; unsigned sum; bool done; };

__device__ inline void mg_warp_lookback(const CutoffArgs &A, LookBack &lb, bool blocking, int lane) {
    const unsigned ep = A.epoch & 0x3FFFFFFFu;
    while (!lb.done) {
        if (lb.idx < 0) { lb.done = true; break; }
        const int u = lb.idx - lane;
        unsigned long long d = mg_desc(MG_FLAG_PFX, ep, 0u);   // before task 0: prefix 0
        if (u >= 0) d = *(volatile const unsigned long long *)(A.desc + u);
        const bool ok = ((unsigned)(d >> 32) & 0x3FFFFFFFu) == ep && (d >> 62) != 0ull;
        const unsigned bad = __ballot_sync(0xFFFFFFFFu, !ok);
        const unsigned pfx = __ballot_sync(0xFFFFFFFFu, ok && (d >> 62) == MG_FLAG_PFX);
        const int first_bad = bad ? __ffs(bad) - 1 : 32, first_pfx = pfx ? __ffs(pfx) - 1 : 32;
        // lanes nearer than the first unpublished predecessor count, up to the nearest prefix
        const int take = first_pfx < first_bad ? first_pfx + 1 : first_bad;
        unsigned val = lane < take ? (unsigned)d : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xFFFFFFFFu, val, o);
        lb.sum += val;
        lb.idx -= take;
        if (first_pfx < first_bad) { lb.done = true; break; }
        if (first_bad < 32) {
            if (!blocking) return;
            __nanosleep(200);
        }
    }
}

// Write one edge: vec = rho (x_j + tau - x_i) in FP64 (fused multiply-adds), rounded once.
__device__ __forceinline__ void mg_emit_edge(const CutoffArgs &A, long long e, int gi, int gj,
                                             const double xi[3], const double L[9], int t0, int t1, int t2) {
    if (e >= A.capacity) return;
    const float *xj = A.pos + 3 * (size_t)gj;
    const double f0 = ((double)xj[0] - xi[0]) + (double)t0;
    const double f1 = ((double)xj[1] - xi[1]) + (double)t1;
    const double f2 = ((double)xj[2] - xi[2]) + (double)t2;
    const double v0 = fma(f2, L[6], fma(f1, L[3], f0 * L[0]));
    const double v1 = fma(f2, L[7], fma(f1, L[4], f0 * L[1]));
    const double v2 = fma(f2, L[8], fma(f1, L[5], f0 * L[2]));
    A.src[e] = gi;
    A.dst[e] = gj;
    A.offset[3 * e] = (int8_t)t0; A.offset[3 * e + 1] = (int8_t)t1; A.offset[3 * e + 2] = (int8_t)t2;
    A.vec[3 * e] = (float)v0; A.vec[3 * e + 1] = (float)v1; A.vec[3 * e + 2] = (float)v2;
    if (A.dist) A.dist[e] = sqrtf((float)fma(v2, v2, fma(v1, v1, v0 * v0)));
}

// Rows of task k whose stash segment overflowed: search again, lanes over the cells of the
// current table tile, loop over j, writing straight to global memory (rare path).
__device__ inline void mg_warp_research(WarpSmem &sw, const CutoffArgs &A, const Task &k, long long base,
                                        const double L[9], int lane) {
    const StructRec *R = A.rec + k.s;
    const int n[3] = {R->n[0], R->n[1], R->n[2]};
    const int ncell = R->ncell, N = k.natoms;
    const float hi2 = R->hi2, lo2 = R->lo2;
    const int center = (n[0] * (2 * n[1] + 1) + n[1]) * (2 * n[2] + 1) + n[2];
    mg_warp_stage(sw, A, k, lane);
    int cur = 0;                                          // lane r: edges of row r written so far
    for (int cell0 = 0; cell0 < ncell; cell0 += MG_WT) {
        const int ncl = min(MG_WT, ncell - cell0), pad = (ncl + 31) & ~31;
        mg_warp_table(sw, n, ncell, cell0, ncl, pad, lane);
        for (int r = 0; r < k.nr; ++r) {
            if (__shfl_sync(0xFFFFFFFFu, k.cnt, r) <= k.cap) continue;
            const int i = k.i0 + r;
            const float4 pi = sw.p[i];
            const double xi[3] = {(double)sw.x[3 * i], (double)sw.x[3 * i + 1], (double)sw.x[3 * i + 2]};
            const long long g0 = base + __shfl_sync(0xFFFFFFFFu, k.off, r);
            int done = __shfl_sync(0xFFFFFFFFu, cur, r);
            for (int c0 = 0; c0 < pad; c0 += 32) {
                const int c = c0 + lane;
                const float4 T = sw.T[c];
                int t0, t1, t2;
                mg_unpack_tau((unsigned)__float_as_int(T.w), t0, t1, t2);
                for (int j = 0; j < N; ++j) {
                    const float4 pj = sw.p[j];
                    const float d2 = mg_d2(__fsub_rn(pj.x, pi.x), __fsub_rn(pj.y, pi.y),
                                           __fsub_rn(pj.z, pi.z), T.x, T.y, T.z);
                    bool hit = d2 < hi2 && !(i == j && cell0 + c == center);
                    if (hit && d2 >= lo2) {
                        double v[3];
                        hit = mg_exact_vec(sw.x + 3 * i, sw.x + 3 * j, t0, t1, t2, sw.lat, v) < (double)A.r_c;
                    }
                    const unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
                    if (hit) mg_emit_edge(A, g0 + done + __popc(m & ((1u << lane) - 1u)), k.first + i,
                                          k.first + j, xi, L, t0, t1, t2);
                    done += __popc(m);
                }
            }
            if (lane == r) cur = done;
        }
    }
}

// Task k's output offset is known: publish its prefix, write row_ptr, expand.
__device__ inline void mg_warp_finish(WarpSmem &sw, const CutoffArgs &A, const Task &k, unsigned base32,
                                      int n_tasks, int lane) {
    const unsigned ep = A.epoch & 0x3FFFFFFFu;
    if (lane == 0) {
        *(volatile unsigned long long *)(A.desc + k.t) = mg_desc(MG_FLAG_PFX, ep, base32 + k.total);
        if ((unsigned long long)base32 + k.total > 0x7FFFFFFFull) atomicOr(A.status, MGS_CAPACITY);
    }
    const long long base = base32;
    if (lane < k.nr) A.row_ptr[k.first + k.i0 + lane] = (int)(base + k.off);
    if (k.t == n_tasks - 1 && lane == 0) {
        const long long tot = base + k.total;
        A.row_ptr[A.n_atoms] = (int)tot;
        *A.n_edges = tot;
        if (!A.count_only && tot > A.capacity) atomicOr(A.status, MGS_CAPACITY);
    }
    if (A.count_only || k.total == 0u) return;
    const float *Lf = A.lattice + 9 * (size_t)k.s;
    double L[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) L[c] = (double)Lf[c];
    const unsigned *stash = sw.stash[k.buf];
    for (int r = 0; r < k.nr; ++r) {
        const int cnt = __shfl_sync(0xFFFFFFFFu, k.cnt, r);
        if (cnt > k.cap) continue;
        const int gi = k.first + k.i0 + r;
        const float *xp = A.pos + 3 * (size_t)gi;
        const double xi[3] = {(double)xp[0], (double)xp[1], (double)xp[2]};
        const long long g0 = base + __shfl_sync(0xFFFFFFFFu, k.off, r);
        const unsigned *seg = stash + r * k.cap;
        for (int e = lane; e < cnt; e += 32) {
            const unsigned code = seg[e];
            int t0, t1, t2;
            mg_unpack_tau(code >> 6, t0, t1, t2);
            mg_emit_edge(A, g0 + e, gi, k.first + (int)(code & 63u), xi, L, t0, t1, t2);
        }
    }
    if (k.over) mg_warp_research(sw, A, k, base, L, lane);
}

__global__ void __launch_bounds__(MG_BLOCK)
mg_cutoff_warp_kernel(const CutoffArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpSmem &sw = reinterpret_cast<WarpSmem *>(smem_raw)[warp];
    const int n_tasks = (int)*(volatile unsigned *)(A.ctl + 6);
    const unsigned ep = A.epoch & 0x3FFFFFFFu;
    Task pend;
    LookBack plb;
    bool have_pend = false;
    for (;;) {
        unsigned t = 0u;
        if (lane == 0) t = atomicAdd(A.ctl, 1u);
        t = __shfl_sync(0xFFFFFFFFu, t, 0);
        const bool have_cur = t < (unsigned)n_tasks;
        Task cur;
        LookBack clb;
        if (have_cur) {
            cur = mg_warp_find(sw, A, t, have_pend ? 1 - pend.buf : 0, lane);
            // publish the total right away: successors can look back through this task
            if (lane == 0)
                *(volatile unsigned long long *)(A.desc + t) = mg_desc(t ? MG_FLAG_AGG : MG_FLAG_PFX, ep, cur.total);
            clb.idx = (int)t - 1; clb.sum = 0u; clb.done = false;
        }
        if (have_pend) {                                   // its predecessors had a whole find phase
            mg_warp_lookback(A, plb, true, lane);
            mg_warp_finish(sw, A, pend, plb.sum, n_tasks, lane);
            have_pend = false;
        }
        if (!have_cur) break;
        mg_warp_lookback(A, clb, false, lane);
        if (clb.done) {
            mg_warp_finish(sw, A, cur, clb.sum, n_tasks, lane);
        } else {                                           // somebody before us is still searching:
            pend = cur; plb = clb; have_pend = true;       // keep the stash, go on with the next task
        }
    }
    // last CTA out resets the ticket for the next launch
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(A.ctl + 1, 1u) == gridDim.x - 1) { A.ctl[0] = 0u; A.ctl[1] = 0u; }
    }
}
