// cutoff_small.cuh — fused cutoff-graph kernel for structures of <= MG_SMALL_MAX_ATOMS atoms.
//
// One launch does bounds (K1) -> distance filter (K3) -> count -> device-wide scan -> emit (K4)
// with batching by ticket (K6); SURVEY.md 8(a).  Unit of scheduling ("chunk") = one structure,
// taken in index order through an atomic ticket so that the decoupled look-back scan over the
// per-chunk edge totals always makes progress.
//
//  phase 0  stage lattice + fractional positions in shared memory, FP64 plane spacings,
//           n_a = floor(r_c/h_a + spread_a) (<= ceil(r_c/h_a) for x in [0,1), R14),
//           FP32 cartesian positions p_j, rounding window [lo2, hi2) of the FP32 filter.
//  phase 1  find: lane <-> ordered pair (i,j); the warp walks the table of lattice translations
//           T_tau (shared memory, broadcast float4 loads) 32 cells at a time, keeps a 32-bit hit
//           mask in a register (d2 < hi2: 3 FADD, 1 FMUL, 2 FFMA, 1 FSETP, 1 LOP per candidate),
//           then appends the hits as 4-byte codes (cell<<6 | j) to the row segment of source i in
//           the shared-memory stash.  Candidates inside the rounding window are decided by the
//           exact FP64 predicate, so the edge set equals Def. 3 evaluated in FP64.
//  phase 2  row counts -> exclusive scan -> chunk total -> decoupled look-back -> base; row_ptr.
//  phase 3  expand: one warp per row turns codes into (src, dst, tau, vec, dist); vec is the FP64
//           value rounded once.  Rows that did not fit their stash segment are re-searched.
#pragma once
#include "common.cuh"

#define MG_TCAP 1024          // translation-table tile (cells)
#define MG_SCAP 8192          // stash entries per CTA
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
    unsigned long long *desc;   // [n_struct] look-back descriptors
    unsigned *ticket;           // [0] next chunk, [1] CTAs done
    unsigned *status;
    unsigned epoch;
    int count_only;
};

struct CutoffSmem {
    float4 T[MG_TCAP];
    unsigned stash[MG_SCAP];
    float4 p[MG_SMALL_MAX_ATOMS];
    float x[MG_SMALL_MAX_ATOMS * 3];
    int rowcnt[MG_SMALL_MAX_ATOMS];
    int rowhole[MG_SMALL_MAX_ATOMS];
    int rowoff[MG_SMALL_MAX_ATOMS + 1];
    int rowcur[MG_SMALL_MAX_ATOMS];
    float lat[9];
    StructGeom g;
    int chunk, first, natoms, cap, any_over;
    unsigned base, total;
};

__device__ __forceinline__ void mg_decode_cell(int cell, const int dim[3], const int n[3], int &t0,
                                               int &t1, int &t2) {
    const int d12 = dim[1] * dim[2];
    const int c0 = cell / d12;
    const int r = cell - c0 * d12;
    const int c1 = r / dim[2];
    t0 = c0 - n[0];
    t1 = c1 - n[1];
    t2 = r - c1 * dim[2] - n[2];
}

// Phase 0 for one structure: geometry + window.  Runs on one thread; positions are already in sm.x.
__device__ inline void mg_cutoff_geometry(CutoffSmem &sm, float r_c) {
    StructGeom &g = sm.g;
    const int N = sm.natoms;
    double vol, h[3];
    g.err = mg_cell_spacings(sm.lat, &vol, h);
    g.ncell = 0;
    if (g.err) return;
    double M = 0.0;
    bool finite = true;
    for (int a = 0; a < 3; ++a) {
        float lo = 0.f, hi = 0.f, xabs = 1.f;
        for (int i = 0; i < N; ++i) {
            const float v = sm.x[3 * i + a];
            finite = finite && isfinite(v);
            lo = (i == 0) ? v : fminf(lo, v);
            hi = (i == 0) ? v : fmaxf(hi, v);
            xabs = fmaxf(xabs, fabsf(v));
        }
        const double spread = (double)hi - (double)lo;
        const double nn = floor((double)r_c / h[a] * (1.0 + 1e-9) + spread);
        if (!(nn <= 127.0)) { g.err = finite ? MGS_OFFSET : MGS_NONFINITE; return; }
        g.n[a] = (int)nn;
        g.dim[a] = 2 * g.n[a] + 1;
        g.h[a] = (float)h[a];
        g.a[a][0] = sm.lat[3 * a]; g.a[a][1] = sm.lat[3 * a + 1]; g.a[a][2] = sm.lat[3 * a + 2];
        const double amax = fmax(fabs((double)sm.lat[3 * a]),
                                 fmax(fabs((double)sm.lat[3 * a + 1]), fabs((double)sm.lat[3 * a + 2])));
        M += (nn + 2.0 * (double)xabs) * amax;
    }
    if (!finite) { g.err = MGS_NONFINITE; return; }
    // every FP32 rounding in p_j, p_i, q = p_j - p_i, T_tau and q + T is <= 2^-24 * M; 12 of them
    // per component
    const double e_comp = 12.0 * 5.9604644775390625e-8 * M;
    const double W = 3.5 * e_comp + 2e-6 * (double)r_c;
    const double lo = (double)r_c - W, hi = (double)r_c + W;
    g.lo2 = lo > 0.0 ? __double2float_rd(lo * lo * (1.0 - 1e-6)) : 0.f;
    g.hi2 = __double2float_ru(hi * hi * (1.0 + 1e-6));
    g.volume = (float)vol;
    g.ncell = g.dim[0] * g.dim[1] * g.dim[2];
}

// Build the translation table for cells [cell0, cell0 + MG_TCAP): T = tau . L in FP32, .w = packed
// tau; the padding up to a multiple of 32 is a far-away sentinel.
__device__ inline void mg_build_table(CutoffSmem &sm, int cell0) {
    const StructGeom &g = sm.g;
    int ncl = g.ncell - cell0;
    if (ncl > MG_TCAP) ncl = MG_TCAP;
    const int padded = (ncl + 31) & ~31;
    for (int c = threadIdx.x; c < padded; c += MG_BLOCK) {
        float4 T;
        if (c < ncl) {
            int t0, t1, t2;
            mg_decode_cell(cell0 + c, g.dim, g.n, t0, t1, t2);
            const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
            T.x = __fmaf_rn(f2, g.a[2][0], __fmaf_rn(f1, g.a[1][0], __fmul_rn(f0, g.a[0][0])));
            T.y = __fmaf_rn(f2, g.a[2][1], __fmaf_rn(f1, g.a[1][1], __fmul_rn(f0, g.a[0][1])));
            T.z = __fmaf_rn(f2, g.a[2][2], __fmaf_rn(f1, g.a[1][2], __fmul_rn(f0, g.a[0][2])));
            T.w = __int_as_float(((t0 & 0xFF) << 16) | ((t1 & 0xFF) << 8) | (t2 & 0xFF));
        } else {
            T = make_float4(1e18f, 1e18f, 1e18f, 0.f);
        }
        sm.T[c] = T;
    }
}

__device__ __forceinline__ void mg_unpack_tau(float w, int &t0, int &t1, int &t2) {
    const int u = __float_as_int(w);
    t0 = (int)(signed char)((u >> 16) & 0xFF);
    t1 = (int)(signed char)((u >> 8) & 0xFF);
    t2 = (int)(signed char)(u & 0xFF);
}

// Phase 1 for the table tile starting at cell0 (already built, block-synchronised).
__device__ inline void mg_cutoff_find(CutoffSmem &sm, const CutoffArgs &A, int cell0) {
    const StructGeom &g = sm.g;
    const int N = sm.natoms, N2 = N * N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int ncl = g.ncell - cell0;
    if (ncl > MG_TCAP) ncl = MG_TCAP;
    const int ncg = (ncl + 31) >> 5;
    const int npb = (N2 + 31) >> 5;
    const int items = npb * ncg;
    const int center = (g.n[0] * g.dim[1] + g.n[1]) * g.dim[2] + g.n[2];   // tau = 0
    const float hi2 = g.hi2, lo2 = g.lo2;
    const int cap = sm.cap;
    for (int item = warp; item < items; item += MG_WARPS) {
        const int pb = item / ncg, cg = item - pb * ncg;
        const int q = pb * 32 + lane;
        const bool valid = q < N2;
        const int i = valid ? q / N : 0;
        const int j = valid ? q - i * N : 0;
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
            int rank = atomicAdd(&sm.rowcnt[i], __popc(mask));
            unsigned *seg = sm.stash + i * cap;
            while (mask) {
                const int b = __ffs(mask) - 1;
                mask &= mask - 1;
                const float4 T = Tg[b];
                unsigned code = ((unsigned)(cell0 + cg * 32 + b) << 6) | (unsigned)j;
                if (mg_d2(qx, qy, qz, T.x, T.y, T.z) >= lo2) {     // inside the rounding window
                    int t0, t1, t2;
                    double v[3];
                    mg_unpack_tau(T.w, t0, t1, t2);
                    const double d = mg_exact_vec(sm.x + 3 * i, sm.x + 3 * j, t0, t1, t2, sm.lat, v);
                    if (!(d < (double)A.r_c)) { code = MG_HOLE; atomicAdd(&sm.rowhole[i], 1); }
                }
                if (rank < cap) seg[rank] = code;
                ++rank;
            }
        }
    }
}

// Remove the (rare) window rejects from the stash rows and correct the counts.
__device__ inline void mg_cutoff_fix_holes(CutoffSmem &sm) {
    const int i = threadIdx.x;
    if (i < sm.natoms) {
        const int holes = sm.rowhole[i], cnt = sm.rowcnt[i];
        if (holes) {
            if (cnt <= sm.cap) {
                unsigned *seg = sm.stash + i * sm.cap;
                int w = 0;
                for (int e = 0; e < cnt; ++e) {
                    const unsigned c = seg[e];
                    if (c != MG_HOLE) seg[w++] = c;
                }
            }
            sm.rowcnt[i] = cnt - holes;
        }
        if (cnt - holes > sm.cap) sm.any_over = 1;   // benign race: all writers store 1
    }
}

// Phase 2: exclusive scan of the <= 64 row counts (warp 0), look-back over the chunk totals.
__device__ inline void mg_cutoff_scan_lookback(CutoffSmem &sm, const CutoffArgs &A) {
    const int lane = threadIdx.x;     // called by warp 0 only
    const int N = sm.natoms, s = sm.chunk;
    const int v0 = lane < N ? sm.rowcnt[lane] : 0;
    const int v1 = lane + 32 < N ? sm.rowcnt[lane + 32] : 0;
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
    if (lane == 0) sm.rowoff[MG_SMALL_MAX_ATOMS] = (int)total;
    unsigned base = 0u;
    if (s > 0) {
        if (lane == 0) mg_st_release(A.desc + s, mg_desc(MG_FLAG_AGG, A.epoch, total));
        int idx = s - 1;
        for (;;) {
            const int k = idx - lane;
            unsigned long long d = mg_desc(MG_FLAG_PFX, A.epoch, 0u);   // before chunk 0: prefix 0
            for (;;) {
                if (k >= 0) d = mg_ld_acquire(A.desc + k);
                const bool ok = ((unsigned)(d >> 32) & 0x3FFFFFFFu) == (A.epoch & 0x3FFFFFFFu) && (d >> 62) != 0ull;
                if (__all_sync(0xFFFFFFFFu, ok)) break;
                __nanosleep(40);
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
        mg_st_release(A.desc + s, mg_desc(MG_FLAG_PFX, A.epoch, base + total));
        sm.base = base;
        sm.total = total;
        if ((unsigned long long)base + total > 0x7FFFFFFFull) atomicOr(A.status, MGS_CAPACITY);
    }
}

// Write one edge.  vec / dist are the FP64 values of Def. 3 rounded once to FP32.
__device__ __forceinline__ void mg_emit_edge(const CutoffArgs &A, const CutoffSmem &sm, long long e,
                                             int i, int j, int t0, int t1, int t2) {
    if (e >= A.capacity) return;
    double v[3];
    const double d = mg_exact_vec(sm.x + 3 * i, sm.x + 3 * j, t0, t1, t2, sm.lat, v);
    A.src[e] = sm.first + i;
    A.dst[e] = sm.first + j;
    A.offset[3 * e] = (int8_t)t0; A.offset[3 * e + 1] = (int8_t)t1; A.offset[3 * e + 2] = (int8_t)t2;
    A.vec[3 * e] = (float)v[0]; A.vec[3 * e + 1] = (float)v[1]; A.vec[3 * e + 2] = (float)v[2];
    if (A.dist) A.dist[e] = (float)d;
}

// Phase 3: rows that fit their stash segment, one warp per row, lanes over consecutive edges.
__device__ inline void mg_cutoff_expand(CutoffSmem &sm, const CutoffArgs &A) {
    const StructGeom &g = sm.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cap = sm.cap;
    for (int i = warp; i < sm.natoms; i += MG_WARPS) {
        const int cnt = sm.rowcnt[i];
        if (cnt > cap) continue;
        const long long g0 = (long long)sm.base + sm.rowoff[i];
        const unsigned *seg = sm.stash + i * cap;
        for (int e = lane; e < cnt; e += 32) {
            const unsigned code = seg[e];
            int t0, t1, t2;
            mg_decode_cell((int)(code >> 6), g.dim, g.n, t0, t1, t2);
            mg_emit_edge(A, sm, g0 + e, i, (int)(code & 63u), t0, t1, t2);
        }
    }
}

// Rows whose segment overflowed: search again, warp per row, lanes over the cells of the current
// table tile, and write straight to global memory (rare path; also taken when cap == 0).
__device__ inline void mg_cutoff_research(CutoffSmem &sm, const CutoffArgs &A, int cell0) {
    const StructGeom &g = sm.g;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int N = sm.natoms;
    int ncl = g.ncell - cell0;
    if (ncl > MG_TCAP) ncl = MG_TCAP;
    const int center = (g.n[0] * g.dim[1] + g.n[1]) * g.dim[2] + g.n[2];
    for (int i = warp; i < N; i += MG_WARPS) {
        if (sm.rowcnt[i] <= sm.cap) continue;
        const float4 pi = sm.p[i];
        int cur = sm.rowcur[i];
        const long long g0 = (long long)sm.base + sm.rowoff[i];
        for (int c = lane; c < ((ncl + 31) & ~31); c += 32) {
            const float4 T = sm.T[c];
            int t0, t1, t2;
            mg_unpack_tau(T.w, t0, t1, t2);
            for (int j = 0; j < N; ++j) {
                const float4 pj = sm.p[j];
                const float d2 = mg_d2(__fsub_rn(pj.x, pi.x), __fsub_rn(pj.y, pi.y),
                                       __fsub_rn(pj.z, pi.z), T.x, T.y, T.z);
                bool hit = d2 < g.hi2 && !(i == j && cell0 + c == center);
                if (hit && d2 >= g.lo2) {
                    double v[3];
                    hit = mg_exact_vec(sm.x + 3 * i, sm.x + 3 * j, t0, t1, t2, sm.lat, v) < (double)A.r_c;
                }
                const unsigned m = __ballot_sync(0xFFFFFFFFu, hit);
                if (hit) mg_emit_edge(A, sm, g0 + cur + __popc(m & ((1u << lane) - 1u)), i, j, t0, t1, t2);
                cur += __popc(m);
            }
        }
        if (lane == 0) sm.rowcur[i] = cur;
    }
}

__global__ void __launch_bounds__(MG_BLOCK)
mg_cutoff_small_kernel(const CutoffArgs A) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    CutoffSmem &sm = *reinterpret_cast<CutoffSmem *>(smem_raw);
    const int tid = threadIdx.x;
    for (;;) {
        __syncthreads();                               // previous chunk fully retired
        if (tid == 0) sm.chunk = (int)atomicAdd(A.ticket, 1u);
        __syncthreads();
        const int s = sm.chunk;
        if (s >= A.n_struct) break;
        // ---- phase 0
        if (tid == 0) {
            sm.first = A.struct_ptr[s];
            sm.natoms = A.struct_ptr[s + 1] - sm.first;
            sm.any_over = 0;
        }
        if (tid >= 32 && tid < 41) sm.lat[tid - 32] = A.lattice[9 * (size_t)s + (tid - 32)];
        __syncthreads();
        int N = sm.natoms;
        const bool too_big = N > MG_SMALL_MAX_ATOMS;
        if (too_big) N = 0;                            // reported below; emits no edges
        if (tid < 3 * N) sm.x[tid] = A.pos[3 * (size_t)sm.first + tid];
        if (tid < MG_SMALL_MAX_ATOMS) { sm.rowcnt[tid] = 0; sm.rowhole[tid] = 0; sm.rowcur[tid] = 0; }
        __syncthreads();
        if (tid == 0) {
            sm.natoms = N;
            mg_cutoff_geometry(sm, A.r_c);
            unsigned err = sm.g.err | (too_big ? MGS_UNSUPPORTED : 0u);
            if (err) atomicOr(A.status, err);
            int cap = 0;
            if (N > 0 && sm.g.ncell > 0 && !A.count_only) {
                // expected row length lambda = N (4/3) pi r_c^3 / V, plus slack
                const float lam = (float)N * 4.18879f * A.r_c * A.r_c * A.r_c / sm.g.volume;
                cap = (int)(1.25f * lam) + 32;
                if (cap * N > MG_SCAP) cap = MG_SCAP / N;
            }
            sm.cap = cap;
        }
        __syncthreads();
        const StructGeom &g = sm.g;
        if (tid < N) {
            const float x0 = sm.x[3 * tid], x1 = sm.x[3 * tid + 1], x2 = sm.x[3 * tid + 2];
            float4 p;
            p.x = __fmaf_rn(x2, g.a[2][0], __fmaf_rn(x1, g.a[1][0], __fmul_rn(x0, g.a[0][0])));
            p.y = __fmaf_rn(x2, g.a[2][1], __fmaf_rn(x1, g.a[1][1], __fmul_rn(x0, g.a[0][1])));
            p.z = __fmaf_rn(x2, g.a[2][2], __fmaf_rn(x1, g.a[1][2], __fmul_rn(x0, g.a[0][2])));
            p.w = 0.f;
            sm.p[tid] = p;
        }
        // ---- phase 1
        const int ncell = N > 0 ? g.ncell : 0;
        for (int cell0 = 0; cell0 < ncell; cell0 += MG_TCAP) {
            __syncthreads();
            mg_build_table(sm, cell0);
            __syncthreads();
            mg_cutoff_find(sm, A, cell0);
        }
        __syncthreads();
        mg_cutoff_fix_holes(sm);
        __syncthreads();
        // ---- phase 2
        if (tid < 32) mg_cutoff_scan_lookback(sm, A);
        __syncthreads();
        const long long base = sm.base;
        if (tid < N) A.row_ptr[sm.first + tid] = (int)(base + sm.rowoff[tid]);
        if (s == A.n_struct - 1 && tid == 0) {
            const long long tot = base + sm.total;
            A.row_ptr[A.n_atoms] = (int)tot;
            *A.n_edges = tot;
            if (!A.count_only && tot > A.capacity) atomicOr(A.status, MGS_CAPACITY);
        }
        if (A.count_only) continue;
        // ---- phase 3
        mg_cutoff_expand(sm, A);
        if (sm.any_over) {
            for (int cell0 = 0; cell0 < ncell; cell0 += MG_TCAP) {
                __syncthreads();
                mg_build_table(sm, cell0);
                __syncthreads();
                mg_cutoff_research(sm, A, cell0);
            }
        }
    }
    // last CTA out resets the ticket for the next launch
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(A.ticket + 1, 1u) == gridDim.x - 1) { A.ticket[0] = 0u; A.ticket[1] = 0u; }
    }
}
