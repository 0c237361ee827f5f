// knn_pairs.cuh — k-nearest-neighbour multigraph, k <= 32 (structures above MG_SMALL_MAX_ATOMS atoms
// go row by row through the growing-radius routine of knn_small.cuh, and so do structures whose atoms are
// given more than 40 cells apart: mg_knn_far).
//
// Problem: per source the k smallest keys (d, dst, tau_x, tau_y, tau_z) over all periodic images
// except (i,i,0) (Alg. 2 lines 2-5, made deterministic: DESIGN.md R2, R8).
// Method (Alg. 1, re-designed).  mg_cut_prep_kernel picks one search radius R per
// structure (expected MG_KNN_ALPHA * k images inside, or the largest k-th distance of the previous
// mg_update_graph call) and, like for the cutoff graph, the per-pair sub-box that holds every image
// closer than R.  One launch, autonomous warps, each owning a contiguous equally expensive range
// of source rows (cutoff_pairs.cuh):
//   find    lane <-> ordered pair (i, j): hit mask over the pair's sub-box (d2 < R^2 in FP32),
//           hits -> shared-memory stash as 64-bit keys (d2 bits | tau + 128 bytes, j) in (row, j)
//           order: "evaluate_area" + "concatenate" of Alg. 1-2.  A sub-box of more than 256 cells
//           (strongly sheared cells) does not fit the warp's table: one row at a time, lanes over the
//           cells of each pair's sub-box (mg_knn_find_cells);
//   select  per source row: bitonic sort of its keys, 32 at a time, keeping the 32 smallest (Alg. 2's
//           "sort, keep k").  Alg. 1 line 4: if the k-th key is not safely inside R (or fewer than k
//           images were found) the row is searched again by the growing-radius routine of
//           knn_small.cuh.  The k selected entries get their exact FP64 distance and their final
//           order (d, dst, tau); vec / dist are the FP64 values rounded once.
#pragma once
#include "common.cuh"
#include "cut_prep.cuh"
#include "cutoff_pairs.cuh"
#include "knn_small.cuh"

#define MG_KSTASH 768              // 64-bit keys per warp

struct KnnPairsArgs {
    const float *pos;
    const float *lattice;
    const int32_t *struct_ptr;
    int n_struct, n_atoms;
    int k;
    int32_t *row_ptr, *src, *dst;
    int8_t *offset;
    float *vec, *dist;
    long long *n_edges;
    float *hint;                   // [n_struct] or NULL: max k-th distance per structure (atomicMax)
    const CutRec *rec;
    const unsigned long long *bpre;
    int n_blocks;
    int n_warps;
    unsigned *status;
    unsigned *dbg;                 // [8, n_warps] phase cycles (MG_PHASE_CLOCKS builds) or NULL
};

struct KnnSmem {
    WarpSmem w;                    // table, staged positions
    unsigned long long stash[MG_KSTASH];
    int rowoff[MG_SMALL_MAX_ATOMS + 1];
    double xd[MG_SMALL_MAX_ATOMS][3];  // positions as given + lattice, promoted once per structure: operands of the
    double latd[9];                    // exact FP64 distance
};

// Exact squared distance of one image from the staged FP64 operands: f = (x_j - x_i) + tau, v = f . L, no FMA
// contraction, sums left to right (R15: the oracle's operation order, so d2 is the oracle's d^2).
__device__ __forceinline__ double mg_knn_exact_d2(const double *xi, const double *xj, int t0, int t1, int t2,
                                                   const double *L, double v[3]) {
    // (double)t without a conversion instruction: 2^52 + 2^31 + t has t + 2^31 in its low mantissa word
    const double f0 = __dadd_rn(__dsub_rn(xj[0], xi[0]), __hiloint2double(0x43300000, t0 ^ 0x80000000) - 4503601774854144.0);
    const double f1 = __dadd_rn(__dsub_rn(xj[1], xi[1]), __hiloint2double(0x43300000, t1 ^ 0x80000000) - 4503601774854144.0);
    const double f2 = __dadd_rn(__dsub_rn(xj[2], xi[2]), __hiloint2double(0x43300000, t2 ^ 0x80000000) - 4503601774854144.0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
        v[c] = __dadd_rn(__dadd_rn(__dmul_rn(f0, L[c]), __dmul_rn(f1, L[3 + c])), __dmul_rn(f2, L[6 + c]));
    return __dadd_rn(__dadd_rn(__dmul_rn(v[0], v[0]), __dmul_rn(v[1], v[1])), __dmul_rn(v[2], v[2]));
}

// Growing-radius search of one source row with the routine of knn_small.cuh (rare path).  Uses the
// table area of the warp's shared memory as scratch: the caller rebuilds the table afterwards.
__device__ __noinline__ void mg_knn_row_fallback(KnnSmem &ks, const KnnPairsArgs &A, int s, int first, int N, int i,
                                                 int lane) {
    const float *lat9 = A.lattice + 9 * (size_t)s;
    float4 *sp = reinterpret_cast<float4 *>(ks.w.T);
    mg_key *buf = reinterpret_cast<mg_key *>(ks.w.T + MG_SMALL_MAX_ATOMS);
    StructRec R;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
    __syncwarp();
    const bool big = N > MG_SMALL_MAX_ATOMS;      // too large to stage: positions on the fly
    for (int j = lane; j < N; j += 32) {
        const float *x = A.pos + 3 * (size_t)(first + j);
        const float x0 = x[0], x1 = x[1], x2 = x[2];
        lo[0] = fminf(lo[0], x0); lo[1] = fminf(lo[1], x1); lo[2] = fminf(lo[2], x2);
        hi[0] = fmaxf(hi[0], x0); hi[1] = fmaxf(hi[1], x1); hi[2] = fmaxf(hi[2], x2);
        if (big) continue;
        float4 p;
        p.x = __fmaf_rn(x2, lat9[6], __fmaf_rn(x1, lat9[3], __fmul_rn(x0, lat9[0])));
        p.y = __fmaf_rn(x2, lat9[7], __fmaf_rn(x1, lat9[4], __fmul_rn(x0, lat9[1])));
        p.z = __fmaf_rn(x2, lat9[8], __fmaf_rn(x1, lat9[5], __fmul_rn(x0, lat9[2])));
        p.w = 0.f;
        sp[j] = p;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            lo[a] = fminf(lo[a], __shfl_xor_sync(0xFFFFFFFFu, lo[a], o));
            hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xFFFFFFFFu, hi[a], o));
        }
    __syncwarp();
    float lat[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) lat[c] = lat9[c];
    double vol = 1.0, h[3] = {1.0, 1.0, 1.0};
    mg_cell_spacings(lat, &vol, h);                   // the lattice is valid: prep checked it
    R.first = first;
    R.natoms = N;
    R.volume = (float)vol;
    R.err = 0u;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        R.xmin[a] = lo[a];
        R.xmax[a] = hi[a];
        R.h_dn[a] = __double2float_rd(h[a] * (1.0 - 1e-6));
        R.invh_up[a] = __double2float_ru((1.0 + 1e-6) / h[a]);
        R.amax[a] = fmaxf(fabsf(lat[3 * a]), fmaxf(fabsf(lat[3 * a + 1]), fabsf(lat[3 * a + 2])));
    }
    KnnArgs K;
    K.pos = A.pos; K.lattice = A.lattice; K.struct_ptr = A.struct_ptr;
    K.n_struct = A.n_struct; K.n_atoms = A.n_atoms; K.k = A.k;
    K.row_ptr = A.row_ptr; K.src = A.src; K.dst = A.dst; K.offset = A.offset;
    K.vec = A.vec; K.dist = A.dist; K.n_edges = A.n_edges;
    float *slot = reinterpret_cast<float *>(ks.w.T + MG_SMALL_MAX_ATOMS + 16);   // k-th distance comes back here
    K.radius_hint = A.hint ? slot - (first + i) : nullptr; K.use_hint = 0;
    K.rec = nullptr; K.atom_struct = nullptr; K.ctl = nullptr; K.status = A.status;
    mg_knn_source<1>(K, R, lat9, big ? nullptr : sp, buf, i, lane);
    __syncwarp();
    if (A.hint && lane == 0) atomicMax(reinterpret_cast<int *>(A.hint + s), __float_as_int(*slot));
    __syncwarp();
}

// Hits of the pairs [qa, qb) (whole rows) of the staged structure -> stash, row offsets -> rowoff.
// Returns the number of hits (positions >= MG_KSTASH are dropped: the caller checks).
template <int W>
__device__ __forceinline__ int mg_knn_find(KnnSmem &ks, const Task &k, const FindCtx &F, int i0, int qa, int qb,
                                           int lane) {
    const WarpSmem &sw = ks.w;
    const int N = k.natoms;
    const float inv_N = 1.f / (float)N;
    int run = 0;
    for (int q0 = qa; q0 < qb; q0 += 32) {
        const int q = q0 + lane;
        const bool valid = q < qb;
        const int i = valid ? mg_fdiv(q, inv_N) : 0, j = valid ? q - i * N : 0;
        const PairLane p = mg_pair_setup(sw, F, valid, i, j);
        unsigned mask[W];
        mg_block_masks<W>(sw, F, p, k.first + i, k.first + j, 0, F.mloc, mask);
        int cnt = 0;
#pragma unroll
        for (int w = 0; w < W; ++w) cnt += __popc(mask[w]);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        int pos = run + incl - cnt;
        if (valid && j == 0) ks.rowoff[i - i0] = pos;
        const unsigned paircode = ((unsigned)(p.l0 + 128) << 24) | ((unsigned)(p.l1 + 128) << 16) |
                                  ((unsigned)(p.l2 + 128) << 8) | (unsigned)j;
#pragma unroll
        for (int w = 0; w < W; ++w) {
            unsigned mk = mask[w];
            while (mk) {
                const int b = __clz(mk);
                mk &= ~(0x80000000u >> b);
                const float4 T = mg_tcell(sw, 32 * w + b);
                const float vx = __fadd_rn(p.qx, T.x), vy = __fadd_rn(p.qy, T.y), vz = __fadd_rn(p.qz, T.z);
                const float d2 = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmul_rn(vx, vx)));
                if (pos < MG_KSTASH)
                    ks.stash[pos] = ((unsigned long long)__float_as_uint(d2) << 32) | (paircode + sw.tcode[32 * w + b]);
                ++pos;
            }
        }
        run += __shfl_sync(0xFFFFFFFFu, incl, 31);
    }
    return run;
}

// 3 CTAs per SM: 168 registers per thread and no spills beat 4 CTAs at 128 registers (A/B: -12 %)
// Wide tables are rare in the headline workload: kept out of line so that they do not cost the
// common path registers.
__device__ __noinline__ int mg_knn_find_wide(KnnSmem &ks, const Task &k, const FindCtx &F, int i0, int qa, int qb,
                                             int lane) {
    if (F.mloc <= 128) return mg_knn_find<4>(ks, k, F, i0, qa, qb, lane);
    return mg_knn_find<8>(ks, k, F, i0, qa, qb, lane);
}

// A structure whose table does not fit the warp's shared memory (mloc > MG_TLOC: strongly skewed cells, which have
// few atoms): ONE source row i at a time, lanes over the CELLS of the pair's sub-box (lane <-> pair would leave all
// but N lanes idle through thousands of cells), the translation t . L evaluated on the fly with the table's
// arithmetic.  The row's hits go to out[0 .. cap) (the stash).  Returns their
// number (hits beyond cap are dropped: the caller checks).
#define MG_KNN_TILED_MAX 4096      // cells; beyond: the growing-radius routine
__device__ __noinline__ int mg_knn_find_cells(KnnSmem &ks, const Task &k, const FindCtx &F, int i, int lane,
                                              unsigned long long *out, int cap) {
    const WarpSmem &sw = ks.w;
    const int N = k.natoms, m1 = (F.m >> 8) & 0xFF, m2 = (F.m >> 16) & 0xFF, M12 = m1 * m2;
    const float inv12 = 1.f / (float)M12, inv2 = 1.f / (float)m2;     // (mloc <= 4096: the float reciprocal is exact)
    const float r2 = -F.nr2;
    const unsigned lt = (1u << lane) - 1u;
    int run = 0;
    for (int j = 0; j < N; ++j) {
        const PairLane p = mg_pair_setup(sw, F, true, i, j);          // the same on every lane
        if (!p.ok) return cap + 1;                                     // offsets outside int8: the growing-radius routine decides (and reports)
        const unsigned paircode = ((unsigned)(p.l0 + 128) << 24) | ((unsigned)(p.l1 + 128) << 16) |
                                  ((unsigned)(p.l2 + 128) << 8) | (unsigned)j;
        // four cells per lane and trip (c0 + lane + 32 u): four independent chains in flight
        for (int c0 = 0; c0 < F.mloc; c0 += 128) {
            bool hit[4];
            unsigned long long key[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int c = c0 + 32 * u + lane;
                const int t0 = mg_fdiv(c, inv12), r = c - t0 * M12, t1 = mg_fdiv(r, inv2), t2 = r - t1 * m2;
                const float f0 = (float)t0, f1 = (float)t1, f2 = (float)t2;
                const float Tx = __fmaf_rn(f2, F.a[6], __fmaf_rn(f1, F.a[3], __fmul_rn(f0, F.a[0])));
                const float Ty = __fmaf_rn(f2, F.a[7], __fmaf_rn(f1, F.a[4], __fmul_rn(f0, F.a[1])));
                const float Tz = __fmaf_rn(f2, F.a[8], __fmaf_rn(f1, F.a[5], __fmul_rn(f0, F.a[2])));
                const float vx = __fadd_rn(p.qx, Tx), vy = __fadd_rn(p.qy, Ty), vz = __fadd_rn(p.qz, Tz);
                const float d2 = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmul_rn(vx, vx)));
                hit[u] = c < F.mloc && d2 < r2 && c != p.self;         // (i, i, 0) is not an edge (R3)
                key[u] = ((unsigned long long)__float_as_uint(d2) << 32) |
                         (paircode + (((unsigned)t0 << 24) | ((unsigned)t1 << 16) | ((unsigned)t2 << 8)));
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit[u]);
                if (hit[u]) {
                    const int pos = run + __popc(bal & lt);
                    if (pos < cap) out[pos] = key[u];
                }
                run += __popc(bal);
            }
        }
    }
    return run;
}

// Could a pair of the staged structure have offsets outside int8?  l_a = e_a + k_ia - k_ja with -rho_a - 2 < e_a <= 1
// and the m_a cells from there on must stay within [-127, 127]: certainly so when every atom is within 40 cells of the
// origin and no axis of the sub-box has more than 40 cells.
__device__ __forceinline__ bool mg_knn_far(const WarpSmem &sw, const FindCtx &F, int N, int lane) {
    bool far = (F.m & 0xFF) > 40 || ((F.m >> 8) & 0xFF) > 40 || ((F.m >> 16) & 0xFF) > 40;
    for (int j = lane; j < N; j += 32) {
        const int kk = __float_as_int(sw.x[j].w);
        far = far || abs((kk & 1023) - 512) > 40 || abs(((kk >> 10) & 1023) - 512) > 40 || abs(((kk >> 20) & 1023) - 512) > 40;
    }
    return __any_sync(0xFFFFFFFFu, far);
}

// The kernel (knn_pairs_kernel.inc) is compiled twice, in two translation units: here as mg_knn_pairs_kernel for
// k <= 16 (the headline), in knn_large.cu (which defines MG_KNN_LARGE_TU) as mg_knn_pairs_large_kernel for k > 16, whose
// rows mostly have 33 .. 64 hits and get a fast path of their own.  Two modules on purpose: with both kernels in one the
// headline's kernel — same SASS, same place in the module — measured 1 us of 57 slower on cold outputs.
#ifdef MG_KNN_LARGE_TU
#define MG_KNN_KERNEL_NAME mg_knn_pairs_large_kernel
#define MG_KNN_LARGE 1
#else
#define MG_KNN_KERNEL_NAME mg_knn_pairs_kernel
#define MG_KNN_LARGE 0
#endif
#include "knn_pairs_kernel.inc"
#undef MG_KNN_KERNEL_NAME
#undef MG_KNN_LARGE
