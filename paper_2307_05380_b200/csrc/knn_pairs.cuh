// knn_pairs.cuh — k-nearest-neighbour multigraph, k <= 32 (structures above MG_SMALL_MAX_ATOMS atoms, and
// structures whose atoms are given more than 40 cells apart (mg_knn_far), go a warp per row over every target
// and the pair's sub-box: mg_knn_row_box; what that does not settle, through the growing-radius routine of
// knn_small.cuh).
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

#define MG_KBOX_HITS 640           // hits of a row the table area of the warp's shared memory holds (atom, offset bytes)
#define MG_KBOX_MAX 512            // cells of a per-pair sub-box mg_knn_row_box walks

// One row of a structure the pair-lane machinery does not take (more atoms than it stages, or atoms many cells from the
// origin) inside a batch of small cells: lanes over (target, cell) of the per-pair sub-box of cut_prep.cuh — wrapped
// coordinates x - floor(x) taken on the fly, u = x_j - x_i, first cell lo_a = floor(-rho_a - u_a) + 1, m_a cells from there —
// d2 in FP32, hits (d2 < R^2) to the stash, (atom, offset bytes) to the table area; then the generic selection: the 32
// smallest FP32 keys, exact FP64 d2 for the k first and every hit FP32 cannot tell from the k-th, final order (d2, dst,
// tau).  The same steps as knn_bins.cu takes for a structure without a cell list.  Alg. 1 line 4: a row that does not
// settle inside R — fewer than k hits, a k-th key within the rounding window of R^2, more hits than the table area holds,
// an offset outside int8, a non-finite coordinate, a sub-box above MG_KBOX_MAX cells — goes to the growing-radius routine
// (227 us for ONE row of a 900-atom structure, which is why it is the last resort and not the rule).  Overwrites the
// stash: for whole structures only, not for a row in the middle of a group of the pair-lane path (whose unsettled rows
// call the growing-radius routine directly; through a wrapper of this name the headline's kernel ran 1.5 us longer).
__device__ __noinline__ void mg_knn_row_box(KnnSmem &ks, const KnnPairsArgs &A, const CutRec *R, int s, int first, int N, int i,
                                            int lane) {
    const int K = A.k, gi = first + i, mloc = R->mloc;
    bool done = false;
    __syncwarp();
    if (mloc > 0 && mloc <= MG_KBOX_MAX) {
        float a[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) a[c] = __ldg(A.lattice + 9 * (size_t)s + c);
        const float rad = R->radius, r2 = __fmul_rn(rad, rad);
        const float win = 1.1920929e-7f * (2.f * rad * (13.f * R->qmax + 2.f * R->amax_sum) + 4.f * rad * rad);
        const float lim2 = __fmaf_rn(-2.f, win, r2);
        const float rho0 = R->rho[0], rho1 = R->rho[1], rho2 = R->rho[2];
        const int m1 = (R->m >> 8) & 0xFF, m2 = (R->m >> 16) & 0xFF, M12 = m1 * m2;
        const bool wide = mloc >= 32;
        const int J = wide ? 1 : 32 / mloc, jl = wide ? 0 : lane / mloc, npass = wide ? (mloc + 31) >> 5 : 1;
        uint2 *meta = reinterpret_cast<uint2 *>(ks.w.T);
        const unsigned lt = (1u << lane) - 1u;
        const float *xg = A.pos + 3 * (size_t)first;
        const float p0 = xg[3 * i], p1 = xg[3 * i + 1], p2 = xg[3 * i + 2];
        const float gi0 = floorf(p0), gi1 = floorf(p1), gi2 = floorf(p2);
        const float xi0 = p0 - gi0, xi1 = p1 - gi1, xi2 = p2 - gi2;
        bool bad = !(fabsf(gi0) <= 500.f && fabsf(gi1) <= 500.f && fabsf(gi2) <= 500.f);      // (true for NaN / inf)
        int run = 0;
        for (int ps = 0; ps < npass; ++ps) {
            const int c = wide ? 32 * ps + lane : lane - jl * mloc;
            const bool cv = wide ? c < mloc : jl < J;
            const int t0 = c / M12, rr = c - t0 * M12, t1 = rr / m2, t2 = rr - t1 * m2;
            for (int j0 = 0; j0 < N; j0 += J) {
                const int j = j0 + jl;
                bool hit = false;
                unsigned long long key = 0ull;
                uint2 m = make_uint2(0u, 0u);
                if (cv && j < N) {
                    const float q0 = xg[3 * j], q1 = xg[3 * j + 1], q2 = xg[3 * j + 2];
                    const float gj0 = floorf(q0), gj1 = floorf(q1), gj2 = floorf(q2);
                    const float u0 = __fsub_rn(q0 - gj0, xi0), u1 = __fsub_rn(q1 - gj1, xi1), u2 = __fsub_rn(q2 - gj2, xi2);
                    const float e0 = floorf(__fsub_rn(-rho0, u0)) + 1.f, e1 = floorf(__fsub_rn(-rho1, u1)) + 1.f,
                                e2 = floorf(__fsub_rn(-rho2, u2)) + 1.f;
                    const float f0 = __fadd_rn(u0, e0 + (float)t0), f1 = __fadd_rn(u1, e1 + (float)t1), f2 = __fadd_rn(u2, e2 + (float)t2);
                    const float vx = __fmaf_rn(f2, a[6], __fmaf_rn(f1, a[3], __fmul_rn(f0, a[0])));
                    const float vy = __fmaf_rn(f2, a[7], __fmaf_rn(f1, a[4], __fmul_rn(f0, a[1])));
                    const float vz = __fmaf_rn(f2, a[8], __fmaf_rn(f1, a[5], __fmul_rn(f0, a[2])));
                    const float d2 = __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmul_rn(vx, vx)));
                    const bool okj = fabsf(gj0) <= 500.f && fabsf(gj1) <= 500.f && fabsf(gj2) <= 500.f;
                    // x_j + tau - x_i = u + e + t: tau = e + t + floor(x_i) - floor(x_j)
                    const int tau0 = (int)e0 + t0 + (int)gi0 - (int)gj0, tau1 = (int)e1 + t1 + (int)gi1 - (int)gj1,
                              tau2 = (int)e2 + t2 + (int)gi2 - (int)gj2;
                    bad = bad || !okj || tau0 < -127 || tau1 < -127 || tau2 < -127 || tau0 > 127 || tau1 > 127 || tau2 > 127;
                    hit = !bad && d2 < r2 && !(i == j && (tau0 | tau1 | tau2) == 0);       // (i, i, 0) is not an edge (R3)
                    key = (unsigned long long)__float_as_uint(d2) << 32;
                    m = make_uint2((unsigned)j, ((unsigned)(tau0 + 128) << 16) | ((unsigned)(tau1 + 128) << 8) | (unsigned)(tau2 + 128));
                }
                const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
                if (hit) {
                    const int pos = run + __popc(bal & lt);
                    if (pos < MG_KBOX_HITS) { ks.stash[pos] = key | (unsigned)pos; meta[pos] = m; }
                }
                run += __popc(bal);
            }
        }
        __syncwarp();
        const int total = __any_sync(0xFFFFFFFFu, bad) ? MG_KBOX_HITS + 1 : run;
        if (total >= K && total <= MG_KBOX_HITS) {
            // the 32 smallest FP32 keys (Alg. 2's "sort, keep k", 32 at a time)
            mg_key key = mg_sort32(lane < total ? ks.stash[lane] : MG_KEY_INF, lane);
            for (int c = 32; c < total; c += 32) {
                mg_key keys1[1] = {key};
                mg_knn_merge<1>(keys1, c + lane < total ? ks.stash[c + lane] : MG_KEY_INF, lane);
                key = keys1[0];
            }
            const mg_key kth = __shfl_sync(0xFFFFFFFFu, key, K - 1);
            const float kth_d2 = __uint_as_float((unsigned)(kth >> 32));
            if (kth != MG_KEY_INF && kth_d2 < lim2) {
                const bool amb = lane >= K && key != MG_KEY_INF && __uint_as_float((unsigned)(key >> 32)) <= __fmaf_rn(2.f, win, kth_d2);
                const int nsel = K + __popc(__ballot_sync(0xFFFFFFFFu, amb));
                int j = 0, tau[3] = {0, 0, 0};
                unsigned long long ord = ~0ull;
                double dd = 1e300, vv[3] = {0.0, 0.0, 0.0};
                if (lane < nsel) {
                    const uint2 m = meta[(unsigned)key];                          // (the key's low word is the hit's number)
                    j = (int)m.x;
                    tau[0] = (int)(m.y >> 16) - 128; tau[1] = (int)((m.y >> 8) & 0xFFu) - 128; tau[2] = (int)(m.y & 0xFFu) - 128;
                    double xi[3], xj[3], L[9];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        xi[c] = (double)xg[3 * i + c];
                        xj[c] = (double)xg[3 * j + c];
                    }
#pragma unroll
                    for (int c = 0; c < 9; ++c) L[c] = (double)a[c];
                    dd = mg_knn_exact_d2(xi, xj, tau[0], tau[1], tau[2], L, vv);
                    ord = ((unsigned long long)(unsigned)j << 24) | m.y;
                }
                int rank = 0;
                for (int l = 0; l < nsel; ++l) {
                    const double od = __shfl_sync(0xFFFFFFFFu, dd, l);
                    const unsigned long long oo = __shfl_sync(0xFFFFFFFFu, ord, l);
                    rank += (od < dd || (od == dd && oo < ord)) ? 1 : 0;
                }
                if (lane < nsel && rank < K) {
                    const long long e = (long long)K * gi + rank;
                    A.src[e] = gi;
                    A.dst[e] = first + j;
                    A.offset[3 * e] = (int8_t)tau[0]; A.offset[3 * e + 1] = (int8_t)tau[1]; A.offset[3 * e + 2] = (int8_t)tau[2];
                    A.vec[3 * e] = (float)vv[0]; A.vec[3 * e + 1] = (float)vv[1]; A.vec[3 * e + 2] = (float)vv[2];
                    if (A.dist) A.dist[e] = __fsqrt_rn((float)dd);
                    if (rank == K - 1 && A.hint) {
                        const float dk = __fsqrt_ru(__double2float_ru(dd));
                        if (dk > 0.f) atomicMax(reinterpret_cast<int *>(A.hint + s), __float_as_int(dk));
                    }
                }
                done = true;
            }
        }
        __syncwarp();
    }
    if (!done) mg_knn_row_fallback(ks, A, s, first, N, i, lane);
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
