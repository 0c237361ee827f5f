// cut_prep.cuh — K1 (per-structure search bounds) + K6 (batching) of the cutoff graph: one THREAD
// per structure, one launch, no waiting between blocks.
//
// For structure s with lattice rows a_0,a_1,a_2 (R5):
//   * plane spacings h_a = V / |a_b x a_c| (BASELINE.json north_star).  The cross
//     products and V are evaluated in FP64 (validity: finite, V > 1e-9), rho_a = r_c / h_a in FP32,
//     inflated so that rho_a is an UPPER bound;
//   * an edge (i, j, tau) has |x_ja - x_ia + tau_a| h_a <= d < r_c (projection on the plane normal,
//     DESIGN.md R14), so for the ordered pair (i, j) only the integers tau_a in the open interval
//     (-rho_a - u_a, rho_a - u_a), u_a = x_ja - x_ia, can be edges: at most m_a = floor(2 rho_a) + 1
//     of them.  The graph kernels evaluate exactly the m_0 m_1 m_2 cells of that per-pair sub-box
//     (a subset of the box |tau_a| <= ceil(r_c / h_a) of north_star);
//   * the constants of the rounding window of the FP32 filter (R23);
//   * an estimated cost per ordered pair (i, j) (1/16 warp instructions) and its prefix over the
//     batch: the graph kernels cut the batch's pairs, in (structure, i, j) order, into one
//     contiguous, equally expensive range per warp.  The prefix is two-level: lpre[s] inside a
//     block of MG_CP_BLOCK structures and, written by the last block to finish, bpre[b] over the
//     blocks.
#pragma once
#include "common.cuh"

#define MG_CP_BLOCK 128
#define MGB_MAXSLAB 16             // cell list (cut_bins.cuh): slabs per axis, at most
#define MGB_MINSLAB 6              // ... fewer than this: the five-slab stencil would cover the axis, one slab instead
#ifndef MG_STASH
#define MG_STASH 1024              // stash entries per warp of the emit kernel (cutoff_pairs.cuh)
#endif
#ifndef MG_KNN_ALPHA
#define MG_KNN_ALPHA 1.45f         // KNN: expected images inside the first search radius, in units of k
#define MG_KNN_RSCALE 1.05f        // ... and the safety factor on that radius
#endif
#ifndef MG_KNN_HINT
#define MG_KNN_HINT 1.08f           // mg_update_graph: search radius in units of the structure's largest k-th distance of the last call
#endif
// cost model of the cutoff path, in warp instructions (tuned on config 2, profiles/)
#ifndef MG_STRUCT_COST
#define MG_STRUCT_COST 900.f       // staging one structure (latency, both launches)
#endif
#ifndef MG_C_CELL
#define MG_C_CELL 14.f             // per candidate cell of a pair (x 1/32 per lane)
#define MG_C_CELL_MID 14.f         // ... tables of 65-128 cells
#define MG_C_CELL_WIDE 24.f        // ... tables of 129-256 cells
#define MG_C_BLOCK 250.f           // per block of 32 pairs
#define MG_C_BLOCK_WIDE 500.f
#define MG_C_EDGE 3.3f             // per emitted edge
#endif
// ... of the scan kernel (cut_scan.cuh), in cycles: see the comment where they are used
#ifndef MG_CS_BLOCK
#define MG_CS_BLOCK 735.f
#define MG_CS_GROUP 182.f
#define MG_CS_EDGE 17.f
#define MG_CS_STRUCT 4000.f
#define MG_CS_ROWCELL 25.f
#define MG_CS_BINCAND 2.f          // binned rows (cut_bins.cuh): per candidate left by the stencil (swept on configs[3]: 16 / 8 / 4 / 2 / 1 -> 153.3 / 152.0 / 151.3 / 148.6 / 148.9 us)
#define MG_CS_BINROW 1500.f        // ... per source row (the stencil's table)
#endif
// ... and of the KNN launch: per candidate cell, per block of 32 pairs, per source row (selection),
// per structure
#ifndef MG_KC_CELL
#define MG_KC_CELL 17.f
#endif
#ifndef MG_KC_BLOCK
#define MG_KC_BLOCK 150.f
#endif
#ifndef MG_KC_ROW
#define MG_KC_ROW 250.f
#endif
#ifndef MG_KC_STRUCT
#define MG_KC_STRUCT 1300.f
#endif

struct CutRec {              // 64 bytes
    float rho[3];            // upper bound of r_c / h_a (plus the guard eps)
    int m;                   // per-pair sub-box m_0 | m_1 << 8 | m_2 << 16
    int mloc;                // m_0 m_1 m_2; 0: the structure emits nothing (invalid / empty)
    int first, natoms;
    unsigned paircost;       // estimated cost of one ordered pair, 1/16 warp instructions (>= 1)
    unsigned err;            // MGS_* bits
    unsigned long long lpre; // prefix of natoms^2 * paircost inside the structure's prep block
    float amax_sum;          // sum_a max_c |L_ac|
    float qmax;              // Q = sum_a (rho_a + 1) max_c |L_ac|
    float radius;            // KNN: search radius of the structure (cutoff graph: r_c)
    int bins;                // cell list (cut_bins.cuh): nb_0 | nb_1 << 8 | nb_2 << 16 | 1 << 24; 0: not binned
};
static_assert(sizeof(CutRec) == 64, "CutRec is one 64-byte line");

struct CutPrepArgs {
    const float *lattice;
    const int32_t *struct_ptr;
    int n_struct, n_atoms;
    float r_c;                     // cutoff graph: the cutoff.  KNN (k > 0): unused
    int k;                         // KNN: neighbours per atom; the radius of structure s is chosen so that
                                   // about MG_KNN_ALPHA * k images are expected inside (or taken from hint[s])
    float *hint;                   // KNN, [n_struct] or NULL: largest k-th distance of the previous call
                                   // (read when use_hint, then reset to 0: the graph kernel maxes into it)
    int use_hint;
    int rows_cost;                 // cutoff: cost model of the scan kernel (cut_scan.cuh)
    const float *radii;            // [n_atoms] or NULL: per-atom cutoffs (cutoff graph); the structure's radius is
                                   // their maximum; a radius that is not a positive finite number makes the
                                   // structure invalid (MGS_UNSUPPORTED)
    const float *pos;              // with xw4: positions of the batch
    float4 *xw4;                   // [n_atoms] or NULL: wrapped fractional coordinates x - floor(x), .w = the integer
                                   // parts packed (mg_wrap_x): written by the blocks after the first n_sblocks ones
    int n_sblocks;                 // blocks that hold structures (the grid may have more: they only wrap coordinates)
    int *binlist;                  // [n_struct] or NULL: the structures that get a cell list (cut_bins.cuh), in any order;
                                   // their number in ctl[13] (zero before the call: the scan kernel leaves it so)
    CutRec *rec;                   // [n_struct]
    unsigned long long *bpre;      // [blocks + 1] block sums -> exclusive prefix; [blocks] = total
    unsigned *ctl;                 // [7] blocks done, [13] structures with a cell list
    unsigned *status;
};

__global__ void __launch_bounds__(MG_CP_BLOCK)
mg_cut_prep_kernel(const CutPrepArgs A) {
    mg_grid_dependency_wait();      // the kernels of the previous call still read rec / bpre
    if (A.xw4) {                     // K2 staging: every atom's wrapped coordinates, once per call
        const int nx = (int)gridDim.x - A.n_sblocks;       // (no extra blocks: the structure blocks do it)
        const int b0 = nx > 0 ? (int)blockIdx.x - A.n_sblocks : (int)blockIdx.x, nb = nx > 0 ? nx : (int)gridDim.x;
        if (b0 >= 0)
            for (int g = b0 * MG_CP_BLOCK + (int)threadIdx.x; g < A.n_atoms; g += nb * MG_CP_BLOCK) {
                const float x0 = A.pos[3 * (size_t)g], x1 = A.pos[3 * (size_t)g + 1], x2 = A.pos[3 * (size_t)g + 2];
                const float g0 = floorf(x0), g1 = floorf(x1), g2 = floorf(x2);
                const bool ok = fabsf(g0) <= 500.f && fabsf(g1) <= 500.f && fabsf(g2) <= 500.f;   // false for NaN / inf
                const int kk = ((int)g0 + 512) | (((int)g1 + 512) << 10) | (((int)g2 + 512) << 20);
                A.xw4[g] = make_float4(x0 - g0, x1 - g1, x2 - g2, __int_as_float(ok ? kk : 0));
            }
        if ((int)blockIdx.x >= A.n_sblocks) return;
    }
    __shared__ unsigned long long s_warp[MG_CP_BLOCK / 32];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int s = blockIdx.x * MG_CP_BLOCK + threadIdx.x;
    unsigned long long cost = 0ull;
    CutRec r;
    if (s < A.n_struct) {
        r.first = A.struct_ptr[s];
        r.natoms = A.struct_ptr[s + 1] - r.first;
        const int N = r.natoms;
        float lat[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) lat[c] = A.lattice[9 * (size_t)s + c];
        double vol = 0.0, h[3] = {1.0, 1.0, 1.0};
        unsigned err = mg_cell_spacings_fast(lat, &vol, h);
        float rc = A.r_c;
        if (A.radii) {
            rc = 0.f;
            bool okr = true;
            for (int i = 0; i < N; ++i) {
                const float ci = A.radii[r.first + i];
                okr = okr && ci > 0.f && isfinite(ci);
                rc = fmaxf(rc, ci);
            }
            if (!okr) err |= MGS_UNSUPPORTED;
            if (!(rc > 0.f) || !isfinite(rc)) rc = 1.f;
        }
        if (A.k > 0) {                                 // KNN: radius from the density, or from the last call
            const float hv = A.hint && A.use_hint ? A.hint[s] : 0.f;
            // expected images inside: 1.45 k + 1; in a large structure (a warp per row through the cell list, knn_bins.cu:
            // a row that comes up short costs a search over all N atoms) k + 4 sqrt(k) + 2 if that is more — for atoms
            // placed at random the count inside R is about Poisson, and 18 expected leave 5 % of the rows below 12
            float expect = MG_KNN_ALPHA * (float)A.k + 1.f;
            if (N > MG_SMALL_MAX_ATOMS || A.binlist) expect = fmaxf(expect, (float)A.k + 4.f * sqrtf((float)A.k) + 2.f);   // (binlist: every row of the batch is a warp's, knn_bins.cu)
            rc = MG_KNN_RSCALE * cbrtf(0.2387324f * expect * (float)vol / (float)max(N, 1));
            if (hv > 0.f && isfinite(hv)) rc = MG_KNN_HINT * hv + 1e-3f;
            if (!(rc > 1e-6f) || !isfinite(rc)) rc = 1.f;
            if (A.hint) A.hint[s] = 0.f;
        }
        r.radius = rc;
        if (N > 46000) err |= MGS_UNSUPPORTED;                            // pair indices are 32 bit
        r.mloc = 0;
        r.m = 0;
        r.amax_sum = 0.f;
        float Q = 0.f;
        int mloc = 1;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float amax = fmaxf(fabsf(lat[3 * a]), fmaxf(fabsf(lat[3 * a + 1]), fabsf(lat[3 * a + 2])));
            r.amax_sum += amax;
            // rho = r_c / h rounded up, plus the guard for the FP32 rounding of u = x_j - x_i and
            // of -rho - u (wrapped coordinates: |u| <= 1)
            const float rho = __double2float_ru((double)rc / h[a] * (1.0 + 4e-6)) + 4e-6f;
            r.rho[a] = rho;
            float mf = floorf(2.f * rho + 1e-5f) + 1.f;
            if (!(mf <= 255.f)) { err |= MGS_OFFSET; mf = 1.f; }
            r.m |= (int)mf << (8 * a);
            mloc *= (int)mf;
            Q += (rho + 1.f) * amax;
        }
        if (!err && N > 0) r.mloc = mloc;
        r.qmax = Q;
        r.err = err;
        if (err) atomicOr(A.status, err);
        r.paircost = 1u;
        r.bins = 0;
        if (r.mloc > 0) {
            const float lam = (float)N * 4.18879f * rc * rc * rc / (float)vol;   // edges per row
            // warp instructions per pair (count + emit launches): 11 per candidate, ~250 per block
            // of 32 pairs, 3.3 per edge; the per-structure staging is spread over its pairs
            // (structures whose table is tiled evaluate their candidates again in the emit launch)
            // and walk them one source row (N of 32 lanes) at a time)
            const float percell = mloc > 256 ? 11.f + 900.f / (float)N : (mloc > 128 ? MG_C_CELL_WIDE : (mloc > 64 ? MG_C_CELL_MID : MG_C_CELL));
            const float perblock = mloc > 256 ? 120.f + 16000.f / (float)N : (mloc > 128 ? MG_C_BLOCK_WIDE : MG_C_BLOCK);
            const float c = ((float)((mloc + 3) & ~3) * percell + perblock) * (1.f / 32.f) +
                            MG_C_EDGE * lam / (float)N + MG_STRUCT_COST / ((float)N * (float)N);
            // KNN: one launch, no edge stream (constants from a sweep over four seeds of config 2 and config 4)
            // (a table above 256 cells: one source row at a time, lanes over the cells of each pair's sub-box, about 35
            // instructions per 32 cells and 80 per pair)
            const float ck = (mloc > 256 ? (float)mloc * (35.f / 32.f) + 80.f : ((float)((mloc + 3) & ~3) * MG_KC_CELL + MG_KC_BLOCK) * (1.f / 32.f)) +
                             MG_KC_ROW / (float)N + MG_KC_STRUCT / ((float)N * (float)N);
            // (KNN above the staging limit inside a batch of small cells: a warp per row, lanes over (target, cell),
            // mg_knn_row_box of knn_pairs.cuh; swept on config 2 plus one or eight structures of 100 / 280 / 900 atoms —
            // flat between 80 and 160 per 32 pair-cells, 800 to 2000 per row; half of that left a warp 20 us behind)
            const float ckb = 120.f * (float)mloc / 32.f + 800.f / (float)N;
            // cutoff, scan kernel (cut_scan.cuh), in cycles a warp spends (fit on BASELINE configs[2], per-warp
            // clocks of an MG_PHASE_CLOCKS build): per block of 32 pairs 735 + 182 per group of four cells it
            // evaluates (two groups per trip), 17 per edge, 4000 per structure visited; a structure the
            // pair-lane path does not take costs about 25 per candidate cell of a pair
            float groups = 0.f;
            for (int w0 = 0; w0 < mloc; w0 += 32) groups += (float)((((min(32, mloc - w0) + 3) >> 2) + 1) & ~1);
            const float cscan = (MG_CS_BLOCK + MG_CS_GROUP * groups) * (1.f / 32.f) + MG_CS_EDGE * lam / (float)N +
                                MG_CS_STRUCT / ((float)N * (float)N);
            const float crow = MG_CS_ROWCELL * (float)mloc + MG_CS_EDGE * lam / (float)N + MG_CS_STRUCT / ((float)N * (float)N);
            const bool rows = N > MG_SMALL_MAX_ATOMS || mloc > MG_PAIR_TL;
            // K2 cell list (cut_bins.cuh): a large structure in the minimum-image regime; nb_a <= 2 / rho_a slabs
            // (with a margin far above the FP32 rounding of the slab index), one slab where the five-slab
            // stencil would cover the axis anyway, and no more bins than atoms
            float frac = 1.f;
            // (the cutoff graph's scan kernel, and KNN on batches of large structures: knn_bins.cu)
            // (... where a small structure gets a list too: one bin, or a few, instead of the growing-radius routine)
            if ((A.k > 0 || A.rows_cost) && A.binlist && (N > MG_SMALL_MAX_ATOMS || A.k > 0) && mloc == 1) {
                int nb[3];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const float f = floorf(2.f / (r.rho[a] * 1.0001f));
                    nb[a] = f >= (float)MGB_MINSLAB ? (int)fminf(f, (float)MGB_MAXSLAB) : 1;
                }
                while (nb[0] * nb[1] * nb[2] > N) {
                    const int a = nb[0] >= nb[1] && nb[0] >= nb[2] ? 0 : (nb[1] >= nb[2] ? 1 : 2);
                    nb[a] = nb[a] > MGB_MINSLAB ? nb[a] - 1 : 1;
                }
                r.bins = nb[0] | (nb[1] << 8) | (nb[2] << 16) | (1 << 24);
                {
                    const unsigned slot = atomicAdd(A.ctl + 13, 1u);
                    if (slot < (unsigned)A.n_struct) A.binlist[slot] = s;      // (always, unless a failed call left its count behind)
                }
#pragma unroll
                for (int a = 0; a < 3; ++a) frac *= nb[a] > 1 ? 5.f / (float)nb[a] : 1.f;
            }
            const float cbin = MG_CS_BINCAND * frac + MG_CS_BINROW / (float)N + MG_CS_EDGE * lam / (float)N +
                               MG_CS_STRUCT / ((float)N * (float)N);
            const float cnew = 0.25f * (r.bins ? cbin : (rows ? crow : cscan));   // (quarter cycles: keeps the prefix far from overflow)
            r.paircost = (unsigned)fminf(16.f * (A.k > 0 ? (N > MG_SMALL_MAX_ATOMS ? ckb : ck) : (A.rows_cost ? cnew : c)) + 1.f, 16777216.f);
        }
        cost = (unsigned long long)((long long)N * N) * r.paircost;
    }
    // ---- block-wide exclusive scan of the cost
    unsigned long long incl = cost;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned long long woff = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < MG_CP_BLOCK / 32; ++w) {
        if (w < warp) woff += s_warp[w];
        btotal += s_warp[w];
    }
    if (s < A.n_struct) {
        r.lpre = woff + incl - cost;
        A.rec[s] = r;
    }
    if (threadIdx.x == 0) A.bpre[blockIdx.x] = btotal;
    if (A.n_sblocks <= 32) return;        // few blocks: the graph kernels scan the raw sums themselves
    // ---- last block out: exclusive scan of the block sums (serial per thread chunk, 64 bit)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(A.ctl + 7, 1u) == (unsigned)A.n_sblocks - 1u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    __shared__ unsigned long long s_part[MG_CP_BLOCK];
    const int nb = A.n_sblocks, per = (nb + MG_CP_BLOCK - 1) / MG_CP_BLOCK;
    const int b = threadIdx.x * per, e = min(nb, b + per);
    unsigned long long sum = 0ull;
    for (int g = b; g < e; ++g) sum += __ldcg(A.bpre + g);
    s_part[threadIdx.x] = sum;
    __syncthreads();
    unsigned long long off = 0ull;
    for (int w = 0; w < (int)threadIdx.x; ++w) off += s_part[w];
    for (int g = b; g < e; ++g) {
        const unsigned long long v = __ldcg(A.bpre + g);
        A.bpre[g] = off;
        off += v;
    }
    if (threadIdx.x == MG_CP_BLOCK - 1) { A.bpre[nb] = off; A.ctl[7] = 0u; }
}
