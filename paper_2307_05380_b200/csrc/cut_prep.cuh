// cut_prep.cuh — K1 (per-structure search bounds) + K6 (batching) of the cutoff graph: one THREAD
// per structure, one launch, decoupled look-back scan of the task counts across the blocks.
//
// For structure s with lattice rows a_0,a_1,a_2 (R5):
//   * plane spacings h_a = V / |a_b x a_c| (BASELINE.json north_star).  The cross
//     products and V are evaluated in FP64 (validity: finite, V > 1e-9), rho_a = r_c / h_a in FP32,
//     inflated so that rho_a is an UPPER bound;
//   * an edge (i, j, tau) has |x_ja - x_ia + tau_a| h_a <= d < r_c (projection on the plane normal,
//     DESIGN.md R14), so for the ordered pair (i, j) only the integers tau_a in the open interval
//     (-rho_a - u_a, rho_a - u_a), u_a = x_ja - x_ia, can be edges: at most m_a = floor(2 rho_a) + 1
//     of them.  The graph kernel evaluates exactly the m_0 m_1 m_2 cells of that per-pair sub-box
//     (a subset of the box |tau_a| <= ceil(r_c / h_a) of north_star);
//   * the rounding window `win` of the FP32 filter (R23);
//   * the split of the structure's source rows into TASKS of about MG_TASK_COST instruction
//     units whose expected edges fit the per-warp stash, the exclusive prefix of the task counts
//     over the batch, and the task -> structure table.
#pragma once
#include "common.cuh"

#define MG_CP_BLOCK 128

struct CutRec {              // 64 bytes
    float rho[3];            // upper bound of r_c / h_a (plus the guard eps)
    float win;               // |d2_fp32 - r_c^2| < win  -> decide in FP64
    int m[3];                // per-pair sub-box: m_a cells along axis a
    int mloc;                // m_0 m_1 m_2; 0: the structure emits nothing (invalid / empty)
    int first, natoms;
    int rpt;                 // source rows per task
    unsigned task0;          // index of the structure's first task
    unsigned err;            // MGS_* bits
    float amax_sum;          // sum_a max_c |L_ac|
    float qmax;              // Q = sum_a (rho_a + 1) max_c |L_ac|
    int pad;
};
static_assert(sizeof(CutRec) == 64, "CutRec is one 64-byte line");

struct CutPrepArgs {
    const float *lattice;
    const int32_t *struct_ptr;
    int n_struct, n_atoms;
    float r_c;
    CutRec *rec;                   // [n_struct]
    unsigned *task_struct;         // [n_atoms + 1] task -> structure
    unsigned long long *pdesc;     // [blocks] look-back descriptors of this kernel
    unsigned *ctl;                 // [6] number of tasks (out), [7] block ticket
    unsigned *status;
    unsigned epoch;
};

#define MG_TASK_COST 24000.f       // instruction units per task (10 per candidate, 50 per edge)
#define MG_STASH 768               // stash entries per buffer (cutoff_pairs.cuh)

__global__ void __launch_bounds__(MG_CP_BLOCK)
mg_cut_prep_kernel(const CutPrepArgs A) {
    __shared__ unsigned s_warp[MG_CP_BLOCK / 32];
    __shared__ unsigned s_block, s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_block = atomicAdd(A.ctl + 7, 1u);     // blocks take chunks in order
    __syncthreads();
    const unsigned blk = s_block;
    const int s = (int)blk * MG_CP_BLOCK + threadIdx.x;
    unsigned ntask = 0;
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
        if (N > MG_SMALL_MAX_ATOMS) err |= MGS_UNSUPPORTED;
        r.mloc = 0;
        r.amax_sum = 0.f;
        float Q = 0.f;
        int mloc = 1;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float amax = fmaxf(fabsf(lat[3 * a]), fmaxf(fabsf(lat[3 * a + 1]), fabsf(lat[3 * a + 2])));
            r.amax_sum += amax;
            // rho = r_c / h rounded up, plus the guard for the FP32 rounding of u and z (the
            // kernel adds the part that grows with |x|)
            const float rho = __double2float_ru((double)A.r_c / h[a] * (1.0 + 4e-6)) + 4e-6f;
            r.rho[a] = rho;
            float mf = floorf(2.f * rho + 1e-5f) + 1.f;
            if (!(mf <= 255.f)) { err |= MGS_OFFSET; mf = 1.f; }
            r.m[a] = (int)mf;
            mloc *= r.m[a];
            Q += (rho + 1.f) * amax;
        }
        if (!err && N > 0) r.mloc = mloc;
        r.qmax = Q;       // Q = sum_a (rho_a + 1) max_c |L_ac| bounds every component of q'; T <= 2Q
        r.win = 0.f;      // completed per task (depends on max |x|): mg_cut_window()
        r.err = err;
        if (err) atomicOr(A.status, err);
        int rpt = 1;
        if (r.mloc > 0) {
            const float lam = (float)N * 4.18879f * A.r_c * A.r_c * A.r_c / (float)vol;   // edges per row
            const float rowcost = (float)N * ((float)((mloc + 3) & ~3) * 10.f + 40.f) + lam * 50.f;
            rpt = (int)(MG_TASK_COST / rowcost);
            const int fit = (int)((float)MG_STASH / (1.2f * lam + 16.f));
            rpt = max(1, min(rpt, min(MG_TASK_ROWS, fit)));
            if (mloc > 128) rpt = 1;                 // several table tiles: one row per task
        } else {
            rpt = MG_TASK_ROWS;                       // rows of invalid structures: row_ptr only
        }
        r.rpt = rpt;
        r.pad = 0;
        ntask = (unsigned)((N + rpt - 1) / rpt);
    }
    // ---- block-wide exclusive scan of ntask
    unsigned incl = ntask;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned woff = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < MG_CP_BLOCK / 32; ++w) {
        if (w < warp) woff += s_warp[w];
        btotal += s_warp[w];
    }
    // ---- decoupled look-back over the blocks before this one (warp 0)
    const unsigned ep = A.epoch & 0x3FFFFFFFu;
    if (warp == 0) {
        if (lane == 0)
            mg_st_release(A.pdesc + blk, mg_desc(blk ? MG_FLAG_AGG : MG_FLAG_PFX, ep, btotal));
        unsigned sum = 0;
        int idx = (int)blk - 1;
        while (idx >= 0) {
            const int u = idx - lane;
            unsigned long long d = mg_desc(MG_FLAG_PFX, ep, 0u);
            if (u >= 0) d = mg_ld_acquire(A.pdesc + u);
            const bool ok = ((unsigned)(d >> 32) & 0x3FFFFFFFu) == ep && (d >> 62) != 0ull;
            const unsigned bad = __ballot_sync(0xFFFFFFFFu, !ok);
            if (bad) continue;                                      // predecessors are running
            const unsigned pfx = __ballot_sync(0xFFFFFFFFu, (d >> 62) == MG_FLAG_PFX);
            const int take = pfx ? __ffs(pfx) : 32;
            unsigned val = lane < take ? (unsigned)d : 0u;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xFFFFFFFFu, val, o);
            sum += val;
            if (pfx) break;
            idx -= 32;
        }
        if (lane == 0) {
            s_base = sum;
            if (blk) mg_st_release(A.pdesc + blk, mg_desc(MG_FLAG_PFX, ep, sum + btotal));
            if (blk == gridDim.x - 1) { A.ctl[6] = sum + btotal; A.ctl[7] = 0u; }
        }
    }
    __syncthreads();
    if (s < A.n_struct) {
        r.task0 = s_base + woff + incl - ntask;
        A.rec[s] = r;
        for (unsigned g = 0; g < ntask; ++g) A.task_struct[r.task0 + g] = (unsigned)s;
    }
}
