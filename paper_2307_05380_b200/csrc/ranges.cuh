// ranges.cuh — what the graph kernels share: the cost-balanced ranges of ordered pairs (K6 batching,
// SURVEY.md 8(a); the cost prefix comes from cut_prep.cuh), pair-index arithmetic, coordinate wrapping and
// the packed FP32 distance filter.
#pragma once
#include "common.cuh"
#include "cut_prep.cuh"

// What the range walk needs (shared by the cutoff and the KNN kernels).
struct RangeCtx {
    const CutRec *rec;
    const unsigned long long *bpre;
    int n_blocks, n_struct, n_ranges;
    // n_blocks <= 32: the prep kernel leaves the raw block sums in bpre and every warp scans them
    // itself (lane b holds the exclusive prefix of block b): no last-block phase in the prep kernel
    bool small;
    unsigned long long my_pre, total;
};

__device__ __forceinline__ void mg_range_init(RangeCtx &RC, const CutRec *rec, const unsigned long long *bpre,
                                              int n_blocks, int n_struct, int n_ranges, int lane) {
    RC.rec = rec; RC.bpre = bpre; RC.n_blocks = n_blocks; RC.n_struct = n_struct; RC.n_ranges = n_ranges;
    RC.small = n_blocks <= 32;
    if (RC.small) {
        const unsigned long long v = lane < n_blocks ? __ldg(bpre + lane) : 0ull;
        unsigned long long incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += t;
        }
        RC.my_pre = incl - v;
        RC.total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    } else {
        RC.my_pre = 0ull;
        RC.total = __ldg(bpre + n_blocks);
    }
}

// Cost prefix of prep block b (b warp-uniform).
__device__ __forceinline__ unsigned long long mg_block_pre(const RangeCtx &RC, int b) {
    return RC.small ? __shfl_sync(0xFFFFFFFFu, RC.my_pre, b) : __ldg(RC.bpre + b);
}

// q / n for 0 <= q < 2^20, 1 <= n (exact: (q + 0.5) / n is never within rounding of an integer)
__device__ __forceinline__ int mg_fdiv(int q, float inv_n) {
    return __float2int_rz(__fmul_rn((float)q + 0.5f, inv_n));
}

// Pair index q -> (i, j), q = i N + j.
__device__ __forceinline__ void mg_qsplit(int q, int N, float inv_N, int &i, int &j) {
    i = N <= 1024 ? mg_fdiv(q, inv_N) : q / N;
    j = q - i * N;
}

// Wrapped fractional coordinates of one atom: x - floor(x), integer parts packed in .w (10 bits per
// axis, biased by 512); .w = 0 marks a non-finite or far-away coordinate.
__device__ __forceinline__ float4 mg_wrap_x(const float *xp) {
    const float x0 = xp[0], x1 = xp[1], x2 = xp[2];
    const float g0 = floorf(x0), g1 = floorf(x1), g2 = floorf(x2);
    const bool ok = fabsf(g0) <= 500.f && fabsf(g1) <= 500.f && fabsf(g2) <= 500.f;   // false for NaN / inf
    const int kk = ((int)g0 + 512) | (((int)g1 + 512) << 10) | (((int)g2 + 512) << 20);
    return make_float4(x0 - g0, x1 - g1, x2 - g2, __int_as_float(ok ? kk : 0));
}


__device__ __forceinline__ float2 mg_add2(float2 a, float2 b) {
    float2 r;
    asm("{\n\t.reg .b64 x, y, z;\n\tmov.b64 x, {%2, %3};\n\tmov.b64 y, {%4, %5};\n\tadd.rn.f32x2 z, x, y;\n\t"
        "mov.b64 {%0, %1}, z;\n\t}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 mg_fma2(float2 a, float2 b, float2 c) {
    float2 r;
    asm("{\n\t.reg .b64 x, y, z, w;\n\tmov.b64 x, {%2, %3};\n\tmov.b64 y, {%4, %5};\n\tmov.b64 z, {%6, %7};\n\t"
        "fma.rn.f32x2 w, x, y, z;\n\tmov.b64 {%0, %1}, w;\n\t}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}
// y = |q + T|^2 - r^2 of four consecutive cells (operation order of the scalar filter).
__device__ __forceinline__ void mg_filter4(const float4 X, const float4 Y, const float4 Z, float2 qx, float2 qy,
                                           float2 qz, float2 nr2, float (&y)[4]) {
    const float2 vx0 = mg_add2(qx, make_float2(X.x, X.y)), vx1 = mg_add2(qx, make_float2(X.z, X.w));
    const float2 vy0 = mg_add2(qy, make_float2(Y.x, Y.y)), vy1 = mg_add2(qy, make_float2(Y.z, Y.w));
    const float2 vz0 = mg_add2(qz, make_float2(Z.x, Z.y)), vz1 = mg_add2(qz, make_float2(Z.z, Z.w));
    const float2 y0 = mg_fma2(vz0, vz0, mg_fma2(vy0, vy0, mg_fma2(vx0, vx0, nr2)));
    const float2 y1 = mg_fma2(vz1, vz1, mg_fma2(vy1, vy1, mg_fma2(vx1, vx1, nr2)));
    y[0] = y0.x; y[1] = y0.y; y[2] = y1.x; y[3] = y1.y;
}


// Cost range of warp w: [c0, c1); the last warp takes everything that is left.
__device__ __forceinline__ void mg_warp_range(const RangeCtx &A, int w, unsigned long long &c0,
                                              unsigned long long &c1) {
    const unsigned long long total = A.total;
    const unsigned long long chunk = (total + (unsigned)A.n_ranges - 1) / (unsigned)A.n_ranges;
    c0 = (unsigned long long)w * chunk;
    c1 = w == A.n_ranges - 1 ? ~0ull : c0 + chunk;
}

// First (structure, pair) of the range that starts at cost c0: the first pair whose cost prefix
// bpre[s / MG_CP_BLOCK] + rec[s].lpre + q * paircost is >= c0.
__device__ inline void mg_range_start(const RangeCtx &A, unsigned long long c0, int &s_out, int &q_out, int lane) {
    int lo = 0, hi = A.n_blocks;                   // last prep block b with bpre[b] <= c0 (32-ary search)
    if (A.small) {
        lo = max(1, __popc(__ballot_sync(0xFFFFFFFFu, lane < A.n_blocks && A.my_pre <= c0))) - 1;
        hi = lo + 1;
    }
    while (hi - lo > 1) {
        const int step = (hi - lo + 31) / 32;
        const int idx = lo + (lane + 1) * step;
        const bool ok = idx < hi && __ldg(A.bpre + idx) <= c0;
        lo += __popc(__ballot_sync(0xFFFFFFFFu, ok)) * step;
        hi = min(hi, lo + step);
    }
    const int b = lo;
    const unsigned long long bp = mg_block_pre(A, b);
    int cnt = 0;                                   // structures of the block whose prefix is <= c0
#pragma unroll
    for (int x = 0; x < MG_CP_BLOCK / 32; ++x) {
        const int s = b * MG_CP_BLOCK + x * 32 + lane;
        const bool ok = s < A.n_struct && bp + A.rec[s].lpre <= c0;
        cnt += __popc(__ballot_sync(0xFFFFFFFFu, ok));
    }
    int s = b * MG_CP_BLOCK + max(cnt, 1) - 1;
    const CutRec *R = A.rec + s;
    const unsigned long long cs = bp + R->lpre;
    const unsigned pc = R->paircost;
    const unsigned long long q = c0 > cs ? (c0 - cs + pc - 1) / pc : 0ull;
    if (q >= (unsigned long long)(R->natoms * R->natoms)) { s_out = s + 1; q_out = 0; }   // later pairs start >= c0
    else { s_out = s; q_out = (int)q; }
}

// The part [qa, qb) of structure s's pairs that belongs to the range ending at cost c1 (qa is
// given: 0, or the range's first pair).  Returns false when the range ends before qa.
__device__ __forceinline__ bool mg_segment(const RangeCtx &A, const CutRec *R, int s, int qa,
                                           unsigned long long c1, int &qb) {
    const unsigned long long cs = mg_block_pre(A, s / MG_CP_BLOCK) + R->lpre;
    const unsigned pc = R->paircost;
    const int NN = R->natoms * R->natoms;
    if (cs + (unsigned long long)qa * pc >= c1) return false;
    // pairs that start before c1: ceil((c1 - cs) / pc), at most NN
    if (c1 == ~0ull || c1 - cs >= (unsigned long long)NN * pc) { qb = NN; return true; }
    qb = (int)((c1 - cs + pc - 1) / pc);
    return true;
}

