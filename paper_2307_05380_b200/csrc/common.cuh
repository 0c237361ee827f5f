// common.cuh — shared device helpers of libmatgraph (sm_100a only).
//
// Nothing here is shared with oracle/ (the FP64 CPU checker): the exact-predicate routine below
// restates Def. 3 in the operation order DESIGN.md R15 fixes, independently.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MG_SMALL_MAX_ATOMS 64      // structures up to this size take the pair-lane "small" path
#define MG_PAIR_TL 320             // cells of the per-warp translation table of the fused cutoff kernel
#define MG_BLOCK 128               // threads per CTA of the graph kernels
#define MG_WARPS (MG_BLOCK / 32)

// device status word bits (first error wins when decoded by mg_check)
#define MGS_SINGULAR   1u
#define MGS_NONFINITE  2u
#define MGS_OFFSET     4u
#define MGS_CAPACITY   8u
#define MGS_UNSUPPORTED 16u

// Per-structure record written by mg_prep_kernel (plane spacings, coordinate extents) and read by the
// warp-per-atom KNN kernel (knn_small.cuh).
struct StructRec {
    float volume;
    unsigned err;       // MGS_* bits
    float h_dn[3];      // plane spacings rounded down  (KNN bounds)
    float invh_up[3];   // 1 / h rounded up
    float xmin[3], xmax[3];
    float amax[3];      // max |component| of each lattice row (rounding-window bound)
    int first, natoms;
    int pad[13];
};
static_assert(sizeof(StructRec) == 128, "StructRec is two 64-byte lines");

// First statement of a kernel launched with programmatic stream serialisation: wait until the
// kernel before it on the stream has completed and its writes are visible (a no-op otherwise).
__device__ __forceinline__ void mg_grid_dependency_wait() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

__device__ __forceinline__ double mg_dot3(const double *u, const double *v) {
    return u[0] * v[0] + u[1] * v[1] + u[2] * v[2];
}

// Plane spacings h_a = V / |a_b x a_c| (BASELINE.json north_star), in FP64 from
// the FP32 lattice.  Returns MGS_* error bits; vol and h are valid only when 0 is returned.
__device__ inline unsigned mg_cell_spacings(const float *lat9, double *vol, double h[3]) {
    double A[3][3];
    bool finite = true;
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
            A[r][c] = (double)lat9[3 * r + c];
            finite = finite && isfinite(A[r][c]);
        }
    if (!finite) return MGS_NONFINITE;
    double c12[3] = {A[1][1] * A[2][2] - A[1][2] * A[2][1], A[1][2] * A[2][0] - A[1][0] * A[2][2],
                     A[1][0] * A[2][1] - A[1][1] * A[2][0]};
    double c20[3] = {A[2][1] * A[0][2] - A[2][2] * A[0][1], A[2][2] * A[0][0] - A[2][0] * A[0][2],
                     A[2][0] * A[0][1] - A[2][1] * A[0][0]};
    double c01[3] = {A[0][1] * A[1][2] - A[0][2] * A[1][1], A[0][2] * A[1][0] - A[0][0] * A[1][2],
                     A[0][0] * A[1][1] - A[0][1] * A[1][0]};
    double V = fabs(mg_dot3(A[0], c12));
    if (!(V > 1e-9) || !isfinite(V)) return MGS_SINGULAR;
    h[0] = V / sqrt(mg_dot3(c12, c12));
    h[1] = V / sqrt(mg_dot3(c20, c20));
    h[2] = V / sqrt(mg_dot3(c01, c01));
    *vol = V;
    return 0u;
}

// Same as mg_cell_spacings but the three 1/|a_b x a_c| come from FP32 rsqrt (relative error
// < 1e-6; callers inflate): cross products, V and the validity test stay FP64.
__device__ inline unsigned mg_cell_spacings_fast(const float *lat9, double *vol, double h[3]) {
    double A[3][3];
    bool finite = true;
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
            A[r][c] = (double)lat9[3 * r + c];
            finite = finite && isfinite(A[r][c]);
        }
    if (!finite) return MGS_NONFINITE;
    double c12[3] = {A[1][1] * A[2][2] - A[1][2] * A[2][1], A[1][2] * A[2][0] - A[1][0] * A[2][2],
                     A[1][0] * A[2][1] - A[1][1] * A[2][0]};
    double c20[3] = {A[2][1] * A[0][2] - A[2][2] * A[0][1], A[2][2] * A[0][0] - A[2][0] * A[0][2],
                     A[2][0] * A[0][1] - A[2][1] * A[0][0]};
    double c01[3] = {A[0][1] * A[1][2] - A[0][2] * A[1][1], A[0][2] * A[1][0] - A[0][0] * A[1][2],
                     A[0][0] * A[1][1] - A[0][1] * A[1][0]};
    const double V = fabs(mg_dot3(A[0], c12));
    if (!(V > 1e-9) || !isfinite(V)) return MGS_SINGULAR;
    const float n0 = (float)mg_dot3(c12, c12), n1 = (float)mg_dot3(c20, c20), n2 = (float)mg_dot3(c01, c01);
    if (!(n0 > 0.f) || !(n1 > 0.f) || !(n2 > 0.f) || !isfinite(n0) || !isfinite(n1) || !isfinite(n2))
        return MGS_SINGULAR;                       // |a_b x a_c|^2 under- or overflows FP32
    const float Vf = (float)V;
    h[0] = (double)(Vf * rsqrtf(n0));
    h[1] = (double)(Vf * rsqrtf(n1));
    h[2] = (double)(Vf * rsqrtf(n2));
    *vol = V;
    return 0u;
}

// Exact FP64 evaluation of one image (Def. 3): f = (x_j - x_i) + tau, v = f . L, no FMA
// contraction, summation left to right (R15).  Returns d^2's square root.
__device__ __forceinline__ double mg_exact_vec(const float *xi, const float *xj, int t0, int t1,
                                               int t2, const float *lat9, double v[3]) {
    const double f0 = __dadd_rn(__dsub_rn((double)xj[0], (double)xi[0]), (double)t0);
    const double f1 = __dadd_rn(__dsub_rn((double)xj[1], (double)xi[1]), (double)t1);
    const double f2 = __dadd_rn(__dsub_rn((double)xj[2], (double)xi[2]), (double)t2);
#pragma unroll
    for (int c = 0; c < 3; ++c)
        v[c] = __dadd_rn(__dadd_rn(__dmul_rn(f0, (double)lat9[c]), __dmul_rn(f1, (double)lat9[3 + c])),
                         __dmul_rn(f2, (double)lat9[6 + c]));
    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(v[0], v[0]), __dmul_rn(v[1], v[1])),
                                __dmul_rn(v[2], v[2]));
    return sqrt(d2);
}

// FP32 filter arithmetic, used identically wherever a candidate is (re-)evaluated.
__device__ __forceinline__ float mg_d2(float qx, float qy, float qz, float tx, float ty, float tz) {
    const float vx = __fadd_rn(qx, tx), vy = __fadd_rn(qy, ty), vz = __fadd_rn(qz, tz);
    return __fmaf_rn(vz, vz, __fmaf_rn(vy, vy, __fmul_rn(vx, vx)));
}

__device__ __forceinline__ unsigned long long mg_ld_acquire(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long mg_ld_relaxed(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void mg_st_release(unsigned long long *p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

