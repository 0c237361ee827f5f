// prep.cuh — K1 (per-structure search bounds) + K6 (batching): one WARP per structure.
//
//  * plane spacings h_a = V / |a_b x a_c| in FP64 from the FP32 lattice, validity (finite, V > 1e-9),
//  * atom -> structure map for the warp-per-atom KNN kernel.
#pragma once
#include "common.cuh"

struct PrepArgs {
    const float *pos;
    const float *lattice;
    const int32_t *struct_ptr;
    int n_struct, n_atoms;
    StructRec *rec;             // [n_struct]
    int32_t *atom_struct;       // [n_atoms]
    unsigned *status;
};

#define MG_PREP_BLOCK 128

__global__ void __launch_bounds__(MG_PREP_BLOCK)
mg_prep_kernel(const PrepArgs A) {
    const int lane = threadIdx.x & 31;
    const int s = blockIdx.x * (MG_PREP_BLOCK / 32) + (threadIdx.x >> 5);
    if (s < A.n_struct) {
        const int first = A.struct_ptr[s];
        const int N = A.struct_ptr[s + 1] - first;
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        float xabs = 1.f;
        bool finite = true;
        for (int j = lane; j < N; j += 32) {
            A.atom_struct[first + j] = s;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float v = A.pos[3 * (size_t)(first + j) + a];
                finite = finite && isfinite(v);
                lo[a] = fminf(lo[a], v);
                hi[a] = fmaxf(hi[a], v);
                xabs = fmaxf(xabs, fabsf(v));
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                lo[a] = fminf(lo[a], __shfl_xor_sync(0xFFFFFFFFu, lo[a], o));
                hi[a] = fmaxf(hi[a], __shfl_xor_sync(0xFFFFFFFFu, hi[a], o));
            }
            xabs = fmaxf(xabs, __shfl_xor_sync(0xFFFFFFFFu, xabs, o));
        }
        finite = __all_sync(0xFFFFFFFFu, finite);
        if (lane == 0) {
            StructRec r;
            r.first = first;
            r.natoms = N;
            float lat[9];
#pragma unroll
            for (int c = 0; c < 9; ++c) lat[c] = A.lattice[9 * (size_t)s + c];
            double vol = 0.0, h[3] = {1.0, 1.0, 1.0};
            unsigned err = mg_cell_spacings(lat, &vol, h);
            if (!finite) err |= MGS_NONFINITE;
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                r.xmin[a] = N ? lo[a] : 0.f;
                r.xmax[a] = N ? hi[a] : 0.f;
                r.h_dn[a] = __double2float_rd(h[a] * (1.0 - 1e-6));
                r.invh_up[a] = __double2float_ru((1.0 + 1e-6) / h[a]);
                r.amax[a] = fmaxf(fabsf(lat[3 * a]), fmaxf(fabsf(lat[3 * a + 1]), fabsf(lat[3 * a + 2])));
            }
            r.volume = (float)vol;
            r.err = err;
            if (err) atomicOr(A.status, err);
#pragma unroll
            for (int c = 0; c < 13; ++c) r.pad[c] = 0;
            A.rec[s] = r;
        }
    }
}
