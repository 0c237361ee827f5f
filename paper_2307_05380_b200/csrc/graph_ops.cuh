// graph_ops.cuh — operations on a finished CSR edge list.
//
//   symmetric graph (section 3 "Symmetric graph"): the KNN graph is directed; the
//     symmetric graph adds, for every edge (i, j, tau), the reverse edge (j, i, -tau) unless it is there
//     already, and keeps edges unique.  Four launches: flag the edges whose reverse is missing and count
//     them per target row; exclusive scan (two launches) -> the new row_ptr; copy the old rows and append the new edges.
//   triplets (Def. 3: Gamma_2, the pairs of edges that share their source; PAPER.md:131
//     "Triplets generation"): for a source of degree d the d (d - 1) ordered pairs (a, b), a != b, of its
//     edges, as two arrays of edge indices, CSR by source.  Three launches: scan of d (d - 1) (two), emit.
#pragma once
#include "common.cuh"

#define MGO_BLOCK 256
#define MGO_SCAN_BLOCK 1024

// Exclusive scan of v(r), r in [0, n), in two launches of ceil(n / MGO_CHUNK) blocks (no block waits for another):
//   mgo_chunk_total   block b sums the values of its chunk [b MGO_CHUNK, (b + 1) MGO_CHUNK) -> partial[b];
//   mgo_chunk_scan    block b adds up the partials before it, scans its chunk (a thread owns MGO_SCAN_ITEMS consecutive
//                     values) and writes out[r] = base(r) + sum_{q < r} v(q); the last block also out[n] = base(n) +
//                     total and *total_out.
// (One block for all rows took 39 us on the 43 578 rows of BASELINE configs[2]: latency, not work.)
#define MGO_SCAN_ITEMS 8
#define MGO_CHUNK (MGO_SCAN_BLOCK * MGO_SCAN_ITEMS)

__host__ __device__ __forceinline__ int mgo_scan_blocks(int n) { return n > 0 ? (n + MGO_CHUNK - 1) / MGO_CHUNK : 1; }

// sum of x over the block (valid on thread 0 ... and, after the barrier, in *s_out for all)
__device__ __forceinline__ long long mgo_block_sum(long long x, long long *s_warp, long long *s_out) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xFFFFFFFFu, x, o);
    if (lane == 0) s_warp[warp] = x;
    __syncthreads();
    if (tid == 0) {
        long long t = 0ll;
        for (int w = 0; w < MGO_SCAN_BLOCK / 32; ++w) t += s_warp[w];
        *s_out = t;
    }
    __syncthreads();
    return *s_out;
}

template <class V>
__device__ __forceinline__ void mgo_chunk_total(int n, V value, long long *partial) {
    __shared__ long long s_warp[MGO_SCAN_BLOCK / 32];
    __shared__ long long s_sum;
    const int rb = (int)blockIdx.x * MGO_CHUNK + (int)threadIdx.x * MGO_SCAN_ITEMS;
    long long own = 0ll;
#pragma unroll
    for (int x = 0; x < MGO_SCAN_ITEMS; ++x) own += rb + x < n ? value(rb + x) : 0ll;
    const long long t = mgo_block_sum(own, s_warp, &s_sum);
    if (threadIdx.x == 0) partial[blockIdx.x] = t;
}

template <class V, class B>
__device__ __forceinline__ void mgo_chunk_scan(int n, V value, B base, const long long *partial, long long *out64,
                                               int32_t *out32, long long *total_out) {
    __shared__ long long s_warp[MGO_SCAN_BLOCK / 32];
    __shared__ long long s_sum;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // the chunks before this one
    long long before = 0ll;
    for (int q = tid; q < (int)blockIdx.x; q += MGO_SCAN_BLOCK) before += partial[q];
    const long long off = mgo_block_sum(before, s_warp, &s_sum);
    __syncthreads();
    // this chunk
    const int rb = (int)blockIdx.x * MGO_CHUNK + tid * MGO_SCAN_ITEMS;
    long long v[MGO_SCAN_ITEMS], own = 0ll;
#pragma unroll
    for (int x = 0; x < MGO_SCAN_ITEMS; ++x) {
        v[x] = rb + x < n ? value(rb + x) : 0ll;
        own += v[x];
    }
    long long incl = own;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const long long t = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    long long woff = 0ll, btotal = 0ll;
    for (int w = 0; w < MGO_SCAN_BLOCK / 32; ++w) {
        const long long t = s_warp[w];
        if (w < warp) woff += t;
        btotal += t;
    }
    long long excl = off + woff + incl - own;
#pragma unroll
    for (int x = 0; x < MGO_SCAN_ITEMS; ++x) {
        const int r = rb + x;
        if (r < n) {
            if (out64) out64[r] = base(r) + excl;
            if (out32) out32[r] = (int32_t)(base(r) + excl);
        }
        excl += v[x];
    }
    if (tid == 0 && blockIdx.x == gridDim.x - 1) {
        const long long tot = base(n) + off + btotal;
        if (out64) out64[n] = tot;
        if (out32) out32[n] = (int32_t)tot;
        *total_out = tot;
    }
}

// ---- symmetric graph ------------------------------------------------------------------------------
struct SymArgs {
    // input graph (CSR by source)
    const int32_t *row_ptr, *src, *dst;
    const int8_t *offset;
    const float *vec, *dist;
    const long long *n_edges_in;
    long long cap_in;          // edges the input arrays hold: a graph whose own call overflowed (n_edges_in above
                               // it) is read up to here only and reported (MGS_CAPACITY)
    int n_atoms;
    // output graph
    int32_t *o_row_ptr, *o_src, *o_dst;
    int8_t *o_offset;
    float *o_vec, *o_dist;
    long long capacity;
    long long *n_edges_out;
    // scratch
    unsigned char *flag;       // [E_in] 1: the reverse edge is missing
    int *extra;                // [n_atoms] missing reverse edges per target row (zero before the call)
    int *fill;                 // [n_atoms] cursor of the appended edges (zero before the call)
    long long *part;           // [ceil(n_atoms / MGO_CHUNK)] chunk totals of the scan
    unsigned *status;
};

// Edge e = (i, j, tau): is (j, i, -tau) in row j?
__global__ void __launch_bounds__(MGO_BLOCK)
mg_sym_flag_kernel(const SymArgs A) {
    mg_grid_dependency_wait();
    long long E = *A.n_edges_in;
    if (E > A.cap_in) {                                    // an incomplete input graph: no read past its arrays
        E = A.cap_in;
        if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(A.status, MGS_CAPACITY);
    }
    for (long long e = (long long)blockIdx.x * MGO_BLOCK + threadIdx.x; e < E; e += (long long)gridDim.x * MGO_BLOCK) {
        const int i = A.src[e], j = A.dst[e];
        const int t0 = -A.offset[3 * e], t1 = -A.offset[3 * e + 1], t2 = -A.offset[3 * e + 2];
        bool found = false;
        for (long long q = A.row_ptr[j], qe = min((long long)A.row_ptr[j + 1], E); q < qe && !found; ++q)
            found = A.dst[q] == i && A.offset[3 * q] == t0 && A.offset[3 * q + 1] == t1 && A.offset[3 * q + 2] == t2;
        A.flag[e] = found ? 0 : 1;
        if (!found) atomicAdd(A.extra + j, 1);
    }
}

__global__ void __launch_bounds__(MGO_SCAN_BLOCK)
mg_sym_part_kernel(const SymArgs A) {
    mg_grid_dependency_wait();
    mgo_chunk_total(A.n_atoms, [&](int r) { return (long long)A.extra[r]; }, A.part);
}

__global__ void __launch_bounds__(MGO_SCAN_BLOCK)
mg_sym_scan_kernel(const SymArgs A) {
    mg_grid_dependency_wait();
    __shared__ long long s_total;
    if (threadIdx.x == 0) s_total = -1ll;
    mgo_chunk_scan(A.n_atoms, [&](int r) { return (long long)A.extra[r]; },
                   [&](int r) { return (long long)A.row_ptr[r]; }, A.part, nullptr, A.o_row_ptr, &s_total);
    if (threadIdx.x == 0 && blockIdx.x == gridDim.x - 1) {       // (thread 0 of the last block wrote s_total itself)
        const long long total = s_total;
        *A.n_edges_out = total;
        if (total > A.capacity || total > 0x7FFFFFFFll) atomicOr(A.status, MGS_CAPACITY);
    }
}

__global__ void __launch_bounds__(MGO_BLOCK)
mg_sym_emit_kernel(const SymArgs A) {
    mg_grid_dependency_wait();
    const long long E = min(*A.n_edges_in, A.cap_in);
    for (long long e = (long long)blockIdx.x * MGO_BLOCK + threadIdx.x; e < E; e += (long long)gridDim.x * MGO_BLOCK) {
        const int i = A.src[e], j = A.dst[e];
        const int8_t t0 = A.offset[3 * e], t1 = A.offset[3 * e + 1], t2 = A.offset[3 * e + 2];
        const float v0 = A.vec[3 * e], v1 = A.vec[3 * e + 1], v2 = A.vec[3 * e + 2];
        const float d = A.dist ? A.dist[e] : 0.f;
        const long long po = (long long)A.o_row_ptr[i] + (e - A.row_ptr[i]);     // the old rows keep their order
        if (po < A.capacity) {
            A.o_src[po] = i; A.o_dst[po] = j;
            A.o_offset[3 * po] = t0; A.o_offset[3 * po + 1] = t1; A.o_offset[3 * po + 2] = t2;
            A.o_vec[3 * po] = v0; A.o_vec[3 * po + 1] = v1; A.o_vec[3 * po + 2] = v2;
            if (A.o_dist) A.o_dist[po] = d;
        }
        if (A.flag[e]) {                               // append (j, i, -tau) to row j
            const int slot = atomicAdd(A.fill + j, 1);
            const long long pr = (long long)A.o_row_ptr[j] + (A.row_ptr[j + 1] - A.row_ptr[j]) + slot;
            if (pr < A.capacity) {
                A.o_src[pr] = j; A.o_dst[pr] = i;
                A.o_offset[3 * pr] = (int8_t)-t0; A.o_offset[3 * pr + 1] = (int8_t)-t1; A.o_offset[3 * pr + 2] = (int8_t)-t2;
                A.o_vec[3 * pr] = -v0; A.o_vec[3 * pr + 1] = -v1; A.o_vec[3 * pr + 2] = -v2;
                if (A.o_dist) A.o_dist[pr] = d;
            }
        }
    }
}

// ---- triplets -------------------------------------------------------------------------------------
struct TripArgs {
    const int32_t *row_ptr;
    int n_atoms;
    long long *tri_ptr;        // [n_atoms + 1]
    int32_t *edge_a, *edge_b;  // [capacity]
    long long capacity;
    long long *n_triplets;
    long long *part;           // [ceil(n_atoms / MGO_CHUNK)] chunk totals of the scan
    unsigned *status;
};

__global__ void __launch_bounds__(MGO_SCAN_BLOCK)
mg_trip_part_kernel(const TripArgs A) {
    mg_grid_dependency_wait();
    mgo_chunk_total(A.n_atoms, [&](int r) { const long long d = A.row_ptr[r + 1] - A.row_ptr[r]; return d * (d - 1); }, A.part);
}

__global__ void __launch_bounds__(MGO_SCAN_BLOCK)
mg_trip_scan_kernel(const TripArgs A) {
    mg_grid_dependency_wait();
    __shared__ long long s_total;
    if (threadIdx.x == 0) s_total = -1ll;
    mgo_chunk_scan(A.n_atoms,
                   [&](int r) { const long long d = A.row_ptr[r + 1] - A.row_ptr[r]; return d * (d - 1); },
                   [&](int) { return 0ll; }, A.part, A.tri_ptr, nullptr, &s_total);
    if (threadIdx.x == 0 && blockIdx.x == gridDim.x - 1) {
        *A.n_triplets = s_total;
        if (s_total > A.capacity) atomicOr(A.status, MGS_CAPACITY);
    }
}

// One warp per source row (rows handed round): triplet t of the row = (a, b) with a = t / (d - 1) and b
// the (t % (d - 1))-th edge other than a; lanes over t, coalesced 4-byte stores.
__global__ void __launch_bounds__(MGO_BLOCK)
mg_trip_emit_kernel(const TripArgs A) {
    mg_grid_dependency_wait();
    const int lane = threadIdx.x & 31;
    const int wid = (int)((blockIdx.x * MGO_BLOCK + threadIdx.x) >> 5), nw = (int)((gridDim.x * MGO_BLOCK) >> 5);
    for (int r = wid; r < A.n_atoms; r += nw) {
        const int e0 = A.row_ptr[r];
        const long long d = A.row_ptr[r + 1] - e0;
        if (d < 2) continue;
        const long long nt = d * (d - 1), base = A.tri_ptr[r];
        const int dm = (int)(d - 1);
        if (nt < (1ll << 20)) {                        // t / dm through the float reciprocal (exact below 2^20)
            const float inv = 1.f / (float)dm;
            int32_t *pa = A.edge_a + base, *pb = A.edge_b + base;
            const long long room = A.capacity - base;
            const int lim = room >= nt ? (int)nt : (room > 0 ? (int)room : 0);
            for (int t = lane; t < lim; t += 32) {
                const int a = __float2int_rz(__fmul_rn((float)t + 0.5f, inv)), bq = t - a * dm;
                pa[t] = e0 + a;
                pb[t] = e0 + bq + (bq >= a ? 1 : 0);
            }
        } else
            for (long long t = lane; t < nt; t += 32) {
                const int a = (int)(t / dm), bq = (int)(t - (long long)a * dm), b = bq + (bq >= a ? 1 : 0);
                if (base + t < A.capacity) {
                    A.edge_a[base + t] = e0 + a;
                    A.edge_b[base + t] = e0 + b;
                }
            }
    }
}
