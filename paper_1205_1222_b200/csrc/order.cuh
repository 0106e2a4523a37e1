// order.cuh -- spatial ordering of the active rows (part of S2, the i-setup).
//
// The paper holds one i-particle per thread and broadcasts every j to all threads of a block; which
// i share a block does not matter there, because its kernel does the same work for every pair.  Here it does:
// the force kernel takes its near path (low words, neighbour test, list append) for a j-pair as soon as ONE of the
// 32 rows of a warp is close to it (force.cuh).  With the rows of a warp scattered over the cluster that happens
// 32 times as often as for one row; with 32 rows that are neighbours in space their near sets almost coincide.
// So the rows are processed in Morton (Z-curve) order of their predicted positions: a 24-bit key, 8 bits per
// coordinate over the bounding box of the active particles (measured: 8 bits order as well as 10 or 16, 6 bits
// lose 1.5 %; 24 bits are three passes of the library's radix sort instead of four).  Outputs still go to the caller's row numbers: the
// kernels map "logical row" -> caller's row through the permutation built here.  Measured with pre-sorted rows
// (B200): config 5 1055 -> 1116 Gpairs/s, config 3 953 -> 1048, config 4 940 -> 991.
//
//   n_i <= kSmallSort : one CTA computes the box and the keys and sorts them with the library's block-wide radix
//                       sort (one launch).
//   larger blocks     : bbox_kernel (block reductions + atomics on order-preserving integer images of the floats),
//                       key_kernel (keys + identity payload; its last block re-zeroes the box words, which live in
//                       the zero-between-calls scratch), then a library radix sort of (key, row) pairs (CUB).
#pragma once
#include <cub/block/block_radix_sort.cuh>

#include "nbreg_common.cuh"
#include "record.cuh"

namespace nbreg {

constexpr int kSmallSort = 8192;      // rows the one-CTA sort handles
constexpr int kSmallSortRadixBits = 5;  // 24-bit keys in five passes (measured: 4 bits +1 %, 6 bits equal)
constexpr int kOrderThreads = 256;

struct OrderArgs {
    RawState raw;           // from_raw: the registered fp64 state and the time to predict to
    bool from_raw;          // the context holds no prediction (fused-prediction call): predict the rows' positions here
    const float4* packed;   // pair-interleaved predicted records (nbreg_common.cuh)
    const int32_t* i_idx;   // [n_i]
    int32_t n_i;
    uint32_t* box;          // [6] order-preserving images: max of x, y, z and max of the complemented images (= min)
    int32_t* ticket;        // [1]
    uint32_t* keys;         // [n_i] out (large path)
    int32_t* rows;          // [n_i] out: identity payload (large path) / the permutation (small path)
};

// float -> uint32 whose unsigned order is the float order (and 0 is below every image of a finite float)
__device__ __forceinline__ uint32_t ordered(float f) {
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float unordered(uint32_t o) {
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}
constexpr int kKeyBits = 24;  // 8 per coordinate
// spread the low 8 bits of v to every third bit
__device__ __forceinline__ uint32_t spread8(uint32_t v) {
    v &= 0xffu;
    v = (v | (v << 8)) & 0x0300f00fu;
    v = (v | (v << 4)) & 0x030c30c3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
__device__ __forceinline__ uint32_t morton_key(float x, float y, float z, const float lo[3], const float scale[3]) {
    const uint32_t qx = (uint32_t)fminf(fmaxf((x - lo[0]) * scale[0], 0.f), 255.f);
    const uint32_t qy = (uint32_t)fminf(fmaxf((y - lo[1]) * scale[1], 0.f), 255.f);
    const uint32_t qz = (uint32_t)fminf(fmaxf((z - lo[2]) * scale[2], 0.f), 255.f);
    return spread8(qx) | (spread8(qy) << 1) | (spread8(qz) << 2);
}
__device__ __forceinline__ float3 row_position(const OrderArgs& a, int32_t q) {
    if (a.from_raw) {  // the same high words the predictor would have written: the same keys, the same order
        const PredRecord r = predict_record(a.raw, a.i_idx[q]);
        return make_float3(r.xh, r.yh, r.zh);
    }
    // the high words of particle i in its pair record: { xh0, xh1, yh0, yh1 } { zh0, zh1, .. }
    const int32_t i = a.i_idx[q];
    const float* rec = reinterpret_cast<const float*>(a.packed + (size_t)(i >> 1) * kQuadsPerPair) + (i & 1);
    return make_float3(__ldg(rec), __ldg(rec + 2), __ldg(rec + 4));
}
__device__ __forceinline__ void box_scale(const uint32_t box[6], float lo[3], float scale[3]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float hi = unordered(box[c]);
        lo[c] = unordered(~box[3 + c]);
        const float ext = hi - lo[c];
        scale[c] = ext > 0.f ? 256.f / ext : 0.f;
    }
}

// ---- small blocks: everything in one CTA (box, keys, block-wide radix sort of (key, row) pairs from the library).
// Two sizes: 512 threads x 8 rows and 1024 x 8 (measured at N = 65536: 1024 x 16 loses to the device-wide sort at
// 16384 rows, 1.149 against 1.134 ms per call).  The sort's temporary storage goes to dynamic shared memory.
template <int THREADS, int ITEMS>
struct OrderSmall {
    using BlockSort = cub::BlockRadixSort<uint32_t, THREADS, ITEMS, int32_t, kSmallSortRadixBits>;
    static constexpr size_t smem_bytes = sizeof(typename BlockSort::TempStorage);
};

template <int THREADS, int ITEMS>
__global__ void __launch_bounds__(THREADS) order_small_kernel(OrderArgs a) {
    using BlockSort = typename OrderSmall<THREADS, ITEMS>::BlockSort;
    extern __shared__ __align__(16) unsigned char order_smem[];
    typename BlockSort::TempStorage& sort_storage = *reinterpret_cast<typename BlockSort::TempStorage*>(order_smem);
    __shared__ uint32_t box[6];
    const int tid = threadIdx.x;
    if (tid < 6) box[tid] = 0u;
    __syncthreads();
    pdl_wait();
    uint32_t m[6] = {0u, 0u, 0u, 0u, 0u, 0u};
    for (int q = tid; q < a.n_i; q += THREADS) {
        const float3 p = row_position(a, q);
        const uint32_t o[3] = {ordered(p.x), ordered(p.y), ordered(p.z)};
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            m[c] = max(m[c], o[c]);
            m[3 + c] = max(m[3 + c], ~o[c]);
        }
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) m[c] = max(m[c], __shfl_xor_sync(0xffffffffu, m[c], off));
    }
    if ((tid & 31) == 0) {
#pragma unroll
        for (int c = 0; c < 6; ++c) atomicMax(&box[c], m[c]);
    }
    __syncthreads();
    float lo[3], scale[3];
    box_scale(box, lo, scale);
    uint32_t key[ITEMS];
    int32_t row[ITEMS];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const int q = tid * ITEMS + k;  // blocked arrangement: a stable sort keeps equal keys in row order
        key[k] = (1u << kKeyBits) - 1u;  // padding: the largest key; the sort is stable and padding has the largest q, so it stays last
        if (q < a.n_i) {
            const float3 p = row_position(a, q);  // second read of the record: an L2 hit, cheaper than 3 registers per row
            key[k] = morton_key(p.x, p.y, p.z, lo, scale);
        }
        row[k] = q;
    }
    BlockSort(sort_storage).Sort(key, row, 0, kKeyBits);
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
        const int q = tid * ITEMS + k;
        if (q < a.n_i) a.rows[q] = row[k];
    }
}

// ---- large blocks, step 1: bounding box of the active particles
__global__ void __launch_bounds__(kOrderThreads) bbox_kernel(OrderArgs a) {
    uint32_t m[6] = {0u, 0u, 0u, 0u, 0u, 0u};
    for (int64_t q = (int64_t)blockIdx.x * kOrderThreads + threadIdx.x; q < a.n_i; q += (int64_t)gridDim.x * kOrderThreads) {
        const float3 p = row_position(a, (int32_t)q);
        const uint32_t o[3] = {ordered(p.x), ordered(p.y), ordered(p.z)};
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            m[c] = max(m[c], o[c]);
            m[3 + c] = max(m[3 + c], ~o[c]);
        }
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) m[c] = max(m[c], __shfl_xor_sync(0xffffffffu, m[c], off));
    }
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int c = 0; c < 6; ++c) atomicMax(a.box + c, m[c]);
    }
}

// ---- large blocks, step 2: keys and identity payload; the last block leaves the box words zeroed again
__global__ void __launch_bounds__(kOrderThreads) key_kernel(OrderArgs a) {
    __shared__ uint32_t box[6];
    if (threadIdx.x < 6) box[threadIdx.x] = a.box[threadIdx.x];
    __syncthreads();
    float lo[3], scale[3];
    box_scale(box, lo, scale);
    const int64_t q = (int64_t)blockIdx.x * kOrderThreads + threadIdx.x;
    if (q < a.n_i) {
        const float3 p = row_position(a, (int32_t)q);
        a.keys[q] = morton_key(p.x, p.y, p.z, lo, scale);
        a.rows[q] = (int32_t)q;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(a.ticket, 1) == (int32_t)gridDim.x - 1) {
#pragma unroll
            for (int c = 0; c < 6; ++c) a.box[c] = 0u;
            *a.ticket = 0;
        }
    }
}

}  // namespace nbreg
