// gather.cuh -- S5: cross-CTA partial-sum reduction and neighbour-list gathering for the j-split path.
//
// "partial forces and partial neighbour lists ... are distributed for multiple thread-blocks ... we prepared
// kernels for force reduction and list gathering ... Partial forces are summed and sparsely scattered partial
// lists are serialized to a linear array".  Here: one warp per row; lanes run over the
// row's j-chunks.  Sums: fp64, lane-strided then a fixed xor-shuffle tree, so the result is deterministic.
// Lists: the chunks were scanned in ascending j, so concatenating them in chunk order gives an ascending
// list; a warp ballot finds the (few) non-empty chunks, a shuffle scan of the chunk counts gives each its
// offset, and the entries are copied with coalesced lane-parallel loads/stores.
#pragma once
#include "nbreg_common.cuh"

namespace nbreg {

struct GatherArgs {
    int32_t n_i;
    int32_t n_chunks;
    int32_t cap;
    const double* part_sum;    // [rows][S][6]
    const int32_t* part_cnt;   // [rows][S]
    const int32_t* part_list;  // [rows][S][cap]
    double* acc;
    double* jerk;
    int32_t* nbr_count;
    int32_t* nbr_list;
    int32_t* n_overflow;
};

constexpr int kGatherWarps = 4;

__global__ void __launch_bounds__(kGatherWarps * 32) reduce_gather_kernel(GatherArgs a) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * kGatherWarps + (threadIdx.x >> 5);
    if (row >= a.n_i) return;  // warp-uniform
    const int S = a.n_chunks;
    const size_t rbase = (size_t)row * S;

    // ---- partial sums (fixed order: chunk = lane, lane + 32, ...; then xor tree 16, 8, 4, 2, 1)
    double s[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int c = lane; c < S; c += 32) {
        const double* ps = a.part_sum + (rbase + c) * 6;
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k] += ps[k];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(0xffffffffu, s[k], off);
    }
    if (lane < 3) {
        a.acc[row * 3 + lane] = (lane == 0) ? s[0] : (lane == 1) ? s[1] : s[2];
        a.jerk[row * 3 + lane] = (lane == 0) ? s[3] : (lane == 1) ? s[4] : s[5];
    }

    // ---- lists: compact the non-empty chunks into the row, ascending j
    int32_t* out = a.nbr_list + (size_t)row * a.cap;
    int32_t base = 0;
    for (int c0 = 0; c0 < S; c0 += 32) {
        const int c = c0 + lane;
        const int32_t cn = (c < S) ? a.part_cnt[rbase + c] : 0;
        int32_t incl = cn;  // inclusive scan over lanes
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int32_t v = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += v;
        }
        const int32_t excl = incl - cn;
        uint32_t nonempty = __ballot_sync(0xffffffffu, cn > 0);
        while (nonempty) {  // popc(nonempty) iterations, warp-uniform
            const int src = __ffs(nonempty) - 1;
            nonempty &= nonempty - 1;
            const int32_t n_src = min(__shfl_sync(0xffffffffu, cn, src), a.cap);  // a partial list holds <= cap
            const int32_t off = base + __shfl_sync(0xffffffffu, excl, src);
            const int32_t* in = a.part_list + (rbase + c0 + src) * a.cap;
            for (int32_t e = lane; e < n_src; e += 32) {
                if (off + e < a.cap) out[off + e] = in[e];
            }
        }
        base += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) {
        a.nbr_count[row] = base;  // true count, may exceed cap
        if (base > a.cap) atomicAdd(a.n_overflow, 1);
    }
}

}  // namespace nbreg
