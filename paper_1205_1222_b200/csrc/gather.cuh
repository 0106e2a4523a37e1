// gather.cuh -- S5: cross-CTA partial-sum reduction and neighbour-list gathering for the j-split rows.
//
// "partial forces and partial neighbour lists ... are distributed for multiple thread-blocks ... we prepared
// kernels for force reduction and list gathering ... Partial forces are summed and sparsely scattered partial
// lists are serialized to a linear array".  Here: one warp per j-split row.  The kernel runs
// after every force launch (with no rows if nothing was split): its last block publishes n_overflow.
//   Sums: fp64; lanes stride over the row's j-chunks, then a fixed xor-shuffle tree: deterministic.
//   Lists: the chunks' CTAs appended their neighbours to the row's final list in arrival order (atomic slot
//   counter, force.cuh).  Each chunk covers a contiguous j-range and its entries arrive in ascending j, so the
//   ascending order is restored by a stable counting sort on the chunk number, done by the warp: a
//   match_any/popc vote groups the lanes of each 32-entry block by chunk (the warp-vote compaction idiom,
//   ballot + popc), per-chunk counters live in shared memory, a shuffle scan turns them into offsets, and a
//   second pass writes every entry to offset[chunk] + its rank among earlier entries of the same chunk.  O(count + S).
#pragma once
#include "nbreg_common.cuh"
#include "fixflag.cuh"

namespace nbreg {

struct GatherArgs {
    int32_t row0;              // first j-split row (rows below were written directly by the force kernel)
    int32_t n_i;
    const int32_t* perm;       // logical row -> caller's row (null: identity), as in ForceArgs
    int32_t n_chunks;
    int32_t chunk_j;           // j-particles per chunk (a multiple of 4, not of the tile size)
    int32_t cap;
    const double* part_sum;    // [split rows][S][7], or [..][8] with the potential: acc, jerk (, pot), error scales (float2)
    FixupFlag fix;             // rows dominated by cancellation are queued for fixup_kernel (fixflag.cuh)
    double* acc;
    double* jerk;
    double* pot;               // null: no potential (6 partial sums per chunk), else 7
    int32_t* nbr_count;
    int32_t* nbr_list;
    int32_t* n_overflow;
    // zero-between-calls scratch (see ForceArgs): this kernel consumes it and leaves it zeroed for the next call
    int32_t* slot_count;       // [split rows] true counts of the j-split rows, complete when this kernel starts
    int32_t* overflow_ws;      // [1]
    int32_t* ticket;           // [1] blocks of this kernel that are done
    // option "ovf_first_in_j": overflowed j-split rows are queued for overflow_list_kernel (fixup.cuh), which rewrites
    // their lists as the first cap neighbours in ascending j (null: off)
    int32_t* ovf_count;        // [1] (zero between calls)
    int32_t* ovf_rows;         // [n_i_max] caller's rows
};

constexpr int kGatherWarps = 4;

__global__ void __launch_bounds__(kGatherWarps * 32) reduce_gather_kernel(GatherArgs a) {
    extern __shared__ int32_t stage_all[];  // kGatherWarps x (cap + S)
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    pdl_wait();
    const int64_t prow = (int64_t)blockIdx.x * kGatherWarps + warp;  // row among the split rows
    const int64_t row = a.row0 + prow;
    if (row < a.n_i) {  // warp-uniform
    const int64_t orow = a.perm ? a.perm[row] : row;
    const int S = a.n_chunks;
    const size_t rbase = (size_t)prow * S;

    // ---- partial sums (fixed order: chunk = lane, lane + 32, ...; then xor tree 16, 8, 4, 2, 1)
    double s[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    float qa = 0.f, qj = 0.f;  // error scales of the chunks (fixflag.cuh)
    const int n_sums = a.pot ? 7 : 6;
    for (int c = lane; c < S; c += 32) {
        const double* ps = a.part_sum + (rbase + c) * (n_sums + 1);
#pragma unroll
        for (int k = 0; k < 7; ++k)
            if (k < n_sums) s[k] += ps[k];
        const float2 q = *reinterpret_cast<const float2*>(ps + n_sums);
        qa += q.x;
        qj += q.y;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int k = 0; k < 7; ++k) s[k] += __shfl_xor_sync(0xffffffffu, s[k], off);
        qa += __shfl_xor_sync(0xffffffffu, qa, off);
        qj += __shfl_xor_sync(0xffffffffu, qj, off);
    }
    if (lane == 0 && a.pot) a.pot[orow] = s[6];
    if (lane < 3) {
        a.acc[orow * 3 + lane] = (lane == 0) ? s[0] : (lane == 1) ? s[1] : s[2];
        a.jerk[orow * 3 + lane] = (lane == 0) ? s[3] : (lane == 1) ? s[4] : s[5];
    }
    if (lane == 0) fixup_flag(a.fix, (int32_t)orow, qa, qj, s[0], s[1], s[2], s[3], s[4], s[5]);

    // ---- list: stable counting sort of the stored entries by chunk number
    const int32_t cnt = a.slot_count[prow];  // true count, may exceed cap
    __syncwarp();
    if (lane == 0) {
        a.nbr_count[orow] = cnt;
        a.slot_count[prow] = 0;
    }
    const int32_t stored = min(cnt, a.cap);
    int32_t* out = a.nbr_list + (size_t)orow * a.cap;
    int32_t* stage = stage_all + (size_t)warp * (a.cap + S);
    int32_t* bin = stage + a.cap;
    const uint32_t lt_mask = (1u << lane) - 1u;
    for (int32_t e = lane; e < stored; e += 32) stage[e] = out[e];
    for (int c = lane; c < S; c += 32) bin[c] = 0;
    __syncwarp();
    for (int32_t e0 = 0; e0 < stored; e0 += 32) {  // pass 1: entries per chunk
        const int32_t e = e0 + lane;
        const bool valid = e < stored;
        const int32_t c = valid ? stage[e] / a.chunk_j : S;
        const uint32_t peers = __match_any_sync(0xffffffffu, c);
        if (valid && (peers & lt_mask) == 0) bin[c] += __popc(peers);  // one leader per chunk in this block
        __syncwarp();
    }
    int32_t carry = 0;
    for (int c0 = 0; c0 < S; c0 += 32) {  // exclusive scan of the counters -> first slot of each chunk
        const int c = c0 + lane;
        const int32_t x = (c < S) ? bin[c] : 0;
        int32_t incl = x;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int32_t y = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += y;
        }
        if (c < S) bin[c] = carry + incl - x;
        carry += __shfl_sync(0xffffffffu, incl, 31);
    }
    __syncwarp();
    for (int32_t e0 = 0; e0 < stored; e0 += 32) {  // pass 2: scatter, arrival order kept within a chunk
        const int32_t e = e0 + lane;
        const bool valid = e < stored;
        const int32_t v = valid ? stage[e] : 0;
        const int32_t c = valid ? v / a.chunk_j : S;
        const uint32_t peers = __match_any_sync(0xffffffffu, c);
        const int32_t before = __popc(peers & lt_mask);
        if (valid) out[bin[c] + before] = v;
        __syncwarp();
        if (valid && before == 0) bin[c] += __popc(peers);
        __syncwarp();
    }
    if (lane == 0 && cnt > a.cap) {
        atomicAdd(a.overflow_ws, 1);
        if (a.ovf_rows) a.ovf_rows[atomicAdd(a.ovf_count, 1)] = (int32_t)orow;
    }
    }  // row < n_i

    // ---- the last block to finish publishes the overflow count of the whole call and re-zeroes the scratch
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(a.ticket, 1) == (int32_t)gridDim.x - 1) {
            *a.n_overflow = atomicExch(a.overflow_ws, 0);
            *a.ticket = 0;
        }
    }
}

// The same job with one BLOCK per row, for rows split into many chunks (small active blocks: hundreds of chunks per
// row and few rows, so a warp per row would leave the machine empty and walk the chunks serially).
//   Sums: the threads stride over the chunks, xor-shuffle tree per warp, then the warp sums are added in
//   warp order: fixed order, deterministic.
//   List: ascending j is plain ascending VALUE, and a row holds few entries compared with its chunks, so each
//   thread ranks one entry against the staged row (rank = number of smaller entries; entries are distinct) and
//   stores it at its rank: O(count^2 / threads) instead of O(chunks).
// Threads per row: 128, or 512 when there are few rows (at most kWideFewRows: then the blocks do not fill the SMs
// anyway, and 2048 chunks are 4 dependent rounds of loads per thread instead of 16).  With many rows 512-thread
// blocks lose: fewer resident blocks, most threads idle in the rank sort (measured: N_i = 4096, 321 -> 340 us).
constexpr int kWideThreads = 128;
constexpr int kWideThreadsFew = 512;
constexpr int64_t kWideFewRows = 296;

__global__ void __launch_bounds__(kWideThreadsFew) reduce_gather_wide_kernel(GatherArgs a) {
    extern __shared__ int32_t stage[];  // cap entries
    __shared__ double warp_sum[kWideThreadsFew / 32][7];
    __shared__ float2 warp_q[kWideThreadsFew / 32];
    __shared__ double row_sum[6];
    const int n_threads = blockDim.x;  // kWideThreads or kWideThreadsFew
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_wait();
    const int64_t prow = blockIdx.x;
    const int64_t lrow = a.row0 + prow;  // grid = split rows exactly
    const int64_t row = a.perm ? a.perm[lrow] : lrow;  // the caller's row
    const int S = a.n_chunks;
    const size_t rbase = (size_t)prow * S;

    double s[7] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    float qa = 0.f, qj = 0.f;  // error scales of the chunks (fixflag.cuh)
    const int n_sums = a.pot ? 7 : 6;
    for (int c = tid; c < S; c += n_threads) {
        const double* ps = a.part_sum + (rbase + c) * (n_sums + 1);
#pragma unroll
        for (int k = 0; k < 7; ++k)
            if (k < n_sums) s[k] += ps[k];
        const float2 q = *reinterpret_cast<const float2*>(ps + n_sums);
        qa += q.x;
        qj += q.y;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int k = 0; k < 7; ++k) s[k] += __shfl_xor_sync(0xffffffffu, s[k], off);
        qa += __shfl_xor_sync(0xffffffffu, qa, off);
        qj += __shfl_xor_sync(0xffffffffu, qj, off);
    }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 7; ++k) warp_sum[warp][k] = s[k];
        warp_q[warp] = make_float2(qa, qj);
    }
    const int32_t cnt = a.slot_count[prow];  // true count, may exceed cap
    const int32_t stored = min(cnt, a.cap);
    int32_t* out = a.nbr_list + (size_t)row * a.cap;
    for (int32_t e = tid; e < stored; e += n_threads) stage[e] = out[e];
    __syncthreads();
    if (tid < 7 && tid < n_sums) {
        double v = warp_sum[0][tid];
        for (int w = 1; w < n_threads / 32; ++w) v += warp_sum[w][tid];  // fixed order
        if (tid < 3) a.acc[row * 3 + tid] = v;
        else if (tid < 6) a.jerk[row * 3 + tid - 3] = v;
        else a.pot[row] = v;
        if (tid < 6) row_sum[tid] = v;
    }
    for (int32_t e = tid; e < stored; e += n_threads) {
        const int32_t v = stage[e];
        int32_t rank = 0;
        for (int32_t k = 0; k < stored; ++k) rank += stage[k] < v;  // broadcast reads
        out[rank] = v;
    }
    __syncthreads();
    if (tid == 0) {
        a.nbr_count[row] = cnt;
        a.slot_count[prow] = 0;
        if (cnt > a.cap) {
            atomicAdd(a.overflow_ws, 1);
            if (a.ovf_rows) a.ovf_rows[atomicAdd(a.ovf_count, 1)] = (int32_t)row;
        }
        float qa = 0.f, qj = 0.f;
        for (int w = 0; w < n_threads / 32; ++w) {  // fixed order
            qa += warp_q[w].x;
            qj += warp_q[w].y;
        }
        fixup_flag(a.fix, (int32_t)row, qa, qj, row_sum[0], row_sum[1], row_sum[2], row_sum[3], row_sum[4], row_sum[5]);
        __threadfence();
        if (atomicAdd(a.ticket, 1) == (int32_t)gridDim.x - 1) {
            *a.n_overflow = atomicExch(a.overflow_ws, 0);
            *a.ticket = 0;
        }
    }
}

// Longest stored list of a block of rows, max_q min(count[q], cap): lets the host entry point copy back only the
// columns of nbr_list that hold entries.  *out must be zero on entry.
__global__ void __launch_bounds__(256) list_width_kernel(const int32_t* nbr_count, int32_t n_rows, int32_t cap,
                                                         int32_t* out) {
    int32_t m = 0;
    for (int64_t q = (int64_t)blockIdx.x * 256 + threadIdx.x; q < n_rows; q += (int64_t)gridDim.x * 256)
        m = max(m, min(nbr_count[q], cap));
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, off));
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

// Host entry point, CSR form: stored entries min(count, cap) of a row (the scan's input), and the packing of the rows'
// stored entries back to back at their offsets (one warp per row, coalesced).
struct StoredLen {
    const int32_t* cnt;
    int32_t cap;
    __host__ __device__ int64_t operator()(int64_t q) const { return (int64_t)min(cnt[q], cap); }
};

__global__ void __launch_bounds__(kGatherWarps * 32) pack_lists_kernel(const int32_t* nbr_count, const int32_t* nbr_list,
                                                                      int32_t n_rows, int32_t cap, const int64_t* offset,
                                                                      int32_t* packed) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * kGatherWarps + (threadIdx.x >> 5);
    if (row >= n_rows) return;
    const int32_t len = min(nbr_count[row], cap);
    const int32_t* src = nbr_list + (size_t)row * cap;
    int32_t* dst = packed + offset[row];
    for (int32_t e = lane; e < len; e += 32) dst[e] = src[e];
}

}  // namespace nbreg
