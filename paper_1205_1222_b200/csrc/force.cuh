// force.cuh -- S2-S4 + S6: the i-block x j-tile regular-force kernel.
//
// What it computes (step (vi)): for every active row q (particle i, radius r_s) and every
// j != i:  neighbour iff |R_ij|^2 < r_s^2 (eq. (2); eq. (11)) -> index appended to the row's
// list, nothing summed; otherwise eq. (9) acc += m_j R_ij/r^3 and eq. (10)
// jerk += m_j [V_ij/r^3 - 3 (R_ij.V_ij) R_ij/r^5].  The pair arithmetic follows Listing B2:
// the neighbour test zeroes rinv ("rinv1 = 0.f") so the `if` is a select, not a branch
// (PAPER.md:120).
//
// How it maps onto a B200 SM (differs from the paper's Fermi kernel):
//   * one i-particle per thread held in registers, IPT of them per thread;
//   * the packed j-records (nbreg_common.cuh) are streamed tile by tile into shared memory by 1-D bulk async
//     copies (cp.async.bulk + mbarrier, SASS UBLKCP), double-buffered, and broadcast to all threads with
//     LDS.128;
//   * TWO j-particles per instruction: sm_100's packed FP32 pipe (add/mul/fma.f32x2 -> FADD2/FMUL2/FFMA2)
//     evaluates j0 and j1 in the two halves of 64-bit register pairs, which halves the issue slots per pair;
//   * coordinate differences are formed from double-single positions ("pseudo double precision",
//     PAPER.md:17, footnote at PAPER.md:154): (xh_j - xh_i) + (xl_j - xl_i), then fp32 with one MUFU.RSQ;
//   * fp32 partial sums are flushed into fp64 running sums after every j-tile (S6);
//   * the list append sits behind a warp-uniform vote so the common path has no store and no branch taken;
//   * when blockDim.y > 1 the j-range is split over CTAs and the kernel writes per-(row,
//     chunk) partial sums / counts / lists for reduce_gather_kernel (gather.cuh).
#pragma once
#include "nbreg_common.cuh"

namespace nbreg {

struct ForceArgs {
    const float4* packed;   // packed j-pair records, n_pad / 2 pairs
    int32_t n;              // real j-particles
    int32_t n_tiles;        // number of JT-sized tiles covering n_pad
    int32_t tiles_per_chunk;
    int32_t n_chunks;       // S = gridDim.y
    int32_t n_i;
    int32_t cap;
    const int32_t* i_idx;
    const double* r_s;
    // final outputs (used when n_chunks == 1)
    double* acc;
    double* jerk;
    int32_t* nbr_count;
    int32_t* nbr_list;
    int32_t* n_overflow;
    // partial outputs (used when n_chunks > 1): [row][chunk]
    double* part_sum;     // [rows][S][6]
    int32_t* part_cnt;    // [rows][S]
    int32_t* part_list;   // [rows][S][cap]
};

// ---------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// 1-D bulk async copy global -> shared, completion counted in bytes on an mbarrier (TMA engine, no tensor map).
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
#ifdef NBREG_EXP_NEWTON
    { float e = fmaf(x * y, -y, 1.0f); y = fmaf(0.5f * y, e, y); }
#endif
    return y;
}

// ---------------------------------------------------------------- per-thread i-state
struct IState {
    // negated and duplicated so that d = j + (-i) is one packed add per component
    float2 nxh, nyh, nzh, nxl, nyl, nzl, nvx, nvy, nvz;
    float h2;        // r_s^2 in fp32, clamped to >= FLT_MIN so that the self pair (r^2 = 0) is always masked
    int32_t self;    // own j-index (never listed)
    int32_t nlim;    // list entries must have j < nlim: n for a normal row, 0 when r_s = 0 (reading R4/R5)
    int32_t cnt;     // neighbours found so far in this CTA's j-range
    int32_t* list;   // where this row's (partial) list goes
};

struct Accum {
    float2 ax, ay, az, jx, jy, jz;  // fp32 partial sums of the current j-tile; .x from j0, .y from j1
};

__device__ __forceinline__ void accum_zero(Accum& s) {
    s.ax = s.ay = s.az = s.jx = s.jy = s.jz = make_float2(0.f, 0.f);
}

// One packed step: the pair (j0, j1) held in q0..q4 against one i.  32 packed FP32 instructions
// (12 FADD2, 7 FMUL2, 13 FFMA2), 2 MUFU.RSQ, 2 FSETP, 2 FSEL.  Returns the two neighbour predicates.
__device__ __forceinline__ void pair_step(const float4& q0, const float4& q1, const float4& q2, const float4& q3,
                                          const float4& q4, const IState& I, Accum& s, bool& nb0, bool& nb1) {
    // double-single coordinate differences ("pseudo double precision for the coordinate differences")
    float2 dx = __fadd2_rn(__fadd2_rn(make_float2(q0.x, q0.y), I.nxh), __fadd2_rn(make_float2(q2.x, q2.y), I.nxl));
    float2 dy = __fadd2_rn(__fadd2_rn(make_float2(q0.z, q0.w), I.nyh), __fadd2_rn(make_float2(q2.z, q2.w), I.nyl));
    float2 dz = __fadd2_rn(__fadd2_rn(make_float2(q1.x, q1.y), I.nzh), __fadd2_rn(make_float2(q3.x, q3.y), I.nzl));
    float2 dvx = __fadd2_rn(make_float2(q3.z, q3.w), I.nvx);
    float2 dvy = __fadd2_rn(make_float2(q4.x, q4.y), I.nvy);
    float2 dvz = __fadd2_rn(make_float2(q4.z, q4.w), I.nvz);
    float2 r2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
    float2 rv = __ffma2_rn(dz, dvz, __ffma2_rn(dy, dvy, __fmul2_rn(dx, dvx)));
    nb0 = r2.x < I.h2;  // eq. (2)/(11): neighbour iff r^2 < r_s^2
    nb1 = r2.y < I.h2;
    float2 ri;
    ri.x = nb0 ? 0.f : rsqrt_approx(r2.x);  // Listing B2 line 31: "rinv1 = 0.f" masks the pair
    ri.y = nb1 ? 0.f : rsqrt_approx(r2.y);
    float2 ri2 = __fmul2_rn(ri, ri);
    float2 mri3 = __fmul2_rn(__fmul2_rn(make_float2(q1.z, q1.w), ri), ri2);
    float2 al = __fmul2_rn(__fmul2_rn(rv, ri2), make_float2(-3.f, -3.f));
    s.ax = __ffma2_rn(mri3, dx, s.ax);
    s.ay = __ffma2_rn(mri3, dy, s.ay);
    s.az = __ffma2_rn(mri3, dz, s.az);
    s.jx = __ffma2_rn(mri3, __ffma2_rn(al, dx, dvx), s.jx);
    s.jy = __ffma2_rn(mri3, __ffma2_rn(al, dy, dvy), s.jy);
    s.jz = __ffma2_rn(mri3, __ffma2_rn(al, dz, dvz), s.jz);
}

__device__ __forceinline__ void append(IState& I, int32_t j, bool nb, int32_t cap) {
    if (nb && j != I.self && j < I.nlim) {
        if (I.cnt < cap) I.list[I.cnt] = j;  // entries past cap are dropped, the count keeps counting (R7)
        ++I.cnt;
    }
}

template <int IPT, int WARPS, int JT, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) force_kernel(ForceArgs a) {
    constexpr int kThreads = WARPS * 32;
    constexpr int kRows = kThreads * IPT;
    constexpr int kTileQuads = JT / 2 * kQuadsPerPair;
    constexpr uint32_t kTileBytes = JT * kBytesPerJ;
    constexpr int kStages = 2;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* tiles = reinterpret_cast<float4*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + kStages * kTileBytes);

    const int tid = threadIdx.x;
    const int chunk = blockIdx.y;
    const int t_begin = chunk * a.tiles_per_chunk;
    const int t_end = min(t_begin + a.tiles_per_chunk, a.n_tiles);
    const int n_t = t_end - t_begin;

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0 && n_t > 0) {  // prologue: first tile in flight while the i-state is gathered
        mbar_arrive_expect_tx(&full[0], kTileBytes);
        bulk_g2s(tiles, a.packed + (size_t)t_begin * kTileQuads, kTileBytes, &full[0]);
    }

    // ---- S2: i-setup.  Gather the active particles' predicted state from the packed records by index.
    IState I[IPT];
    Accum s[IPT];
    double sum[IPT][6];
    int64_t rows[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int64_t row = (int64_t)blockIdx.x * kRows + u * kThreads + tid;
        rows[u] = row;
        const bool live = row < a.n_i;
        const int32_t i = live ? a.i_idx[row] : 0;
        const float* rec = reinterpret_cast<const float*>(a.packed + (size_t)(i >> 1) * kQuadsPerPair);
        const int h = i & 1;
        const float xh = rec[0 + h], yh = rec[2 + h], zh = rec[4 + h];
        const float xl = rec[8 + h], yl = rec[10 + h], zl = rec[12 + h];
        const float vx = rec[14 + h], vy = rec[16 + h], vz = rec[18 + h];
        I[u].nxh = make_float2(-xh, -xh); I[u].nyh = make_float2(-yh, -yh); I[u].nzh = make_float2(-zh, -zh);
        I[u].nxl = make_float2(-xl, -xl); I[u].nyl = make_float2(-yl, -yl); I[u].nzl = make_float2(-zl, -zl);
        I[u].nvx = make_float2(-vx, -vx); I[u].nvy = make_float2(-vy, -vy); I[u].nvz = make_float2(-vz, -vz);
        const double rs = live ? a.r_s[row] : 0.0;
        const float h2 = __double2float_rn(rs * rs);
        // dead rows (past n_i) get h2 < 0: nothing is ever a neighbour, nothing is written
        I[u].h2 = live ? fmaxf(h2, 1.17549435e-38f) : -1.f;
        I[u].self = i;
        I[u].nlim = (live && h2 >= 1.17549435e-38f) ? a.n : 0;
        I[u].cnt = 0;
        if (a.n_chunks == 1) {
            I[u].list = a.nbr_list + (size_t)row * a.cap;
        } else {
            I[u].list = a.part_list + ((size_t)row * a.n_chunks + chunk) * a.cap;
        }
        accum_zero(s[u]);
#pragma unroll
        for (int c = 0; c < 6; ++c) sum[u][c] = 0.0;
    }

    // ---- S3/S4: stream the j-tiles
    for (int lt = 0; lt < n_t; ++lt) {
        const int st = lt & 1;
        if (tid == 0 && lt + 1 < n_t) {  // prefetch the next tile into the other stage (freed by the barrier below)
            mbar_arrive_expect_tx(&full[st ^ 1], kTileBytes);
            bulk_g2s(tiles + (st ^ 1) * kTileQuads, a.packed + (size_t)(t_begin + lt + 1) * kTileQuads, kTileBytes,
                     &full[st ^ 1]);
        }
        mbar_wait(&full[st], (lt >> 1) & 1);
        const float4* tp = tiles + st * kTileQuads;
        const int32_t jbase = (t_begin + lt) * JT;
#pragma unroll 2
        for (int p = 0; p < JT / 2; ++p) {
            const float4 q0 = tp[p * 5 + 0], q1 = tp[p * 5 + 1], q2 = tp[p * 5 + 2], q3 = tp[p * 5 + 3],
                         q4 = tp[p * 5 + 4];
            bool nb0[IPT], nb1[IPT];
            bool any = false;
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                pair_step(q0, q1, q2, q3, q4, I[u], s[u], nb0[u], nb1[u]);
                any = any || nb0[u] || nb1[u];
            }
            if (__any_sync(0xffffffffu, any)) {  // S4: rare path, warp-uniform branch
                const int32_t j = jbase + 2 * p;
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    append(I[u], j, nb0[u], a.cap);
                    append(I[u], j + 1, nb1[u], a.cap);
                }
            }
        }
        // ---- S6: flush the tile's fp32 partial sums into the fp64 running sums
#pragma unroll
        for (int u = 0; u < IPT; ++u) {
            sum[u][0] += (double)s[u].ax.x + (double)s[u].ax.y;
            sum[u][1] += (double)s[u].ay.x + (double)s[u].ay.y;
            sum[u][2] += (double)s[u].az.x + (double)s[u].az.y;
            sum[u][3] += (double)s[u].jx.x + (double)s[u].jx.y;
            sum[u][4] += (double)s[u].jy.x + (double)s[u].jy.y;
            sum[u][5] += (double)s[u].jz.x + (double)s[u].jz.y;
            accum_zero(s[u]);
        }
        if (WARPS > 1) __syncthreads(); else __syncwarp();  // every warp is done with stage st before it is refilled
    }

    // ---- outputs
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int64_t row = rows[u];
        if (row >= a.n_i) continue;
        if (a.n_chunks == 1) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a.acc[row * 3 + c] = sum[u][c];
                a.jerk[row * 3 + c] = sum[u][3 + c];
            }
            a.nbr_count[row] = I[u].cnt;
            if (I[u].cnt > a.cap) atomicAdd(a.n_overflow, 1);
        } else {
            double* ps = a.part_sum + ((size_t)row * a.n_chunks + chunk) * 6;
#pragma unroll
            for (int c = 0; c < 6; ++c) ps[c] = sum[u][c];
            a.part_cnt[(size_t)row * a.n_chunks + chunk] = I[u].cnt;
        }
    }
}

}  // namespace nbreg
