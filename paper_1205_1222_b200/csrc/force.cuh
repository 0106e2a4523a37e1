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
//   * the j-range of the last ("tail") row blocks is split over several CTAs so that the
//     CTA count fills whole waves of the 148 SMs; those CTAs write per-(row, chunk) partial sums for
//     reduce_gather_kernel (gather.cuh) and share the row's list through an atomic slot counter.  Small active
//     blocks are all tail.
#pragma once
#include "nbreg_common.cuh"
#include "record.cuh"
#include "fixflag.cuh"

namespace nbreg {

// Far/near split: pairs farther than kappa X (X = largest |coordinate| of i) may skip the low words; kappa = 1/4.
// A smaller kappa makes the near path rarer (kappa = 1/8: +5 % throughput at N = 2^20) but doubles the far path's
// per-pair position error, and the worst jerk rows of config 5 then pass 1e-5 (measured).
#ifndef NBREG_KAPPA2
#define NBREG_KAPPA2 0.0625f
#endif
constexpr float kFarFraction2 = NBREG_KAPPA2;

// j-pairs per trip of the inner loop (unrolled), and the grain of a j-chunk's length that follows from it
#ifndef NBREG_JUNROLL
#define NBREG_JUNROLL 2
#endif
constexpr int kJUnroll = NBREG_JUNROLL;
constexpr int kChunkGrain = 2 * kJUnroll;

struct ForceArgs {
    RawState raw;           // PRED: the registered fp64 state and the time to predict to
    const float4* packed;   // packed j-pair records, n_pad / 2 pairs
    int32_t n;              // real j-particles
    int32_t n_pad;          // j-particles in the packed array (a multiple of kJPad; the padding is massless)
    // CTA b < main_blocks: row block b against the whole j-range, final outputs written directly.
    // CTA b >= main_blocks ("tail"): t = b - main_blocks, row block main_blocks + t / n_chunks against j-chunk
    // t % n_chunks = particles [chunk * chunk_j, (chunk + 1) * chunk_j), partial outputs for reduce_gather_kernel
    // (PAPER.md:122-126).  chunk_j is any multiple of 4 (not of the tile size): the planner cuts the j-range into
    // exactly as many equal chunks as fill whole waves of CTA slots; a chunk's last tile is shorter than the others.
    int32_t main_blocks;
    int32_t chunk_j;
    int32_t n_chunks;       // S >= 2 for the tail blocks (unused when there is no tail)
    int32_t n_i;
    int32_t cap;
    const int32_t* i_idx;
    const double* r_s;
    // Rows are processed in the order perm gives (Morton order of the predicted positions, order.cuh; null = as
    // given): thread "row" below is the LOGICAL row, perm[row] the caller's row all inputs and outputs refer to.
    const int32_t* perm;
    const double* dtr;       // VEL: regular time-step per row, eq. (3)
    const float* tile_vmax;  // VEL: speed bound per 256 consecutive j (predict.cuh)
    double* pot;             // POT: sum m_j / r over the summed pairs ("fo.pot += mrinv1")
    // final outputs (main blocks)
    double* acc;
    double* jerk;
    int32_t* nbr_count;
    int32_t* nbr_list;
    int32_t* n_overflow;    // not touched here: reduce_gather_kernel publishes it
    // zero-between-calls scratch in the workspace (reduce_gather_kernel leaves it zeroed again):
    int32_t* slot_count;    // [tail rows] list-slot counters of the j-split rows
    int32_t* overflow_ws;   // [1] rows with count > cap found so far in this call
    // partial sums of the tail blocks, indexed by tail row = row - main_blocks * rows_per_cta: [tail row][S][kSums + 1]
    // (the last slot holds the two error-scale sums as a float2).  Their list entries go straight to nbr_list through
    // the atomic slot counters slot_count.
    double* part_sum;
    FixupFlag fix;          // rows whose result is dominated by cancellation are queued for fixup_kernel (fixup.cuh)
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
__device__ __forceinline__ float rsqrt_approx(float x) {  // MUFU.RSQ; rsqrt(+inf) = 0
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {  // MUFU.RCP; rcp(+inf) = 0
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---------------------------------------------------------------- per-thread i-state
struct IState {
    // negated, so that d = j + (-i) is one packed add per component (the scalar is broadcast to both halves)
    float nxh, nyh, nzh, nxl, nyl, nzl, nvx, nvy, nvz;
    float h2;        // r_s^2 in fp32, clamped to >= FLT_MIN so that the self pair (r^2 = 0) is always masked
    float hfar2;     // pairs with |R_hi|^2 >= hfar2 take the far path (no low words, surely not a neighbour)
    // velocity criterion only: hfar2 is refreshed per j-tile as max(hfar_x, hfar_r + dtr vmax_tile)^2, so that a far
    // pair cannot come within r_s during dtr either: |R + dtr V| >= |R| - dtr (|v_i| + |v_j|)
    float hfar_x;    // kappa X
    float hfar_r;    // r_s (1 + 2^-11) + dtr |v_i|
    float dtr;
    int32_t self;    // own j-index (never listed)
    int32_t nlim;    // list entries must have j < nlim: n for a normal row, 0 when r_s = 0 (reading R4/R5)
    int32_t cnt;     // main path: neighbours found so far
    int32_t pend_j, pend_pos;  // j-split path: the append whose slot number is still in flight (pend_j < 0: none)
    int32_t* list;   // where this row's (partial) list goes
};

struct Accum {
    float2 ax, ay, az, jx, jy, jz;  // fp32 partial sums of the current j-tile; .x from j0, .y from j1
    float2 pot;                     // used by the POT variant only
};

__device__ __forceinline__ void accum_zero(Accum& s) {
    s.ax = s.ay = s.az = s.jx = s.jy = s.jz = s.pot = make_float2(0.f, 0.f);
}

__device__ __forceinline__ float2 bc(float a) { return make_float2(a, a); }

// The packed pair arithmetic, two j-particles (the halves of each float2) against one i.
//
// Far/near split (what keeps the common path at 25 packed FP32 instructions per two pairs):
//   * every pair first forms R from the HIGH words only, R_hi = xh_j - xh_i, and r_hi^2;
//   * if r_hi^2 >= hfar2 for both halves in every lane of the warp, the pair is FAR: it cannot be a neighbour
//     (hfar2 >= r_s^2 (1 + 2^-10)) and R_hi is used as R.  The omitted low words change r by at most
//     2^-24 (2 sqrt(3) X / r + 1) relative, X = max |x_i| component; hfar2 >= (X/4)^2 bounds that by 8.9e-7
//     (worst case);
//   * otherwise the warp takes the NEAR path: R = R_hi + (xl_j - xl_i) ("pseudo double precision for the
//     coordinate differences", footnote at PAPER.md:154), r^2 is recomputed, the neighbour test
//     eq. (2)/(11) is made on it, neighbours are appended to the list and masked by r^2 := +inf, so that
//     rsqrt and rcp return 0 ("rinv1 = 0.f", Listing B2) and the pair adds nothing.
struct PairGeom {
    float2 dx, dy, dz, r2;
};

__device__ __forceinline__ void geom_hi(const float4& q0, const float4& q1, const IState& I, PairGeom& g) {
    g.dx = __fadd2_rn(make_float2(q0.x, q0.y), bc(I.nxh));
    g.dy = __fadd2_rn(make_float2(q0.z, q0.w), bc(I.nyh));
    g.dz = __fadd2_rn(make_float2(q1.x, q1.y), bc(I.nzh));
    g.r2 = __ffma2_rn(g.dz, g.dz, __ffma2_rn(g.dy, g.dy, __fmul2_rn(g.dx, g.dx)));
}

__device__ __forceinline__ void geom_lo(const float2& xl, const float4& q4, const IState& I, PairGeom& g) {
    g.dx = __fadd2_rn(g.dx, __fadd2_rn(xl, bc(I.nxl)));
    g.dy = __fadd2_rn(g.dy, __fadd2_rn(make_float2(q4.x, q4.y), bc(I.nyl)));
    g.dz = __fadd2_rn(g.dz, __fadd2_rn(make_float2(q4.z, q4.w), bc(I.nzl)));
    g.r2 = __ffma2_rn(g.dz, g.dz, __ffma2_rn(g.dy, g.dy, __fmul2_rn(g.dx, g.dx)));
}

// eq. (9), (10) for the two pairs: 3 FADD2 (V), 3 (R.V), 2 (m/r^3), 2 (alpha), 9 FFMA2 (sums); 2 MUFU.RSQ + 2 MUFU.RCP.
// POT adds one packed add: pot += m ri (Listing B2: "fo.pot += mrinv1").
// REFINE (near path only): one Newton step on the MUFU results, rsqrt to ~0.5 ulp and rcp likewise.  The pairs of the
// near path are the closest ones a row sums, i.e. the largest jerk terms, whose rounding decides how close a row
// whose terms cancel can stay to the fp64 result; the common path pays nothing for it.
// The caller passes r^2 = +inf for a masked (neighbour) pair: rsqrt and rcp give 0 and the Newton residuals are
// formed so that no inf * 0 arises (the masked r^2 is replaced by 1 and the pair's mass by 0).
template <bool POT, bool REFINE>
__device__ __forceinline__ void pair_sum(const float4& q1, const float4& q2, const float2& vz, const IState& I,
                                         const PairGeom& g, Accum& s) {
    const float2 dvx = __fadd2_rn(make_float2(q2.x, q2.y), bc(I.nvx));
    const float2 dvy = __fadd2_rn(make_float2(q2.z, q2.w), bc(I.nvy));
    const float2 dvz = __fadd2_rn(vz, bc(I.nvz));
    const float2 rv = __ffma2_rn(g.dz, dvz, __ffma2_rn(g.dy, dvy, __fmul2_rn(g.dx, dvx)));
    float2 ri, ri2, mj = make_float2(q1.z, q1.w);
    if (REFINE) {
        const float inf = __int_as_float(0x7f800000);
        const float2 x = make_float2(g.r2.x == inf ? 1.f : g.r2.x, g.r2.y == inf ? 1.f : g.r2.y);
        mj = make_float2(g.r2.x == inf ? 0.f : mj.x, g.r2.y == inf ? 0.f : mj.y);
        const float2 y0 = make_float2(rsqrt_approx(x.x), rsqrt_approx(x.y));
        const float2 z0 = make_float2(rcp_approx(x.x), rcp_approx(x.y));
        const float2 ey = __ffma2_rn(__fmul2_rn(x, y0), make_float2(-y0.x, -y0.y), bc(1.f));  // 1 - x y0^2
        ri = __ffma2_rn(__fmul2_rn(y0, bc(0.5f)), ey, y0);                                      // y0 + y0 e / 2
        const float2 ez = __ffma2_rn(x, make_float2(-z0.x, -z0.y), bc(1.f));                    // 1 - x z0
        ri2 = __ffma2_rn(z0, ez, z0);                                                           // z0 + z0 e
    } else {
        ri = make_float2(rsqrt_approx(g.r2.x), rsqrt_approx(g.r2.y));
        ri2 = make_float2(rcp_approx(g.r2.x), rcp_approx(g.r2.y));
    }
    const float2 mri = __fmul2_rn(mj, ri);
    const float2 mri3 = __fmul2_rn(mri, ri2);
    if (POT) s.pot = __fadd2_rn(s.pot, mri);
    const float2 al = __fmul2_rn(__fmul2_rn(rv, ri2), bc(-3.f));
    s.ax = __ffma2_rn(mri3, g.dx, s.ax);
    s.ay = __ffma2_rn(mri3, g.dy, s.ay);
    s.az = __ffma2_rn(mri3, g.dz, s.az);
    s.jx = __ffma2_rn(mri3, __ffma2_rn(al, g.dx, dvx), s.jx);
    s.jy = __ffma2_rn(mri3, __ffma2_rn(al, g.dy, dvy), s.jy);
    s.jz = __ffma2_rn(mri3, __ffma2_rn(al, g.dz, dvz), s.jz);
}

// Velocity criterion eq. (3), near path only: r_min^2 = min(|R|^2, |R + dtr V|^2) with the full-precision R
// (Listing B2 lines 17-19, 22, 26).
__device__ __forceinline__ float2 rmin2_velocity(const float4& q2, const float2& vz, const IState& I, const PairGeom& g) {
    const float2 dvx = __fadd2_rn(make_float2(q2.x, q2.y), bc(I.nvx));
    const float2 dvy = __fadd2_rn(make_float2(q2.z, q2.w), bc(I.nvy));
    const float2 dvz = __fadd2_rn(vz, bc(I.nvz));
    const float2 px = __ffma2_rn(bc(I.dtr), dvx, g.dx);
    const float2 py = __ffma2_rn(bc(I.dtr), dvy, g.dy);
    const float2 pz = __ffma2_rn(bc(I.dtr), dvz, g.dz);
    const float2 r2p = __ffma2_rn(pz, pz, __ffma2_rn(py, py, __fmul2_rn(px, px)));
    return make_float2(fminf(g.r2.x, r2p.x), fminf(g.r2.y, r2p.y));
}

// S4: "the index j is written to the neighbour list in the memory".  A main-path row is owned by
// one thread for the whole j-range: private counter, entries land in ascending j.  A j-split row is shared by
// the CTAs of its chunks: a slot is reserved with an atomic on the row's final count (reduce_gather_kernel puts
// the row in order afterwards).  The atomic's return value takes an L2 round trip, so the store that needs it
// is DEFERRED to the thread's next append (or the end of the chunk): the warp never waits for it in the j-loop.
// Entries past cap are dropped, the count keeps counting (reading R7).
__device__ __forceinline__ void flush_pending(IState& I, int32_t cap) {
    if (I.pend_j >= 0 && I.pend_pos < cap) I.list[I.pend_pos] = I.pend_j;
    I.pend_j = -1;
}
__device__ __forceinline__ void append(IState& I, int32_t j, bool nb, int32_t cap, int32_t* shared_count) {
    if (nb && j != I.self && j < I.nlim) {
        if (shared_count) {
            flush_pending(I, cap);
            I.pend_pos = atomicAdd(shared_count, 1);
            I.pend_j = j;
        } else {
            if (I.cnt < cap) I.list[I.cnt] = j;
            ++I.cnt;
        }
    }
}

// PRED: the predictor fused into the kernel (north_star: "fused with the Hermite predictor of the j-particles").  Used
// for small active blocks (N_i <= 128: one to four row blocks), whose j-range is split over the CTAs so that every j is
// predicted by the CTA that uses it (once per row block): each thread predicts one pair of consecutive j per tile from the
// registered fp64 state (predict_record: the arithmetic of predict.cuh, the same records bit for bit) and writes its
// packed record straight into the shared-memory tile -- no prediction pass (25 us at N = 2^20), no packed records in
// HBM.  The CTAs resident on an SM hide each other's load latency; there is one tile stage and no bulk copy.
template <int IPT, int WARPS, int JT, int MINB, bool VEL, bool POT, bool PRED = false>
__global__ void __launch_bounds__(WARPS * 32, MINB) force_kernel(ForceArgs a) {
    static_assert(!PRED || (IPT == 1 && JT == 2 * WARPS * 32 && !VEL), "PRED: one j-pair per thread per tile");
    constexpr int kSums = POT ? 7 : 6;  // fp64 running sums per row: acc, jerk (, pot)
    constexpr int kThreads = WARPS * 32;
    constexpr int kRows = kThreads * IPT;
    constexpr int kTileQuads = JT / 2 * kQuadsPerPair;
    constexpr uint32_t kTileBytes = JT * kBytesPerJ;  // a full tile; a chunk's last tile may be shorter
    constexpr int kStages = PRED ? 1 : 2;  // the fused-prediction variant fills its one stage itself

    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* tiles = reinterpret_cast<float4*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + kStages * kTileBytes);
    // The fp64 running sums (S6) live in shared memory, [component][i-of-thread][thread]: they are touched once per
    // j-tile, and without their 12 registers per i the kernel fits 64 registers = 32 resident warps per SM
    // (measured: 1108 -> 1140 Gpairs/s at config 5).
    double* ssum = reinterpret_cast<double*>(smem_raw + kStages * kTileBytes + 2 * sizeof(uint64_t));
#define NB_SUM(u, c) ssum[((c) * IPT + (u)) * kThreads + tid]
    // Error scale of the row (fixup.cuh): the squared norms of the per-tile fp32 partial sums, added up over the
    // tiles -- sum_T |acc_T|^2 and sum_T |jerk_T|^2.  Touched once per tile, like the running sums.
    float2* sq = reinterpret_cast<float2*>(ssum + kSums * kRows);
#define NB_Q(u) sq[(u) * kThreads + tid]

    const int tid = threadIdx.x;
    const bool split = (int)blockIdx.x >= a.main_blocks;
    int row_block = blockIdx.x, chunk = 0;
    int32_t j_begin = 0, j_end = a.n_pad;
    if (split) {
        const int t = blockIdx.x - a.main_blocks;
        row_block = a.main_blocks + t / a.n_chunks;
        chunk = t % a.n_chunks;
        j_begin = chunk * a.chunk_j;
        j_end = min(j_begin + a.chunk_j, a.n_pad);
    }
    const int n_t = (j_end - j_begin + JT - 1) / JT;  // tiles of this CTA; the last one may be short (a multiple of 4 j)
    const int64_t tail_row0 = (int64_t)a.main_blocks * kRows;

    if (!PRED && tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    if (!PRED) __syncthreads();
    pdl_wait();     // the predictor (or the row ordering) has finished; before this line nothing touched global memory
    if (!PRED && tid == 0 && n_t > 0) {  // prologue: first tile in flight while the i-state is gathered
        const uint32_t bytes = (uint32_t)min(JT, j_end - j_begin) * kBytesPerJ;
        mbar_arrive_expect_tx(&full[0], bytes);
        bulk_g2s(tiles, a.packed + (size_t)(j_begin >> 1) * kQuadsPerPair, bytes, &full[0]);
    }

    // ---- S2: i-setup.  Gather the active particles' predicted state from the packed records by index.
    IState I[IPT];
    Accum s[IPT];
    int64_t rows[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int64_t row = (int64_t)row_block * kRows + u * kThreads + tid;
        rows[u] = row;
        const bool live = row < a.n_i;
        const int64_t orow = (live && a.perm) ? a.perm[row] : row;  // the caller's row
        const int32_t i = live ? a.i_idx[orow] : 0;
        float xh, yh, zh, vx, vy, vz, xl, yl, zl;
        if (PRED) {
            const PredRecord ri = predict_record(a.raw, i);
            xh = ri.xh; yh = ri.yh; zh = ri.zh; vx = ri.vx; vy = ri.vy; vz = ri.vz; xl = ri.xl; yl = ri.yl; zl = ri.zl;
        } else {
            const float* rec = reinterpret_cast<const float*>(a.packed + (size_t)(i >> 1) * kQuadsPerPair);
            const int h = i & 1;
            xh = rec[0 + h]; yh = rec[2 + h]; zh = rec[4 + h];
            vx = rec[8 + h]; vy = rec[10 + h]; vz = rec[12 + h];
            xl = rec[14 + h]; yl = rec[16 + h]; zl = rec[18 + h];
        }
        I[u].nxh = -xh; I[u].nyh = -yh; I[u].nzh = -zh;
        I[u].nxl = -xl; I[u].nyl = -yl; I[u].nzl = -zl;
        I[u].nvx = -vx; I[u].nvy = -vy; I[u].nvz = -vz;
        const double rs = live ? a.r_s[orow] : 0.0;
        const float h2 = __double2float_rn(rs * rs);
        // dead rows (past n_i) get h2 < 0: nothing is ever a neighbour, nothing is written
        I[u].h2 = live ? fmaxf(h2, 1.17549435e-38f) : -1.f;
        // far threshold: beyond r_s with a 2^-10 margin, and beyond X/4 (X = largest |coordinate| of i), see above
        const float xmax = fmaxf(fabsf(xh), fmaxf(fabsf(yh), fabsf(zh)));
        I[u].hfar2 = live ? fmaxf(I[u].h2 * 1.0009765625f, kFarFraction2 * xmax * xmax) : -1.f;
        if (VEL) {
            const float dtr = live ? fabsf(__double2float_rn(a.dtr[orow])) : 0.f;
            const float vi = sqrtf(vx * vx + vy * vy + vz * vz) * 1.000001f;
            I[u].dtr = live ? __double2float_rn(a.dtr[orow]) : 0.f;
            I[u].hfar_x = live ? sqrtf(kFarFraction2) * xmax : 0.f;  // dead rows: hfar2 = 0, never near
            I[u].hfar_r = live ? fmaf(dtr, vi, sqrtf(I[u].h2) * 1.00048828125f) : 0.f;
        }
        I[u].self = i;
        I[u].nlim = (live && h2 >= 1.17549435e-38f) ? a.n : 0;
        I[u].cnt = 0;
        I[u].pend_j = -1;
        I[u].pend_pos = 0;
        I[u].list = a.nbr_list + (size_t)orow * a.cap;
        accum_zero(s[u]);
#pragma unroll
        for (int c = 0; c < kSums; ++c) NB_SUM(u, c) = 0.0;
        NB_Q(u) = make_float2(0.f, 0.f);
    }

    // ---- S3/S4: stream the j-tiles
    for (int lt = 0; lt < n_t; ++lt) {
        const int st = PRED ? 0 : (lt & 1);
        const int32_t jbase = j_begin + lt * JT;             // first particle of this tile
        const int32_t tile_j = min(JT, j_end - jbase);       // particles in it
        if (PRED) {  // predict this thread's j-pair of the tile into shared memory (layout of nbreg_common.cuh)
            const int32_t j0 = jbase + 2 * tid;
            PredRecord r0, r1;
            r0.xh = r0.yh = r0.zh = kFarAway; r0.m = r0.xl = r0.yl = r0.zl = r0.vx = r0.vy = r0.vz = 0.f;
            r1 = r0;  // padding particles past n: massless, far away, at rest
            if (2 * tid < tile_j) {  // (a short last tile: the other threads have nothing to predict)
                if (j0 < a.n) r0 = predict_record(a.raw, j0);
                if (j0 + 1 < a.n) r1 = predict_record(a.raw, j0 + 1);
            }
            float4* o = tiles + tid * kQuadsPerPair;
            o[0] = make_float4(r0.xh, r1.xh, r0.yh, r1.yh);
            o[1] = make_float4(r0.zh, r1.zh, r0.m, r1.m);
            o[2] = make_float4(r0.vx, r1.vx, r0.vy, r1.vy);
            o[3] = make_float4(r0.vz, r1.vz, r0.xl, r1.xl);
            o[4] = make_float4(r0.yl, r1.yl, r0.zl, r1.zl);
            if (WARPS > 1) __syncthreads(); else __syncwarp();
        }
        if (!PRED && tid == 0 && lt + 1 < n_t) {  // prefetch the next tile into the other stage (freed by the barrier below)
            const uint32_t bytes = (uint32_t)min(JT, j_end - jbase - JT) * kBytesPerJ;
            mbar_arrive_expect_tx(&full[st ^ 1], bytes);
            bulk_g2s(tiles + (st ^ 1) * kTileQuads, a.packed + (size_t)((jbase + JT) >> 1) * kQuadsPerPair, bytes,
                     &full[st ^ 1]);
        }
        if (!PRED) mbar_wait(&full[st], (lt >> 1) & 1);
        const float4* tp = tiles + st * kTileQuads;
        if (VEL) {  // far threshold of this tile: its fastest particle cannot bring a far pair within r_s during dtr
            // (speed bounds are kept per 256 consecutive particles; a tile overlaps at most two such blocks)
            const float vmax = fmaxf(__ldg(a.tile_vmax + (jbase >> 8)), __ldg(a.tile_vmax + ((jbase + tile_j - 1) >> 8)));
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                const float hf = fmaxf(I[u].hfar_x, fmaf(fabsf(I[u].dtr), vmax, I[u].hfar_r));
                I[u].hfar2 = hf * hf;
            }
        }
        const int n_pp = tile_j / (2 * kJUnroll);  // the tile's j-pairs, kJUnroll per trip (tile_j is a multiple of kChunkGrain)
#pragma unroll 1
        for (int pp = 0; pp < n_pp; ++pp) {
#pragma unroll
        for (int ph = 0; ph < kJUnroll; ++ph) {
            const int p = kJUnroll * pp + ph;
            const float4 q0 = tp[p * 5 + 0], q1 = tp[p * 5 + 1], q2 = tp[p * 5 + 2];
            const float2 vz = *reinterpret_cast<const float2*>(tp + p * 5 + 3);
            PairGeom g[IPT];
            bool near = false;
#pragma unroll
            for (int u = 0; u < IPT; ++u) {
                geom_hi(q0, q1, I[u], g[u]);
                near = near || fminf(g[u].r2.x, g[u].r2.y) < I[u].hfar2;
            }
            if (__any_sync(0xffffffffu, near)) {  // NEAR path (S4 lives here): rare, warp-uniform branch
                const float2 xl = *(reinterpret_cast<const float2*>(tp + p * 5 + 3) + 1);
                const float4 q4 = tp[p * 5 + 4];
                const int32_t j = jbase + 2 * p;
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    geom_lo(xl, q4, I[u], g[u]);
                    // eq. (2)/(11): neighbour iff r^2 < r_s^2; eq. (3): iff min(r^2, |R + dtr V|^2) < r_s^2
                    const float2 rm = VEL ? rmin2_velocity(q2, vz, I[u], g[u]) : g[u].r2;
                    const bool nb0 = rm.x < I[u].h2;
                    const bool nb1 = rm.y < I[u].h2;
                    int32_t* shared_count = split ? a.slot_count + (rows[u] - tail_row0) : nullptr;
                    append(I[u], j, nb0, a.cap, shared_count);
                    append(I[u], j + 1, nb1, a.cap, shared_count);
                    if (nb0) g[u].r2.x = __int_as_float(0x7f800000);
                    if (nb1) g[u].r2.y = __int_as_float(0x7f800000);
                    pair_sum<POT, true>(q1, q2, vz, I[u], g[u], s[u]);
                }
                continue;  // the near path finishes the pair itself: nothing flows back into the common path
            }
#pragma unroll
            for (int u = 0; u < IPT; ++u) pair_sum<POT, false>(q1, q2, vz, I[u], g[u], s[u]);
        }
        }
        // ---- S6: flush the tile's fp32 partial sums into the fp64 running sums
#pragma unroll
        for (int u = 0; u < IPT; ++u) {
            // Error scale: a tile's partial sums are sums of ~JT terms of mixed direction, so their squared norms add up
            // (over the tiles) to an estimate of sum_j |term_j|^2, the variance scale of the row's fp32 rounding error
            // (fixflag.cuh).  Component by component, so that no more registers are live than without it.
#define NB_FLUSH(c, f, qq)                                    \
    {                                                         \
        const float t = (f).x + (f).y;                        \
        NB_SUM(u, c) += (double)(f).x + (double)(f).y;        \
        (f) = make_float2(0.f, 0.f);                          \
        qq = fmaf(t, t, qq);                                  \
    }
            // (shared-memory reductions instead of a read-modify-write through registers: the kernel keeps its 64
            // registers = 32 resident warps per SM; with q in registers across the flush ptxas needs 68)
            float qq = 0.f;
            NB_FLUSH(0, s[u].ax, qq)
            NB_FLUSH(1, s[u].ay, qq)
            NB_FLUSH(2, s[u].az, qq)
            atomicAdd(&NB_Q(u).x, qq);
            qq = 0.f;
            NB_FLUSH(3, s[u].jx, qq)
            NB_FLUSH(4, s[u].jy, qq)
            NB_FLUSH(5, s[u].jz, qq)
            atomicAdd(&NB_Q(u).y, qq);
#undef NB_FLUSH
            if (POT) {
                NB_SUM(u, kSums - 1) += (double)s[u].pot.x + (double)s[u].pot.y;
                s[u].pot = make_float2(0.f, 0.f);
            }
        }
        if (WARPS > 1) __syncthreads(); else __syncwarp();  // every warp is done with stage st before it is refilled
    }

    pdl_trigger();  // the gather kernel may be scheduled once every CTA of this launch is through its j-loop

    // ---- outputs
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int64_t row = rows[u];
        const int64_t orow = (row < a.n_i && a.perm) ? a.perm[row] : row;
        if (row >= a.n_i) continue;
        if (!split) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a.acc[orow * 3 + c] = NB_SUM(u, c);
                a.jerk[orow * 3 + c] = NB_SUM(u, 3 + c);
            }
            if (POT) a.pot[orow] = NB_SUM(u, kSums - 1);
            a.nbr_count[orow] = I[u].cnt;
            if (I[u].cnt > a.cap) atomicAdd(a.overflow_ws, 1);
            const float2 q = NB_Q(u);
            fixup_flag(a.fix, (int32_t)orow, q.x, q.y, NB_SUM(u, 0), NB_SUM(u, 1), NB_SUM(u, 2), NB_SUM(u, 3),
                       NB_SUM(u, 4), NB_SUM(u, 5));
        } else {
            flush_pending(I[u], a.cap);
            const size_t pi = (size_t)(row - tail_row0) * a.n_chunks + chunk;
            double* ps = a.part_sum + pi * (kSums + 1);
#pragma unroll
            for (int c = 0; c < kSums; ++c) ps[c] = NB_SUM(u, c);
            *reinterpret_cast<float2*>(ps + kSums) = NB_Q(u);
        }
    }
}

#undef NB_SUM
#undef NB_Q

}  // namespace nbreg
