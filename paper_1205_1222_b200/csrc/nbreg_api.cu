// nbreg_api.cu -- the C ABI of include/nbreg.h: context, argument checks, launch planning, launches.
// Every step of the path runs in the kernels of predict.cuh / force.cuh / gather.cuh; nothing here computes.
#include "../../include/nbreg.h"

#include <cstdio>
#include <algorithm>
#include <cmath>
#include <cstring>
#include <utility>

#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <thrust/iterator/counting_iterator.h>
#include <thrust/iterator/transform_iterator.h>
#include <new>

#include "force.cuh"
#include "fixup.cuh"
#include "gather.cuh"
#include "irregular.cuh"
#include "corrector.cuh"
#include "order.cuh"
#include "nbreg_common.cuh"
#include "predict.cuh"

using namespace nbreg;

// Resident 256-thread CTAs per SM the 256-row force kernel is compiled for (register cap 65536 / (256 *
// NBREG_CTAS256)).
#ifndef NBREG_CTAS256
#define NBREG_CTAS256 3
#endif
// Resident warps per SM the smaller shapes (128, 64, 32 rows per CTA) are compiled for: 28 = 65536 / (72 * 32), a
// granularity the 256-thread shape cannot reach (3 CTAs = 24 warps, 4 would need <= 64 registers).  Measured on
// B200: 28 warps are 1-3 % faster than 24-26 (config 5: 1064 against 1054 Gpairs/s).
#ifndef NBREG_WARPS_SMALL
#define NBREG_WARPS_SMALL 28
#endif
// ... and the fused-prediction variants of those shapes (PRED, force.cuh).  Measured at N = 2^20, N_i = 32 / 64 / 128, us per
// call: 28 warps (72 registers, 44 B spilled) 73.6 / 105.2 / 189.1; 24 warps (80 registers) 72.1 / 101.2 / 179.2; 20 warps (96
// registers, no spills) 70.4 / 105.0 / 184.8.
#ifndef NBREG_WARPS_PRED
#define NBREG_WARPS_PRED 24
#endif

namespace {

thread_local char g_errbuf[256] = "";

// Launch with the programmatic-stream-serialization attribute (nbreg_common.cuh: pdl_wait / pdl_trigger): the kernel may
// be scheduled while the tail of the kernel before it is still running; it waits for that kernel's completion itself.
bool g_pdl = true;  // "pdl" option of any context switches it for the process (a debugging aid)
template <typename... KArgs, typename... Args>
cudaError_t launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = g_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error in %s: %s", what, cudaGetErrorString(e));
    return NB_E_CUDA;
}
#define NB_CUDA(call)                                   \
    do {                                                \
        cudaError_t e_ = (call);                        \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
    } while (0)

// CTA shapes of the force kernel: rows per CTA, i per thread, warps, particles per shared-memory j-tile.  The 256-row
// shape holds NBREG_CTAS256 CTAs (24 warps) per SM, the smaller ones NBREG_WARPS_SMALL warps; the 512-row shape (two
// i per thread) is only used when asked for ("i_block" option).
constexpr int kNumShapes = 5;
struct Shape {
    int rows, ipt, warps, jt;
};
constexpr Shape kShapes[kNumShapes] = {{256, 1, 8, 256}, {128, 1, 4, 256}, {64, 1, 2, 128}, {32, 1, 1, 64},
                                       {512, 2, 8, 256}};

// Launch plan of the force kernel: CTA shape, how many row blocks run the whole j-range in one CTA ("main"),
// and the j-split of the remaining ("tail") row blocks.
struct Plan {
    int shape;          // index into kShapes
    int n_pad;          // j-particles of the packed array (n rounded up to kJPad)
    int n_blocks;       // row blocks
    int main_blocks;    // row blocks handled by one CTA each
    int n_chunks;       // S: j-chunks per tail row block (1 = no tail: main_blocks == n_blocks)
    int chunk_j;        // particles per chunk: a multiple of kChunkGrain, not of the tile size
    int grid;           // CTAs
    double cost;        // model cost in units of (one j against one CTA's rows)
};

struct WorkspaceLayout {
    size_t packed_off, packed_bytes;
    size_t psum_off, psum_bytes;
    size_t gather_off, gather_bytes;  // particle-major predicted records, 48 B per j
    size_t vmax_off, vmax_bytes;   // float speed bound per 256 consecutive j (predictor -> velocity criterion)
    size_t sort_off, sort_bytes;   // row ordering: keys and rows, two buffers each, + the library sort's scratch
    size_t sort_temp_bytes;
    size_t fixrow_off, fixrow_bytes;  // int32 caller's rows queued for the fp64 fix-up pass (fixup.cuh)
    size_t escale_off, escale_bytes;  // float2 error scales per caller's row (fixflag.cuh)
    size_t ovfrow_off, ovfrow_bytes;  // int32 caller's rows queued for overflow_list_kernel (option "ovf_first_in_j")
    size_t slot_off, slot_bytes;   // int32 list-slot counters of the j-split rows (zero between calls)
    size_t ftick_off, ftick_bytes; // int32 chunk tickets of the fix-up groups (zero between calls)
    // int32 {overflow count, gather ticket, order ticket, -, 6 box words, -, -, -, -, -, -, fix-up queue length, fix-up
    // CTA ticket} (zero between calls), then {rows of the last fix-up, -, rows since nb_create (64 bit)}
    size_t ctl_off, ctl_bytes;
    int64_t row_chunk_limit;  // (row, j-chunk) slots of partial sums
    size_t total;
};

// The j-split workspace holds 7 doubles per (row, chunk): enough slots for 256 chunks per row of the largest
// block, at least 131072 (small blocks are split hundreds of ways), at most 2M (112 MB).
int64_t row_chunk_slots(int64_t n_i_max) {
    return std::min<int64_t>(std::max<int64_t>(256 * n_i_max, 131072), 2097152);
}

WorkspaceLayout layout(int64_t n_max, int64_t n_i_max, int32_t cap) {
    WorkspaceLayout w{};
    (void)cap;
    const int64_t n_pad = round_up(n_max, kJPad);
    w.row_chunk_limit = row_chunk_slots(n_i_max);
    size_t off = 0;
    auto place = [&](size_t bytes, size_t& o, size_t& b) {
        o = off;
        b = bytes;
        off += (size_t)round_up((int64_t)bytes, 256);
    };
    place((size_t)n_pad * kBytesPerJ, w.packed_off, w.packed_bytes);
    // acc, jerk, pot, error scales per (row, chunk); the fix-up pass, which runs after the gather, keeps the partial sums
    // of its (group, chunk) items in the same region: fewer than grid + groups items of kFixWarps x 6 doubles
    place(std::max((size_t)w.row_chunk_limit * 8 * sizeof(double),
                   ((size_t)kFixMaxGrid * kFixWarps + (size_t)n_i_max + kFixWarps) * 6 * sizeof(double)),
          w.psum_off, w.psum_bytes);
    place((size_t)n_pad * kGatherQuads * sizeof(float4), w.gather_off, w.gather_bytes);
    place((size_t)(n_pad / kJPad) * sizeof(float), w.vmax_off, w.vmax_bytes);
    {
        const int64_t ni = std::max<int64_t>(n_i_max, 1);
        size_t temp = 0;
        cub::DoubleBuffer<uint32_t> dk(nullptr, nullptr);
        cub::DoubleBuffer<int32_t> dv(nullptr, nullptr);
        cub::DeviceRadixSort::SortPairs(nullptr, temp, dk, dv, (int)ni, 0, kKeyBits);
        w.sort_temp_bytes = (size_t)round_up((int64_t)temp, 256) + 256;
        place(4 * (size_t)round_up(ni * 4, 256) + w.sort_temp_bytes, w.sort_off, w.sort_bytes);
    }
    place((size_t)(n_i_max + 1) * sizeof(int32_t), w.fixrow_off, w.fixrow_bytes);
    place((size_t)(n_i_max + 1) * sizeof(float2), w.escale_off, w.escale_bytes);
    place((size_t)(n_i_max + 1) * sizeof(int32_t), w.ovfrow_off, w.ovfrow_bytes);
    place((size_t)(n_i_max + 512) * sizeof(int32_t), w.slot_off, w.slot_bytes);
    place((size_t)(n_i_max / kFixWarps + 34) * sizeof(int32_t), w.ftick_off, w.ftick_bytes);
    place(128, w.ctl_off, w.ctl_bytes);
    w.total = off;
    return w;
}

}  // namespace

// Default thresholds of the fp64 fix-up (calibrated against the fp64 oracle on every row of
// configs 3 and 5): a row's fp32 error is ~ eps sqrt(q) with eps up to ~1e-6 in the far tail, so C = S eps / tolerance.
constexpr int64_t kFixCaMilli = 2000;  // C_a = 2.0
constexpr int64_t kFixCjMilli = 200;   // C_j = 0.2

// nb_regular_force_host splits large active blocks into up to kHostChunks row chunks so that the device-to-host copy
// of one chunk's outputs (the list array dominates) runs while the next chunk is computed
constexpr int kHostChunks = 8;
constexpr int64_t kHostChunkMinRows = 16384;

struct nb_ctx {
    int device = 0;
    int num_sms = 0;
    int ctas_per_sm[4][kNumShapes] = {};  // resident CTAs per SM of each force-kernel variant and shape
    int ctas_per_sm_pred[kNumShapes] = {}; // ... of the fused-prediction variant (shapes 1-3; others 0)
    int64_t n_max = 0, n_i_max = 0;
    int32_t cap = 0;
    unsigned char* ws = nullptr;
    bool ws_owned = false;
    WorkspaceLayout lay{};
    // registered j-state (device pointers owned by the caller)
    int64_t n = 0;
    const double *x0 = nullptr, *v0 = nullptr, *a0 = nullptr, *j0 = nullptr, *m = nullptr, *t0 = nullptr;
    bool predicted = false;
    double t_pred = 0.0;
    // the particle-major copy of the predicted records (gathers of single particles: irregular force, corrector) is
    // written by a prediction pass only once a call has asked for it (or option "gather_copy" = 1)
    bool gather_wanted = false, gather_valid = false;
    int64_t opt_gather_copy = 0;
    // options
    int64_t opt_j_split = 0, opt_i_block = 0, opt_order_rows = 1, opt_irr_pred = 0, opt_fuse_pred = 1;
    // fp64 fix-up of cancellation-dominated rows (fixflag.cuh): a row is recomputed iff C_a sqrt(q_a) > |acc| or
    // C_j sqrt(q_j) > |jerk|; the options hold 1000 C_a and 1000 C_j
    int64_t opt_fixup = 1, opt_fix_ca_milli = kFixCaMilli, opt_fix_cj_milli = kFixCjMilli;
    int64_t opt_ovf_first = 0;  // overflowed j-split rows keep the first nbr_cap neighbours in j (overflow_list_kernel)
    // last launch
    int64_t info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    // host path: device mirrors owned by the context
    cudaStream_t hstream = nullptr, hcopy = nullptr;  // compute and device-to-host copy streams
    cudaEvent_t hdone[kHostChunks] = {};              // "rows of chunk k are final"
    int32_t* hovf = nullptr;                          // pinned: overflow count, then longest list, of each chunk
    unsigned char* hbuf = nullptr;
    size_t hbuf_bytes = 0;
    unsigned char* hcsr = nullptr;                    // CSR host path: packed lists, row offsets, scan scratch
};

namespace {

// Cost model behind the plan, in units of "one j against the rows of one CTA".  All
// resident warps share an SM evenly, so a CTA needs a time proportional to the j it covers, plus a prologue worth
// ~kPrologueJ j, whatever its shape.  Row blocks that fill whole waves of CTA slots run the full j-range in one
// CTA and write their outputs directly.  The remaining ("tail") blocks -- all blocks of a small active block --
// are split S ways along j.  Measured on B200 (profiles/, planner calibration): G equal CTAs
// of duration t on `slots` slots take about w t + 0.2 t, w between G / slots and its ceiling; the last term is the
// ragged end, which is why several waves of short CTAs beat one wave of long ones.
// rows split into more than kWideGatherChunks chunks are gathered by a block each, if there are few enough of them
// that a warp per row would leave SMs idle
// Largest block that predicts inside the force kernel.  Round 2, after the predictor pass got its bandwidth back (38 ->
// 25 us at N = 2^20), pass -> fused per call with a fresh prediction, replayed from a CUDA graph: N = 2^20: 32 rows 82 -> 68 us,
// 64 rows 117 -> 106, 128 rows 190 -> 184, 256 rows 338 -> 346; N = 524288: 47 -> 43, 64 -> 61, 101 -> 101, 176 -> 182;
// N = 262144: 33 -> 31, 42 -> 39, 60 -> 59, 98 -> 100.
constexpr int kFusePredMaxRows = 128;
constexpr int64_t kFusePredMinN = 262144;  // smallest n for which a one-row-block call predicts inside the force kernel
constexpr int kOrderMinRows = 256;  // smaller active blocks are processed in the order given
constexpr int kWideGatherChunks = 64;
constexpr int64_t kWideGatherRows = 4096;
constexpr double kPrologueJ = 48.0;
constexpr double kRaggedEnd = 0.2;
constexpr int64_t kMinChunkJ = 64;   // shortest chunk worth a CTA

struct Machine {
    int64_t n;        // j-particles
    int64_t row_chunk_limit;
    int num_sms;
    int ctas_per_sm[kNumShapes];
};

Plan plan_for_shape(const Machine* c, int32_t n_i, int shape, int64_t force_split) {
    const Shape& sh = kShapes[shape];
    Plan p{};
    p.shape = shape;
    const int64_t n_pad = round_up(c->n, kJPad);
    p.n_pad = (int)n_pad;
    p.n_blocks = (int)((n_i + sh.rows - 1) / sh.rows);
    const int64_t sms = c->num_sms > 0 ? c->num_sms : 148;
    const int64_t slots = sms * (c->ctas_per_sm[shape] > 0 ? c->ctas_per_sm[shape] : 1);
    const double t_full = kPrologueJ + (double)n_pad;
    // S chunks of equal length (a multiple of kChunkGrain particles, whatever the tile size: a chunk's last tile is
    // simply shorter), none empty
    auto chunking = [&](int64_t S) {
        const int64_t cj = std::max<int64_t>(kMinChunkJ, round_up((n_pad + S - 1) / S, kChunkGrain));
        return std::pair<int, int>((int)cj, (int)((n_pad + cj - 1) / cj));
    };
    auto tail_cost = [&](int64_t tail, const std::pair<int, int>& ch) {
        const double t = kPrologueJ + (double)ch.first;
        const double waves = (double)(tail * ch.second) / (double)slots;
        // few waves run almost in lockstep (the count rounds up), many waves overlap freely
        const double eff_waves = std::max(1.0, 0.5 * std::ceil(waves) + 0.5 * waves);
        // (The gather kernel's cost grows with the (row, chunk) partial sums, ~4e-4 j per partial sum: an exhaustive
        // timing of every shape and split for 512 ... 8192 rows found no plan more than 1.5 % better than this model's.)
        return eff_waves * t + kRaggedEnd * t;
    };
    int64_t tail = p.n_blocks, S = 1;
    if (force_split > 0) {
        S = force_split;
    } else {
        tail = p.n_blocks % slots;
        if (tail > 0) {
            int64_t s_max = std::min<int64_t>(n_pad / kMinChunkJ, c->row_chunk_limit / (tail * sh.rows));
            s_max = std::max<int64_t>(1, std::min<int64_t>(s_max, kMaxChunks));
            double best = 1e300;
            int last_chunks = 0;
            for (int64_t s = 1; s <= s_max; ++s) {
                const auto ch = chunking(s);
                if (ch.second == last_chunks) continue;  // same chunking as a smaller s
                last_chunks = ch.second;
                // an unsplit tail (s = 1) is one more full-length wave
                const double cost = (ch.second == 1) ? t_full : tail_cost(tail, ch);
                if (cost < best) {
                    best = cost;
                    S = s;
                }
            }
        }
    }
    if (S > n_pad / kMinChunkJ) S = std::max<int64_t>(1, n_pad / kMinChunkJ);
    if (S > kMaxChunks) S = kMaxChunks;
    if (S > 1 && tail * sh.rows * S > c->row_chunk_limit) S = std::max<int64_t>(1, c->row_chunk_limit / (tail * sh.rows));
    const auto ch = chunking(S);
    p.chunk_j = ch.first;
    p.n_chunks = ch.second;
    if (p.n_chunks <= 1) {
        p.n_chunks = 1;
        p.chunk_j = (int)n_pad;
        tail = 0;
    }
    p.main_blocks = (int)(p.n_blocks - tail);
    p.grid = (int)(p.main_blocks + tail * p.n_chunks);
    const double main_waves = (double)((p.main_blocks + slots - 1) / slots);
    p.cost = main_waves * t_full + (tail ? tail_cost(tail, ch) : 0.0);
    return p;
}

Plan make_plan(const Machine* c, int32_t n_i, int64_t opt_i_block, int64_t opt_j_split) {
    if (opt_i_block) {
        int shape = 0;
        for (int k = 0; k < kNumShapes; ++k)
            if (kShapes[k].rows == opt_i_block) shape = k;
        return plan_for_shape(c, n_i, shape, opt_j_split);
    }
    // measured preferences: the 128-row shape holds 28 warps per SM against 24 of the 256-row shape (1-3 % faster);
    // still smaller CTAs pay a little more for staging the j-tiles (fewer warps share one bulk copy)
    const double penalty[4] = {1.02, 1.0, 1.02, 1.04};
    Plan best{};
    double best_cost = 1e300;
    // A CTA shape at least twice as tall as the whole active block would run with half or more of its warps on rows
    // that do not exist (they compute like any other warp and write nothing): such shapes are left out (N_i = 32 at
    // N = 2^20: 83 -> measured below with the 32-row shape instead of the 64-row one, same chunking).
    const int64_t rows_needed = round_up(std::max<int32_t>(n_i, 1), 32);
    for (int k = 0; k < 4; ++k) {
        if (kShapes[k].rows >= 2 * rows_needed && kShapes[k].rows > 32) continue;
        const Plan p = plan_for_shape(c, n_i, k, opt_j_split);
        if (p.cost * penalty[k] < best_cost) {
            best_cost = p.cost * penalty[k];
            best = p;
        }
    }
    return best;
}

// j-tile stages (two; one for the fused-prediction variant, PRED) + two mbarriers + the fp64 running sums (6 per row, 7
// with the potential).
// Per row also one float2 of error scales (fixflag.cuh).
size_t force_smem_bytes(int ipt, int warps, int jt, bool pot, int stages = 2) {
    return (size_t)stages * jt * kBytesPerJ + 2 * sizeof(uint64_t) +
           (size_t)ipt * warps * 32 * ((pot ? 7 : 6) * sizeof(double) + sizeof(float2));
}

template <int IPT, int WARPS, int JT, int MINB, bool VEL, bool POT>
int query_force(int* per_sm) {
    auto kern = force_kernel<IPT, WARPS, JT, MINB, VEL, POT>;
    const size_t smem = force_smem_bytes(IPT, WARPS, JT, POT);
    NB_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    NB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, WARPS * 32, smem));
    return NB_OK;
}

template <int IPT, int WARPS, int JT, int MINB, bool VEL, bool POT>
int launch_force(const Plan& p, const ForceArgs& fa, cudaStream_t st) {
    const size_t smem = force_smem_bytes(IPT, WARPS, JT, POT);
    NB_CUDA(launch_k(force_kernel<IPT, WARPS, JT, MINB, VEL, POT>, p.grid, WARPS * 32, smem, st, fa));
    return NB_OK;
}

// The fused-prediction variant (force.cuh, PRED): plain criterion, no potential, shapes of 128 / 64 / 32 rows, one tile
// stage.  per_sm != null: query the resident CTAs per SM instead of launching (the planner's slot count).
int force_pred_dispatch(int shape, int* per_sm, const Plan* p, const ForceArgs* fa, cudaStream_t st) {
#define NB_PRED(WARPS, JT, MINB)                                                                           \
    {                                                                                                      \
        auto kern = force_kernel<1, WARPS, JT, MINB, false, false, true>;                                  \
        const size_t smem = force_smem_bytes(1, WARPS, JT, false, 1); /* <= 17 KB: no opt-in needed */     \
        if (per_sm) {                                                                                      \
            NB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, WARPS * 32, smem));        \
            return NB_OK;                                                                                  \
        }                                                                                                  \
        NB_CUDA(launch_k(kern, p->grid, WARPS * 32, smem, st, *fa));                                       \
        return NB_OK;                                                                                      \
    }
    switch (shape) {
        case 1: NB_PRED(4, 256, NBREG_WARPS_PRED / 4)
        case 2: NB_PRED(2, 128, NBREG_WARPS_PRED / 2)
        case 3: NB_PRED(1, 64, NBREG_WARPS_PRED)
        default: return NB_E_INVAL;
    }
#undef NB_PRED
}

// one switch for both: keeps the template arguments of query and launch in one place.  variant: bit 0 = velocity
// criterion eq. (3), bit 1 = potential output (the kernel variants of Listing B2)
template <bool VEL, bool POT>
int force_dispatch_v(int shape, int* per_sm, const Plan* p, const ForceArgs* fa, cudaStream_t st) {
#define NB_SHAPE(IPT, WARPS, JT, MINB)                               \
    (per_sm ? query_force<IPT, WARPS, JT, MINB, VEL, POT>(per_sm) \
            : launch_force<IPT, WARPS, JT, MINB, VEL, POT>(*p, *fa, st))
    switch (shape) {
        case 0: return NB_SHAPE(1, 8, 256, NBREG_CTAS256);
        case 1: return NB_SHAPE(1, 4, 256, NBREG_WARPS_SMALL / 4);
        case 2: return NB_SHAPE(1, 2, 128, NBREG_WARPS_SMALL / 2);
        case 3: return NB_SHAPE(1, 1, 64, NBREG_WARPS_SMALL);
        default: return NB_SHAPE(2, 8, 256, 1);
    }
#undef NB_SHAPE
}

int force_dispatch(int variant, int shape, int* per_sm, const Plan* p, const ForceArgs* fa, cudaStream_t st) {
    switch (variant & 3) {
        case 0: return force_dispatch_v<false, false>(shape, per_sm, p, fa, st);
        case 1: return force_dispatch_v<true, false>(shape, per_sm, p, fa, st);
        case 2: return force_dispatch_v<false, true>(shape, per_sm, p, fa, st);
        default: return force_dispatch_v<true, true>(shape, per_sm, p, fa, st);
    }
}

int run_predict(nb_ctx* c, double t, cudaStream_t st, double* xp_out, double* vp_out, bool with_gather = false) {
    PredictArgs pa{};
    pa.n = c->n;
    pa.n_pairs = round_up(c->n, kJPad) / 2;
    pa.x0 = c->x0; pa.v0 = c->v0; pa.a0 = c->a0; pa.j0 = c->j0; pa.m = c->m; pa.t0 = c->t0;
    pa.t = t;
    pa.packed = reinterpret_cast<float4*>(c->ws + c->lay.packed_off);
    pa.gather = reinterpret_cast<float4*>(c->ws + c->lay.gather_off);
    pa.tile_vmax = reinterpret_cast<float*>(c->ws + c->lay.vmax_off);
    pa.xp_out = xp_out;
    pa.vp_out = vp_out;
    const int threads = 256;
    if (xp_out) {
        const int64_t pairs = (c->n + 1) / 2;
        pa.n_pairs = pairs;
        NB_CUDA(launch_k(predict_kernel<true, false>, (unsigned)((pairs + threads - 1) / threads), threads, 0, st, pa));
    } else if (with_gather) {
        NB_CUDA(launch_k(predict_kernel<false, true>, (unsigned)((pa.n_pairs + threads - 1) / threads), threads, 0, st, pa));
    } else {
        NB_CUDA(launch_k(predict_kernel<false, false>, (unsigned)((pa.n_pairs + threads - 1) / threads), threads, 0, st, pa));
    }
    return NB_OK;
}

// The kernels that gather single particles (irregular force, corrector) read the particle-major copy of the predicted
// records, which the predictor writes only on demand: make sure the context holds a prediction at t WITH that copy.
// The first such call of a context sets gather_wanted, so that from then on every prediction pass writes it.
int ensure_gather_prediction(nb_ctx* c, double t, void* stream) {
    c->gather_wanted = true;
    if (c->predicted && c->t_pred == t && c->gather_valid) return NB_OK;
    return nb_predict_j(c, t, stream);
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

extern "C" {

int nb_version(void) { return 100; }

const char* nb_strerror(int code) {
    switch (code) {
        case NB_OK: return "ok";
        case NB_E_INVAL: return "invalid argument";
        case NB_E_STATE: return "call out of order (no j-state registered / nothing predicted yet)";
        case NB_E_NOMEM: return "workspace too small or device allocation failed";
        case NB_E_CUDA: return g_errbuf[0] ? g_errbuf : "CUDA error";
        case NB_E_LIMIT:
            return "size beyond the limits of the static-scratch entry point nb_regular_force_static "
                   "(n <= 65536, n_i <= 4096, nbr_cap <= 512): use nb_create + nb_regular_force";
        default: return "unknown error code";
    }
}

size_t nb_workspace_bytes(int64_t n_max, int64_t n_i_max, int32_t nbr_cap) {
    if (n_max < 1 || n_i_max < 0 || nbr_cap < 1 || nbr_cap > kMaxNbrCap || n_max > 0x7fffff00LL ||
        n_i_max > 0x7fffffffLL)
        return 0;
    return layout(n_max, n_i_max, nbr_cap).total;
}

int nb_create(nb_ctx** out, int device, int64_t n_max, int64_t n_i_max, int32_t nbr_cap, void* dev_workspace,
              size_t workspace_bytes) {
    if (!out) return NB_E_INVAL;
    *out = nullptr;
    const size_t need = nb_workspace_bytes(n_max, n_i_max, nbr_cap);
    if (need == 0) return NB_E_INVAL;
    if (dev_workspace && workspace_bytes < need) return NB_E_NOMEM;
    if (dev_workspace && (reinterpret_cast<uintptr_t>(dev_workspace) & 255u)) return NB_E_INVAL;
    int ndev = 0;
    NB_CUDA(cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(device));
    nb_ctx* c = new (std::nothrow) nb_ctx();
    if (!c) return NB_E_NOMEM;
    c->device = device;
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
    // function attributes are per process, not per context: allow the largest list capacity any context may ask for
    if (cudaFuncSetAttribute(reduce_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)((size_t)kGatherWarps * (kMaxNbrCap + kMaxChunks) * sizeof(int32_t))) != cudaSuccess) {
        delete c;
        return cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(reduce_gather_kernel)");
    }
    if (cudaFuncSetAttribute(reduce_gather_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)((size_t)kMaxNbrCap * sizeof(int32_t))) != cudaSuccess) {
        delete c;
        return cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(reduce_gather_wide_kernel)");
    }
    if (cudaFuncSetAttribute(order_small_kernel<512, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)OrderSmall<512, 8>::smem_bytes) != cudaSuccess ||
        cudaFuncSetAttribute(order_small_kernel<1024, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)OrderSmall<1024, 8>::smem_bytes) != cudaSuccess) {
        delete c;
        return cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(order_small_kernel)");
    }
    for (int v = 0; v < 4; ++v) {
        for (int k = 0; k < kNumShapes; ++k) {
            const int rc = force_dispatch(v, k, &c->ctas_per_sm[v][k], nullptr, nullptr, nullptr);
            if (rc != NB_OK) {
                delete c;
                return rc;
            }
        }
    }
    for (int k = 1; k <= 3; ++k) {
        const int rc = force_pred_dispatch(k, &c->ctas_per_sm_pred[k], nullptr, nullptr, nullptr);
        if (rc != NB_OK) {
            delete c;
            return rc;
        }
    }
    c->n_max = n_max;
    c->n_i_max = n_i_max;
    c->cap = nbr_cap;
    c->lay = layout(n_max, n_i_max, nbr_cap);
    if (dev_workspace) {
        c->ws = static_cast<unsigned char*>(dev_workspace);
    } else {
        if (cudaMalloc(&c->ws, need) != cudaSuccess) {
            cudaGetLastError();
            delete c;
            return NB_E_NOMEM;
        }
        c->ws_owned = true;
    }
    // the list-slot counters and the control words are zero between calls: the gather kernel re-zeroes what a
    // call used, so they are cleared once, here
    if (cudaMemset(c->ws + c->lay.slot_off, 0, c->lay.ctl_off + c->lay.ctl_bytes - c->lay.slot_off) != cudaSuccess) {
        const int rc = cuda_fail(cudaGetLastError(), "cudaMemset(workspace scratch)");
        if (c->ws_owned) cudaFree(c->ws);
        delete c;
        return rc;
    }
    *out = c;
    return NB_OK;
}

int nb_destroy(nb_ctx* c) {
    if (!c) return NB_OK;
    cudaSetDevice(c->device);
    if (c->hstream) {
        cudaStreamSynchronize(c->hstream);
        cudaStreamDestroy(c->hstream);
    }
    if (c->hcopy) {
        cudaStreamSynchronize(c->hcopy);
        cudaStreamDestroy(c->hcopy);
    }
    for (int k = 0; k < kHostChunks; ++k)
        if (c->hdone[k]) cudaEventDestroy(c->hdone[k]);
    if (c->hovf) cudaFreeHost(c->hovf);
    if (c->hbuf) cudaFree(c->hbuf);
    if (c->hcsr) cudaFree(c->hcsr);
    if (c->ws_owned && c->ws) cudaFree(c->ws);
    delete c;
    return NB_OK;
}

int nb_set_j(nb_ctx* c, int64_t n, const double* x0, const double* v0, const double* a0, const double* j0,
             const double* m, const double* t0) {
    if (!c || !x0 || !v0 || !a0 || !j0 || !m || !t0) return NB_E_INVAL;
    if (n < 1 || n > c->n_max) return NB_E_INVAL;
    if (!aligned16(x0) || !aligned16(v0) || !aligned16(a0) || !aligned16(j0) || !aligned16(m) || !aligned16(t0))
        return NB_E_INVAL;  // the predictor reads 16-byte vectors
    c->n = n;
    c->x0 = x0; c->v0 = v0; c->a0 = a0; c->j0 = j0; c->m = m; c->t0 = t0;
    c->predicted = false;
    c->gather_valid = false;
    return NB_OK;
}

int nb_predict_j(nb_ctx* c, double t, void* stream) {
    if (!c) return NB_E_INVAL;
    if (c->n < 1) return NB_E_STATE;
    NB_CUDA(cudaSetDevice(c->device));
    const bool with_gather = c->gather_wanted || c->opt_gather_copy == 1;
    int rc = run_predict(c, t, static_cast<cudaStream_t>(stream), nullptr, nullptr, with_gather);
    if (rc != NB_OK) return rc;
    c->predicted = true;
    c->t_pred = t;
    c->gather_valid = with_gather;
    return NB_OK;
}

int nb_get_predicted(nb_ctx* c, double* xp, double* vp, void* stream) {
    if (!c || !xp || !vp) return NB_E_INVAL;
    if (c->n < 1 || !c->predicted) return NB_E_STATE;
    if (!aligned16(xp) || !aligned16(vp)) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(c->device));
    return run_predict(c, c->t_pred, static_cast<cudaStream_t>(stream), xp, vp);
}

int nb_regular_force(nb_ctx* c, int32_t n_i, const int32_t* i_idx, const double* r_s, double t, double* acc,
                     double* jerk, int32_t* nbr_count, int32_t* nbr_list, int32_t* n_overflow, void* stream) {
    return nb_regular_force_ex(c, n_i, i_idx, r_s, nullptr, t, acc, jerk, nullptr, nbr_count, nbr_list, n_overflow,
                               stream);
}

int nb_regular_force_ex(nb_ctx* c, int32_t n_i, const int32_t* i_idx, const double* r_s, const double* dtr, double t,
                        double* acc, double* jerk, double* pot, int32_t* nbr_count, int32_t* nbr_list,
                        int32_t* n_overflow, void* stream) {
    if (!c || !n_overflow) return NB_E_INVAL;
    if (n_i < 0 || n_i > c->n_i_max) return NB_E_INVAL;
    if (n_i > 0 && (!i_idx || !r_s || !acc || !jerk || !nbr_count || !nbr_list)) return NB_E_INVAL;
    if (c->n < 1) return NB_E_STATE;
    NB_CUDA(cudaSetDevice(c->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int launches = 0;
    const bool stale = !c->predicted || c->t_pred != t;
    // A small block (<= 128 rows) with the plain criterion predicts inside the force kernel: its j-range is split over
    // the CTAs, so every j is predicted by the CTA that uses it (force.cuh, PRED).
    bool fuse_pred = false;
    // It pays when the prediction pass is long: measured at N = 2^20, N_i = 32: 94.8 -> 73.4 us per call (the pass costs
    // 38 us, reading the fp64 state in the force kernel 19 us); at N = 65536 the pass costs 5 us and the fused kernel's
    // exposed load latency more (29.4 -> 32.1 us), hence the size limit ("fuse_pred" = 2 lifts it).
    const bool big = c->n >= kFusePredMinN || c->opt_fuse_pred == 2;
    if (stale && n_i > 0 && !dtr && !pot && c->opt_fuse_pred && big) {
        Machine m0{};
        m0.n = c->n;
        m0.row_chunk_limit = c->lay.row_chunk_limit;
        m0.num_sms = c->num_sms;
        // planned with the occupancy of the PRED instantiations (24 resident warps, not the 28 of the plain ones)
        for (int k = 0; k < kNumShapes; ++k)
            m0.ctas_per_sm[k] = (k >= 1 && k <= 3) ? c->ctas_per_sm_pred[k] : c->ctas_per_sm[0][k];
        const Plan p0 = make_plan(&m0, n_i, c->opt_i_block, c->opt_j_split);
        // one row block: every j predicted once.  A few row blocks: each predicts its j again, ~3 % more instructions
        // per block and 112 B/j of HBM reads that hide under the pair arithmetic, against a 38 us pass that nothing
        // overlaps.  It pays up to 128 rows (kFusePredMaxRows).  The row ordering, if forced, then predicts its rows'
        // positions itself (order.cuh, from_raw).
        fuse_pred = n_i <= kFusePredMaxRows && p0.shape >= 1 && p0.shape <= 3;
    }
    if (stale && !fuse_pred) {  // the fused call: S1 first, same stream
        int rc = nb_predict_j(c, t, stream);
        if (rc != NB_OK) return rc;
        ++launches;
    }
    if (n_i == 0) {
        NB_CUDA(cudaMemsetAsync(n_overflow, 0, sizeof(int32_t), st));
        c->info[5] = launches;
        return NB_OK;
    }
    Machine mach{};
    mach.n = c->n;
    mach.row_chunk_limit = c->lay.row_chunk_limit;
    mach.num_sms = c->num_sms;
    const int variant = (dtr ? 1 : 0) | (pot ? 2 : 0);
    for (int k = 0; k < kNumShapes; ++k)
        mach.ctas_per_sm[k] = (fuse_pred && k >= 1 && k <= 3) ? c->ctas_per_sm_pred[k] : c->ctas_per_sm[variant][k];
    const Plan p = make_plan(&mach, n_i, c->opt_i_block, c->opt_j_split);
    ForceArgs fa{};
    fa.raw = RawState{c->x0, c->v0, c->a0, c->j0, c->m, c->t0, t};
    fa.packed = reinterpret_cast<const float4*>(c->ws + c->lay.packed_off);
    fa.n = (int32_t)c->n;
    fa.n_pad = p.n_pad;
    fa.main_blocks = p.main_blocks;
    fa.chunk_j = p.chunk_j;
    fa.n_chunks = p.n_chunks;
    fa.n_i = n_i;
    fa.cap = c->cap;
    fa.i_idx = i_idx;
    fa.r_s = r_s;
    fa.dtr = dtr;
    fa.tile_vmax = reinterpret_cast<const float*>(c->ws + c->lay.vmax_off);
    fa.pot = pot;
    fa.acc = acc; fa.jerk = jerk; fa.nbr_count = nbr_count; fa.nbr_list = nbr_list; fa.n_overflow = n_overflow;
    fa.part_sum = reinterpret_cast<double*>(c->ws + c->lay.psum_off);
    const Shape& sh = kShapes[p.shape];
    const int64_t row0 = (int64_t)p.main_blocks * sh.rows;
    const bool has_split = p.n_chunks > 1 && row0 < n_i;
    int32_t* ctl = reinterpret_cast<int32_t*>(c->ws + c->lay.ctl_off);
    // S2, first half: process the rows in Morton order of their predicted positions (order.cuh)
    fa.perm = nullptr;
    // ... when the force kernel is long enough for the 2-5 % it gains to pay for the sort (12-18 us in one CTA up to
    // 8192 rows, ~60 us for the device-wide sort of larger blocks).  Measured break-even (A/B in one process, round 2):
    // N = 65536: 8192 rows (5.4e8 pairs) -1 %, 16384 rows (1.1e9) +2 %; N = 2^20: 512 rows (5.4e8) -1 %, 1024 rows
    // (1.1e9) +0.5 %, 8192 rows +3.4 %; N = 200000, 8192 rows (1.6e9) +1.6 %.
    const bool order_pays = (double)n_i * (double)c->n >= 1.0e9;
    if (c->opt_order_rows == 2 || (c->opt_order_rows == 1 && n_i >= kOrderMinRows && order_pays)) {
        const size_t seg = (size_t)round_up((int64_t)std::max<int64_t>(c->n_i_max, 1) * 4, 256);
        unsigned char* sb = c->ws + c->lay.sort_off;
        OrderArgs oa{};
        oa.raw = fa.raw;
        oa.from_raw = fuse_pred;
        oa.packed = fa.packed;
        oa.i_idx = i_idx;
        oa.n_i = n_i;
        oa.box = reinterpret_cast<uint32_t*>(ctl + 4);
        oa.ticket = ctl + 2;
        oa.keys = reinterpret_cast<uint32_t*>(sb);
        oa.rows = reinterpret_cast<int32_t*>(sb + 2 * seg);
        if (n_i <= kSmallSort) {
            if (n_i <= 4096)
                NB_CUDA(launch_k(order_small_kernel<512, 8>, 1, 512, OrderSmall<512, 8>::smem_bytes, st, oa));
            else
                NB_CUDA(launch_k(order_small_kernel<1024, 8>, 1, 1024, OrderSmall<1024, 8>::smem_bytes, st, oa));
            fa.perm = oa.rows;
            ++launches;
        } else {
            const unsigned blocks = (unsigned)((n_i + kOrderThreads - 1) / kOrderThreads);
            bbox_kernel<<<std::min<unsigned>(blocks, 4u * (unsigned)c->num_sms), kOrderThreads, 0, st>>>(oa);
            NB_CUDA(cudaGetLastError());
            key_kernel<<<blocks, kOrderThreads, 0, st>>>(oa);
            NB_CUDA(cudaGetLastError());
            cub::DoubleBuffer<uint32_t> dk(oa.keys, reinterpret_cast<uint32_t*>(sb + seg));
            cub::DoubleBuffer<int32_t> dv(oa.rows, reinterpret_cast<int32_t*>(sb + 3 * seg));
            size_t temp = c->lay.sort_temp_bytes;
            NB_CUDA(cub::DeviceRadixSort::SortPairs(sb + 4 * seg, temp, dk, dv, (int)n_i, 0, kKeyBits, st));
            fa.perm = dv.Current();
            launches += 3;  // bbox, keys, and the library sort counted as one
        }
    }
    fa.slot_count = reinterpret_cast<int32_t*>(c->ws + c->lay.slot_off);
    fa.overflow_ws = ctl;
    fa.fix.count = ctl + 16;
    fa.fix.rows = reinterpret_cast<int32_t*>(c->ws + c->lay.fixrow_off);
    fa.fix.escale = reinterpret_cast<float2*>(c->ws + c->lay.escale_off);
    {
        const float ca = c->opt_fixup ? 1e-3f * (float)c->opt_fix_ca_milli : 0.f;
        const float cj = c->opt_fixup ? 1e-3f * (float)c->opt_fix_cj_milli : 0.f;
        fa.fix.ca2 = ca * ca;
        fa.fix.cj2 = cj * cj;
        // rows run by one CTA over the whole j-range.  (One tile says nothing about the spread of the terms: inv_tiles = 0
        // then queues every row -- such a system is a few hundred particles, fp64 costs nothing.)
        const int64_t tiles_main = (p.n_pad + sh.jt - 1) / sh.jt;
        fa.fix.inv_tiles = tiles_main > 1 ? 1.0f / (float)tiles_main : 0.f;
    }
    int rc = fuse_pred ? force_pred_dispatch(p.shape, nullptr, &p, &fa, st)
                       : force_dispatch(variant, p.shape, nullptr, &p, &fa, st);
    if (rc != NB_OK) return rc;
    ++launches;
    {  // S5 + n_overflow: always launched, with no rows when nothing was split
        GatherArgs ga{};
        ga.row0 = (int32_t)(has_split ? row0 : n_i); ga.n_i = n_i; ga.n_chunks = p.n_chunks; ga.cap = c->cap;
        ga.perm = fa.perm;
        ga.chunk_j = p.chunk_j;
        ga.part_sum = fa.part_sum;
        ga.fix = fa.fix;
        ga.fix.inv_tiles = 1.0f / (float)((int64_t)p.n_chunks * ((p.chunk_j + sh.jt - 1) / sh.jt));  // j-split rows
        ga.acc = acc; ga.jerk = jerk; ga.pot = pot; ga.nbr_count = nbr_count; ga.nbr_list = nbr_list; ga.n_overflow = n_overflow;
        ga.slot_count = fa.slot_count; ga.overflow_ws = ctl; ga.ticket = ctl + 1;
        if (c->opt_ovf_first) {
            ga.ovf_count = ctl + 24;
            ga.ovf_rows = reinterpret_cast<int32_t*>(c->ws + c->lay.ovfrow_off);
        }
        const int64_t split_rows = has_split ? n_i - row0 : 0;
        const unsigned blocks = (unsigned)std::max<int64_t>(1, (split_rows + kGatherWarps - 1) / kGatherWarps);
        if (has_split && p.n_chunks > kWideGatherChunks && split_rows <= kWideGatherRows) {  // few rows, many chunks
            NB_CUDA(launch_k(reduce_gather_wide_kernel, (unsigned)split_rows,
                             split_rows <= kWideFewRows ? kWideThreadsFew : kWideThreads, (size_t)c->cap * sizeof(int32_t), st,
                             ga));
        } else {
            const size_t stage = (size_t)kGatherWarps * (c->cap + p.n_chunks) * sizeof(int32_t);
            NB_CUDA(launch_k(reduce_gather_kernel, blocks, kGatherWarps * 32, stage, st, ga));
        }
        ++launches;
    }
    if (c->opt_ovf_first && has_split) {  // reproducible lists for overflowed j-split rows (fixup.cuh)
        OverflowListArgs oa{};
        oa.raw = fa.raw;
        oa.packed = fuse_pred ? nullptr : fa.packed;
        oa.n = (int32_t)c->n; oa.cap = c->cap;
        oa.i_idx = i_idx; oa.r_s = r_s; oa.dtr = dtr;
        oa.nbr_list = nbr_list;
        oa.count = ctl + 24; oa.rows = reinterpret_cast<int32_t*>(c->ws + c->lay.ovfrow_off); oa.done = ctl + 25;
        const unsigned grid = (unsigned)(2 * c->num_sms);
        if (dtr) NB_CUDA(launch_k(overflow_list_kernel<true>, grid, kOvfWarps * 32, 0, st, oa));
        else NB_CUDA(launch_k(overflow_list_kernel<false>, grid, kOvfWarps * 32, 0, st, oa));
        ++launches;
    }
    if (c->opt_fixup) {  // fp64 fix-up of the rows the two kernels queued (usually none: every CTA returns at once)
        FixupArgs xa{};
        xa.raw = fa.raw;
        xa.n = (int32_t)c->n;
        xa.i_idx = i_idx; xa.r_s = r_s; xa.dtr = dtr;
        xa.acc = acc; xa.jerk = jerk;
        xa.count = fa.fix.count; xa.rows = fa.fix.rows;
        xa.part = fa.part_sum;
        xa.tickets = reinterpret_cast<int32_t*>(c->ws + c->lay.ftick_off);
        xa.done = ctl + 17;
        xa.stat_last = ctl + 18;
        xa.stat_total = reinterpret_cast<unsigned long long*>(ctl + 20);
        const unsigned grid = (unsigned)std::min(kFixMaxGrid, 2 * c->num_sms);
        if (dtr) NB_CUDA(launch_k(fixup_kernel<true>, grid, kFixThreads, 0, st, xa));
        else NB_CUDA(launch_k(fixup_kernel<false>, grid, kFixThreads, 0, st, xa));
        ++launches;
    }
    c->info[0] = sh.rows; c->info[1] = sh.ipt; c->info[2] = p.n_chunks; c->info[3] = p.grid;
    c->info[4] = p.n_blocks - p.main_blocks; c->info[5] = launches; c->info[6] = sh.jt;
    c->info[7] = mach.ctas_per_sm[p.shape];
    return NB_OK;
}

namespace {

constexpr int64_t kIrrActRatio = 96;

int irregular_launch(nb_ctx* c, int32_t n_i, const int32_t* i_idx, const int32_t* nbr_count, const int32_t* nbr_list,
                     int32_t list_stride, double t, double* acc, double* jerk, void* stream, bool act) {
    if (!c) return NB_E_INVAL;
    if (n_i < 0 || n_i > c->n_i_max || list_stride < 1) return NB_E_INVAL;
    if (n_i > 0 && (!i_idx || !nbr_count || !nbr_list || !acc || !jerk)) return NB_E_INVAL;
    if (c->n < 1) return NB_E_STATE;
    NB_CUDA(cudaSetDevice(c->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (!act) {  // predict all particles first, same stream (PRED_ALL), unless the context already holds them
        int rc = ensure_gather_prediction(c, t, stream);
        if (rc != NB_OK) return rc;
    }
    if (n_i == 0) return NB_OK;
    IrregularArgs ia{};
    ia.raw = RawState{c->x0, c->v0, c->a0, c->j0, c->m, c->t0, t};
    ia.gather = reinterpret_cast<const float4*>(c->ws + c->lay.gather_off);
    ia.n = (int32_t)c->n;
    ia.n_i = n_i;
    ia.list_stride = list_stride;
    ia.i_idx = i_idx; ia.nbr_count = nbr_count; ia.nbr_list = nbr_list;
    ia.acc = acc; ia.jerk = jerk;
    const unsigned blocks = (unsigned)((n_i + kIrrWarps - 1) / kIrrWarps);
    if (act) irregular_kernel<true><<<blocks, kIrrWarps * 32, 0, st>>>(ia);
    else irregular_kernel<false><<<blocks, kIrrWarps * 32, 0, st>>>(ia);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

}  // namespace

int nb_irregular_force(nb_ctx* c, int32_t n_i, const int32_t* i_idx, const int32_t* nbr_count,
                       const int32_t* nbr_list, int32_t list_stride, double t, double* acc, double* jerk,
                       void* stream) {
    // The paper's switch between PRED_ALL and PRED_ACT (NPACT of Listing C1): with no prediction at t in
    // the context, a block of at most n / kIrrActRatio rows predicts what it gathers (measured turn-around: ~3000 rows
    // at n = 65536, ~10000 at n = 2^20).  Both modes return the same bits.
    const bool stale = c && (!c->predicted || c->t_pred != t || !c->gather_valid);
    const bool act = c && (c->opt_irr_pred == 2 ||
                           (c->opt_irr_pred == 0 && stale && (int64_t)n_i * kIrrActRatio <= c->n));
    return irregular_launch(c, n_i, i_idx, nbr_count, nbr_list, list_stride, t, acc, jerk, stream, act);
}

int nb_irregular_force_act(nb_ctx* c, int32_t n_i, const int32_t* i_idx, const int32_t* nbr_count,
                           const int32_t* nbr_list, int32_t list_stride, double t, double* acc, double* jerk,
                           void* stream) {
    return irregular_launch(c, n_i, i_idx, nbr_count, nbr_list, list_stride, t, acc, jerk, stream, true);
}

int nb_regular_correct(nb_ctx* c, int32_t n_i, const nb_corrector_io* io, double t, void* stream) {
    if (!c || !io) return NB_E_INVAL;
    if (n_i < 0 || n_i > c->n_i_max || io->list_stride < 1 || io->old_stride < 1) return NB_E_INVAL;
    if (n_i > 0 && (!io->i_idx || !io->dt_r || !io->fr0 || !io->frd0 || !io->acc || !io->jerk || !io->nbr_count ||
                    !io->nbr_list || !io->old_count || !io->old_list || !io->f1 || !io->fd1 || !io->d2 || !io->d3 ||
                    !io->dx || !io->dv))
        return NB_E_INVAL;
    if (io->r_s_new && (!io->r_s || !io->n_p)) return NB_E_INVAL;
    if (c->n < 1) return NB_E_STATE;
    NB_CUDA(cudaSetDevice(c->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // as nb_irregular_force: a small block without a prediction at t predicts what it gathers ("irr_pred")
    const bool stale = !c->predicted || c->t_pred != t || !c->gather_valid;
    const bool act = c->opt_irr_pred == 2 || (c->opt_irr_pred == 0 && stale && (int64_t)n_i * kIrrActRatio <= c->n);
    if (!act) {
        int rc = ensure_gather_prediction(c, t, stream);
        if (rc != NB_OK) return rc;
    }
    if (n_i == 0) return NB_OK;
    CorrectorArgs ca{};
    ca.raw = RawState{c->x0, c->v0, c->a0, c->j0, c->m, c->t0, t};
    ca.gather = reinterpret_cast<const float4*>(c->ws + c->lay.gather_off);
    ca.n = (int32_t)c->n;
    ca.n_i = n_i;
    ca.i_idx = io->i_idx; ca.dt_r = io->dt_r; ca.fr0 = io->fr0; ca.frd0 = io->frd0;
    ca.acc = io->acc; ca.jerk = io->jerk;
    ca.new_count = io->nbr_count; ca.new_list = io->nbr_list; ca.new_stride = io->list_stride;
    ca.old_count = io->old_count; ca.old_list = io->old_list; ca.old_stride = io->old_stride;
    ca.r_s = io->r_s; ca.n_p = io->n_p;
    ca.f1 = io->f1; ca.fd1 = io->fd1; ca.d2 = io->d2; ca.d3 = io->d3; ca.dx = io->dx; ca.dv = io->dv;
    ca.r_s_new = io->r_s_new;
    const unsigned blocks = (unsigned)((n_i + kIrrWarps - 1) / kIrrWarps);
    if (act) corrector_kernel<true><<<blocks, kIrrWarps * 32, 0, st>>>(ca);
    else corrector_kernel<false><<<blocks, kIrrWarps * 32, 0, st>>>(ca);
    NB_CUDA(cudaGetLastError());
    return NB_OK;
}

static int regular_force_host_impl(nb_ctx* c, int64_t n, const double* x0, const double* v0, const double* a0,
                                   const double* j0, const double* m, const double* t0, int32_t n_i,
                                   const int32_t* i_idx, const double* r_s, double t, double* acc, double* jerk,
                                   int32_t* nbr_count, int32_t* nbr_list, int64_t* nbr_offset, int32_t* nbr_packed,
                                   int64_t packed_capacity, int32_t* n_overflow);

int nb_regular_force_host(nb_ctx* c, int64_t n, const double* x0, const double* v0, const double* a0,
                          const double* j0, const double* m, const double* t0, int32_t n_i, const int32_t* i_idx,
                          const double* r_s, double t, double* acc, double* jerk, int32_t* nbr_count,
                          int32_t* nbr_list, int32_t* n_overflow) {
    if (n_i > 0 && !nbr_list) return NB_E_INVAL;
    const int rc = regular_force_host_impl(c, n, x0, v0, a0, j0, m, t0, n_i, i_idx, r_s, t, acc, jerk, nbr_count,
                                           nbr_list, nullptr, nullptr, 0, n_overflow);
    if (rc != NB_OK && c) {  // leave nothing of this call in flight: the caller may free or reuse its host buffers
        if (c->hstream) cudaStreamSynchronize(c->hstream);
        if (c->hcopy) cudaStreamSynchronize(c->hcopy);
    }
    return rc;
}

int nb_regular_force_host_csr(nb_ctx* c, int64_t n, const double* x0, const double* v0, const double* a0,
                              const double* j0, const double* m, const double* t0, int32_t n_i, const int32_t* i_idx,
                              const double* r_s, double t, double* acc, double* jerk, int32_t* nbr_count,
                              int64_t* nbr_offset, int32_t* nbr_packed, int64_t packed_capacity, int32_t* n_overflow) {
    if (!nbr_offset || packed_capacity < 0 || (packed_capacity > 0 && !nbr_packed)) return NB_E_INVAL;
    const int rc = regular_force_host_impl(c, n, x0, v0, a0, j0, m, t0, n_i, i_idx, r_s, t, acc, jerk, nbr_count,
                                           nullptr, nbr_offset, nbr_packed, packed_capacity, n_overflow);
    if (rc != NB_OK && c) {
        if (c->hstream) cudaStreamSynchronize(c->hstream);
        if (c->hcopy) cudaStreamSynchronize(c->hcopy);
    }
    return rc;
}

static int regular_force_host_impl(nb_ctx* c, int64_t n, const double* x0, const double* v0, const double* a0,
                                   const double* j0, const double* m, const double* t0, int32_t n_i,
                                   const int32_t* i_idx, const double* r_s, double t, double* acc, double* jerk,
                                   int32_t* nbr_count, int32_t* nbr_list, int64_t* nbr_offset, int32_t* nbr_packed,
                                   int64_t packed_capacity, int32_t* n_overflow) {
    const bool csr = nbr_offset != nullptr;
    if (!c || !x0 || !v0 || !a0 || !j0 || !m || !t0 || !n_overflow) return NB_E_INVAL;
    if (n < 1 || n > c->n_max || n_i < 0 || n_i > c->n_i_max) return NB_E_INVAL;
    if (n_i > 0 && (!i_idx || !r_s || !acc || !jerk || !nbr_count)) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(c->device));
    if (!c->hstream) NB_CUDA(cudaStreamCreateWithFlags(&c->hstream, cudaStreamNonBlocking));
    if (!c->hcopy) NB_CUDA(cudaStreamCreateWithFlags(&c->hcopy, cudaStreamNonBlocking));
    for (int k = 0; k < kHostChunks; ++k)
        if (!c->hdone[k]) NB_CUDA(cudaEventCreateWithFlags(&c->hdone[k], cudaEventDisableTiming));
    if (!c->hovf) NB_CUDA(cudaMallocHost(&c->hovf, 2 * kHostChunks * sizeof(int32_t) + kHostChunks * sizeof(int64_t)));
    // device mirrors, carved from one allocation sized for n_max / n_i_max / cap
    const size_t nmax = (size_t)c->n_max, imax = (size_t)c->n_i_max;
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off += (size_t)round_up((int64_t)bytes, 256); return o; };
    const size_t o_x0 = carve(nmax * 24), o_v0 = carve(nmax * 24), o_a0 = carve(nmax * 24), o_j0 = carve(nmax * 24);
    const size_t o_m = carve(nmax * 8), o_t0 = carve(nmax * 8);
    const size_t o_idx = carve(imax * 4), o_rs = carve(imax * 8);
    const size_t o_acc = carve(imax * 24), o_jrk = carve(imax * 24), o_cnt = carve(imax * 4);
    const size_t o_lst = carve(imax * (size_t)c->cap * 4), o_ovf = carve(256);
    if (!c->hbuf) {
        if (cudaMalloc(&c->hbuf, off) != cudaSuccess) {
            cudaGetLastError();
            return NB_E_NOMEM;
        }
        c->hbuf_bytes = off;
    }
    // CSR mode: the stored entries of every row packed back to back (first use allocates; worst case n_i_max x cap),
    // row offsets (local to a row chunk), and the scan's scratch
    size_t scan_temp = 0;
    if (csr) {
        StoredLen f{nullptr, c->cap};
        auto it = thrust::make_transform_iterator(thrust::counting_iterator<int64_t>(0), f);
        cub::DeviceScan::ExclusiveSum(nullptr, scan_temp, it, (int64_t*)nullptr, (int)(c->n_i_max + 1));  // rows + the total
        scan_temp = (size_t)round_up((int64_t)scan_temp, 256) + 256;
        if (!c->hcsr) {
            const size_t bytes = (size_t)round_up((int64_t)(imax * (size_t)c->cap * 4), 256) +
                                 (size_t)round_up((int64_t)((imax + 1) * 8), 256) + scan_temp + 256;
            if (cudaMalloc(&c->hcsr, bytes) != cudaSuccess) {
                cudaGetLastError();
                return NB_E_NOMEM;
            }
        }
    }
    int32_t* d_packed = reinterpret_cast<int32_t*>(c->hcsr);
    int64_t* d_off = csr ? reinterpret_cast<int64_t*>(c->hcsr + (size_t)round_up((int64_t)(imax * (size_t)c->cap * 4), 256))
                         : nullptr;
    unsigned char* d_scan = csr ? reinterpret_cast<unsigned char*>(d_off) + (size_t)round_up((int64_t)((imax + 1) * 8), 256)
                                : nullptr;
    unsigned char* b = c->hbuf;
    cudaStream_t st = c->hstream, cs = c->hcopy;
    const size_t nn = (size_t)n, ni = (size_t)n_i, cap = (size_t)c->cap;
    NB_CUDA(cudaMemcpyAsync(b + o_x0, x0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_v0, v0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_a0, a0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_j0, j0, nn * 24, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_m, m, nn * 8, cudaMemcpyHostToDevice, st));
    NB_CUDA(cudaMemcpyAsync(b + o_t0, t0, nn * 8, cudaMemcpyHostToDevice, st));
    if (n_i > 0) {
        NB_CUDA(cudaMemcpyAsync(b + o_idx, i_idx, ni * 4, cudaMemcpyHostToDevice, st));
        NB_CUDA(cudaMemcpyAsync(b + o_rs, r_s, ni * 8, cudaMemcpyHostToDevice, st));
    }
    int rc = nb_set_j(c, n, (const double*)(b + o_x0), (const double*)(b + o_v0), (const double*)(b + o_a0),
                      (const double*)(b + o_j0), (const double*)(b + o_m), (const double*)(b + o_t0));
    if (rc != NB_OK) return rc;
    // row chunks: compute chunk k on the compute stream, copy its rows back on the copy stream meanwhile
    // ... when that pays: a row costs ~N ns of compute per 1000 j and (4 cap + 52) B of copy at ~50 GB/s (dense lists;
    // ~4 x 100 + 60 B in CSR form); splitting a block costs a few per cent of kernel efficiency, so it is done only if
    // the copy is >= 10 % of the compute
    // (CSR form: a row is ~460 B; every row chunk also costs its own launches, a scan and a host synchronisation, so the
    // copy must be a quarter of the compute before chunks pay: config 3 in 4 chunks 5.16 ms, in one 4.8 ms)
    const double row_bytes = csr ? 460.0 : (double)(4 * (int64_t)c->cap + 52);
    const bool overlap_pays = row_bytes / 50.0 >= (csr ? 0.25 : 0.1) * (double)n / 1000.0;
    int64_t rows_per_chunk = std::max<int64_t>(kHostChunkMinRows, (n_i + kHostChunks - 1) / kHostChunks);
    rows_per_chunk = round_up(rows_per_chunk, 1024);
    if (!overlap_pays) rows_per_chunk = round_up(std::max<int64_t>(n_i, 1), 1024);
    const int n_chunks = n_i > 0 ? (int)((n_i + rows_per_chunk - 1) / rows_per_chunk) : 1;
    // first everything that computes, then, chunk by chunk as they finish, the copies.  Dense mode: only the columns of
    // nbr_list that hold entries travel (the longest stored list of the chunk, rounded up to 32).  CSR mode: the stored
    // entries are packed on the device (exclusive scan of min(count, cap) + one warp per row) and travel back to back.
    int32_t* d_ovf = (int32_t*)(b + o_ovf);          // [kHostChunks] overflow counts
    int32_t* d_wid = d_ovf + kHostChunks;            // [kHostChunks] longest stored lists
    int64_t* d_tot = (int64_t*)(d_wid + kHostChunks);  // [kHostChunks] stored entries of each chunk (CSR)
    int64_t* h_tot = (int64_t*)(c->hovf + 2 * kHostChunks);
    NB_CUDA(cudaMemsetAsync(d_wid, 0, kHostChunks * sizeof(int32_t), st));
    for (int k = 0; k < n_chunks; ++k) {
        const size_t r0 = (size_t)k * (size_t)rows_per_chunk;
        const size_t nr = n_i > 0 ? std::min<size_t>((size_t)rows_per_chunk, ni - r0) : 0;
        rc = nb_regular_force(c, (int32_t)nr, (const int32_t*)(b + o_idx) + r0, (const double*)(b + o_rs) + r0, t,
                              (double*)(b + o_acc) + 3 * r0, (double*)(b + o_jrk) + 3 * r0, (int32_t*)(b + o_cnt) + r0,
                              (int32_t*)(b + o_lst) + r0 * cap, d_ovf + k, st);
        if (rc != NB_OK) return rc;
        if (nr > 0 && !csr) {
            const unsigned blocks = (unsigned)std::min<size_t>((nr + 255) / 256, 1024);
            list_width_kernel<<<blocks, 256, 0, st>>>((const int32_t*)(b + o_cnt) + r0, (int32_t)nr, c->cap, d_wid + k);
            NB_CUDA(cudaGetLastError());
        }
        if (csr) {  // offsets of the chunk's rows (local: the chunk's first row starts at 0), its total, the packed entries
            StoredLen f{(const int32_t*)(b + o_cnt) + r0, c->cap};
            auto it = thrust::make_transform_iterator(thrust::counting_iterator<int64_t>(0), f);
            size_t temp = scan_temp;
            NB_CUDA(cub::DeviceScan::ExclusiveSum(d_scan, temp, it, d_off + r0, (int)nr + 1, st));  // [nr] = the total
            NB_CUDA(cudaMemcpyAsync(d_tot + k, d_off + r0 + nr, sizeof(int64_t), cudaMemcpyDeviceToDevice, st));
            if (nr > 0) {
                const unsigned blocks = (unsigned)((nr + kGatherWarps - 1) / kGatherWarps);
                pack_lists_kernel<<<blocks, kGatherWarps * 32, 0, st>>>((const int32_t*)(b + o_cnt) + r0,
                                                                       (const int32_t*)(b + o_lst) + r0 * cap, (int32_t)nr,
                                                                       c->cap, d_off + r0, d_packed + r0 * cap);
                NB_CUDA(cudaGetLastError());
            }
            NB_CUDA(cudaMemcpyAsync(h_tot + k, d_tot + k, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        }
        NB_CUDA(cudaMemcpyAsync(c->hovf + k, d_ovf + k, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        NB_CUDA(cudaMemcpyAsync(c->hovf + kHostChunks + k, d_wid + k, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        NB_CUDA(cudaEventRecord(c->hdone[k], st));
    }
    int64_t base = 0;      // CSR: entries of the chunks before this one
    int64_t bases[kHostChunks + 1] = {0};
    bool fits = true;
    for (int k = 0; k < n_chunks; ++k) {
        const size_t r0 = (size_t)k * (size_t)rows_per_chunk;
        const size_t nr = n_i > 0 ? std::min<size_t>((size_t)rows_per_chunk, ni - r0) : 0;
        NB_CUDA(cudaEventSynchronize(c->hdone[k]));  // chunk k is final on the device, its list width / total is known
        bases[k] = base;
        if (nr == 0) continue;
        NB_CUDA(cudaMemcpyAsync(acc + 3 * r0, (double*)(b + o_acc) + 3 * r0, nr * 24, cudaMemcpyDeviceToHost, cs));
        NB_CUDA(cudaMemcpyAsync(jerk + 3 * r0, (double*)(b + o_jrk) + 3 * r0, nr * 24, cudaMemcpyDeviceToHost, cs));
        NB_CUDA(cudaMemcpyAsync(nbr_count + r0, (int32_t*)(b + o_cnt) + r0, nr * 4, cudaMemcpyDeviceToHost, cs));
        if (csr) {
            const int64_t tot = h_tot[k];
            NB_CUDA(cudaMemcpyAsync(nbr_offset + r0, d_off + r0, nr * 8, cudaMemcpyDeviceToHost, cs));
            if (base + tot <= packed_capacity) {
                if (tot > 0)
                    NB_CUDA(cudaMemcpyAsync(nbr_packed + base, d_packed + r0 * cap, (size_t)tot * 4, cudaMemcpyDeviceToHost, cs));
            } else {
                fits = false;  // offsets and counts still arrive, so the caller knows the size to come back with
            }
            base += tot;
        } else {
            const size_t width = std::min<size_t>(cap, (size_t)round_up(c->hovf[kHostChunks + k], 32));
            if (width > 0)
                NB_CUDA(cudaMemcpy2DAsync(nbr_list + r0 * cap, cap * 4, (int32_t*)(b + o_lst) + r0 * cap, cap * 4, width * 4,
                                          nr, cudaMemcpyDeviceToHost, cs));
        }
    }
    NB_CUDA(cudaStreamSynchronize(st));
    NB_CUDA(cudaStreamSynchronize(cs));
    if (csr) {  // chunk-local offsets -> global
        for (int k = 1; k < n_chunks; ++k) {
            const size_t r0 = (size_t)k * (size_t)rows_per_chunk;
            const size_t nr = std::min<size_t>((size_t)rows_per_chunk, ni - r0);
            for (size_t q = 0; q < nr; ++q) nbr_offset[r0 + q] += bases[k];
        }
        nbr_offset[ni] = base;
    }
    int32_t total_overflow = 0;
    for (int k = 0; k < n_chunks; ++k) total_overflow += c->hovf[k];
    *n_overflow = total_overflow;
    // the registered pointers are the context's own mirrors; they stay valid, but a new host call overwrites them
    return fits ? NB_OK : NB_E_NOMEM;
}

int nb_get_error_scale(nb_ctx* c, int32_t n_i, float* escale, void* stream) {
    if (!c || n_i < 0 || n_i > c->n_i_max || (n_i > 0 && !escale)) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(c->device));
    if (n_i > 0)
        NB_CUDA(cudaMemcpyAsync(escale, c->ws + c->lay.escale_off, (size_t)n_i * sizeof(float2),
                                cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(stream)));
    return NB_OK;
}

int nb_fixup_stats(nb_ctx* c, int64_t stats[2], void* stream) {
    if (!c || !stats) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(c->device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int32_t h[4] = {0, 0, 0, 0};
    NB_CUDA(cudaMemcpyAsync(h, c->ws + c->lay.ctl_off + 18 * sizeof(int32_t), sizeof(h), cudaMemcpyDeviceToHost, st));
    NB_CUDA(cudaStreamSynchronize(st));
    unsigned long long total;
    memcpy(&total, h + 2, sizeof(total));
    stats[0] = h[0];
    stats[1] = (int64_t)total;
    return NB_OK;
}

int nb_set_option(nb_ctx* c, const char* key, int64_t value) {
    if (!c || !key || value < 0) return NB_E_INVAL;
    if (!strcmp(key, "j_split")) {
        c->opt_j_split = value;
        return NB_OK;
    }
    if (!strcmp(key, "order_rows")) {
        if (value > 2) return NB_E_INVAL;
        c->opt_order_rows = value;
        return NB_OK;
    }
    if (!strcmp(key, "fuse_pred")) {
        if (value > 2) return NB_E_INVAL;
        c->opt_fuse_pred = value;
        return NB_OK;
    }
    if (!strcmp(key, "pdl")) {
        if (value > 1) return NB_E_INVAL;
        g_pdl = value != 0;
        return NB_OK;
    }
    if (!strcmp(key, "gather_copy")) {
        if (value > 1) return NB_E_INVAL;
        c->opt_gather_copy = value;
        return NB_OK;
    }
    if (!strcmp(key, "ovf_first_in_j")) {
        if (value > 1) return NB_E_INVAL;
        c->opt_ovf_first = value;
        return NB_OK;
    }
    if (!strcmp(key, "fixup")) {
        if (value > 1) return NB_E_INVAL;
        c->opt_fixup = value;
        return NB_OK;
    }
    if (!strcmp(key, "fixup_ca_milli")) {
        c->opt_fix_ca_milli = value;
        return NB_OK;
    }
    if (!strcmp(key, "fixup_cj_milli")) {
        c->opt_fix_cj_milli = value;
        return NB_OK;
    }
    if (!strcmp(key, "irr_pred")) {
        if (value > 2) return NB_E_INVAL;
        c->opt_irr_pred = value;
        return NB_OK;
    }
    if (!strcmp(key, "i_block")) {
        if (value != 0 && value != 32 && value != 64 && value != 128 && value != 256 && value != 512)
            return NB_E_INVAL;
        c->opt_i_block = value;
        return NB_OK;
    }
    return NB_E_INVAL;
}

int nb_plan(int64_t n, int32_t n_i, int32_t num_sms, const int32_t ctas_per_sm[5], int64_t i_block, int64_t j_split,
            int64_t info[8]) {
    if (n < 1 || n_i < 1 || num_sms < 1 || !ctas_per_sm || !info || j_split < 0) return NB_E_INVAL;
    if (i_block != 0 && i_block != 32 && i_block != 64 && i_block != 128 && i_block != 256 && i_block != 512)
        return NB_E_INVAL;
    Machine mach{};
    mach.n = n;
    mach.row_chunk_limit = row_chunk_slots(n_i);
    mach.num_sms = num_sms;
    for (int k = 0; k < kNumShapes; ++k) {
        if (ctas_per_sm[k] < 1) return NB_E_INVAL;
        mach.ctas_per_sm[k] = ctas_per_sm[k];
    }
    const Plan p = make_plan(&mach, n_i, i_block, j_split);
    const Shape& sh = kShapes[p.shape];
    info[0] = sh.rows; info[1] = sh.ipt; info[2] = p.n_chunks; info[3] = p.grid;
    info[4] = p.n_blocks - p.main_blocks; info[5] = p.chunk_j; info[6] = sh.jt;
    info[7] = mach.ctas_per_sm[p.shape];
    return NB_OK;
}

int nb_last_launch_info(const nb_ctx* c, int64_t info[8]) {
    if (!c || !info) return NB_E_INVAL;
    for (int k = 0; k < 8; ++k) info[k] = c->info[k];
    return NB_OK;
}

}  // extern "C"

// =====================================================================================================================
// nb_regular_force_static: the regular-force call for callers that must not allocate (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  No context, no workspace argument, no cudaMalloc / cudaFree /
// allocating library routine anywhere on its path: ALL scratch of the call -- the packed predicted j-records, the
// partial sums of the j-split rows, the list-slot counters, the queues and control words of the gather and fix-up
// kernels -- lives in ONE file-scope device array of kStaticScratchBytes = 8 MiB, which every GPU that loads the library
// holds until the process exits.  Hence the limits: n <= 65536, n_i <= 4096, nbr_cap <= 512.
//
// g_static_scratch below is, in HOST code, a host-side stand-in for the device array, not a device address: a kernel
// handed that name would fault (or, where the GPU can reach host memory, silently use the wrong memory).  The device
// address is obtained once per device, with that device current, by cudaGetSymbolAddress, and it is that pointer the
// kernels get.  The same kernels as nb_regular_force run (predict_kernel, force_kernel, the gather kernel, fixup_kernel),
// planned with the smaller number of (row, j-chunk) slots the array has room for.
//
// Every call on a device shares the array, and it keeps the last call's contents: the words that must start at zero
// (slot counters, tickets, queue lengths) are cleared at the start of every call, on the caller's stream.  Calls that
// overlap on the GPU (two streams, two host threads) RACE on the array: keep the calls of one device on one stream.
// The host-side set-up of a device (symbol address, kernel attributes, occupancy) happens in the first call for that
// device: make that call outside a graph capture.
namespace {

constexpr size_t kStaticScratchBytes = 8u << 20;
constexpr int64_t kStaticMaxN = 65536, kStaticMaxNi = 4096;
constexpr int32_t kStaticMaxCap = 512;
constexpr int64_t kStaticRowChunkSlots = 65536;  // (row, j-chunk) partial sums of 64 B: 4 MiB of the array
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

struct StaticSlot {
    bool ready = false;
    nb_ctx ctx;  // a context object in static storage (never nb_create'd, never destroyed); ctx.ws = the symbol's address
};
StaticSlot g_static[kStaticMaxDevices];

// The workspace layout of layout() (above) cut down to what the static call uses: no particle-major copy (no gathering
// consumer), no row-ordering buffers (blocks this small are processed in the order given), kStaticRowChunkSlots slots.
WorkspaceLayout static_layout() {
    WorkspaceLayout w{};
    const int64_t n_pad = round_up(kStaticMaxN, kJPad);
    w.row_chunk_limit = kStaticRowChunkSlots;
    size_t off = 0;
    auto place = [&](size_t bytes, size_t& o, size_t& b) {
        o = off;
        b = bytes;
        off += (size_t)round_up((int64_t)bytes, 256);
    };
    place((size_t)n_pad * kBytesPerJ, w.packed_off, w.packed_bytes);
    place(std::max((size_t)w.row_chunk_limit * 8 * sizeof(double),
                   ((size_t)kFixMaxGrid * kFixWarps + (size_t)kStaticMaxNi + kFixWarps) * 6 * sizeof(double)),
          w.psum_off, w.psum_bytes);
    place((size_t)(n_pad / kJPad) * sizeof(float), w.vmax_off, w.vmax_bytes);
    place((size_t)(kStaticMaxNi + 1) * sizeof(int32_t), w.fixrow_off, w.fixrow_bytes);
    place((size_t)(kStaticMaxNi + 1) * sizeof(float2), w.escale_off, w.escale_bytes);
    place((size_t)(kStaticMaxNi + 1) * sizeof(int32_t), w.ovfrow_off, w.ovfrow_bytes);
    // from here on: zero at the start of every call
    place((size_t)(kStaticMaxNi + 512) * sizeof(int32_t), w.slot_off, w.slot_bytes);
    place((size_t)(kStaticMaxNi / kFixWarps + 34) * sizeof(int32_t), w.ftick_off, w.ftick_bytes);
    place(128, w.ctl_off, w.ctl_bytes);
    w.total = off;
    return w;
}

// Once per device, with that device current: the device address of the scratch array, the kernel attributes and
// occupancy figures nb_create would have set up.  Nothing here allocates.
int static_setup(int device, StaticSlot** out) {
    if (device < 0 || device >= kStaticMaxDevices) return NB_E_INVAL;
    StaticSlot& sl = g_static[device];
    *out = &sl;
    if (sl.ready) return NB_OK;
    int ndev = 0;
    NB_CUDA(cudaGetDeviceCount(&ndev));
    if (device >= ndev) return NB_E_INVAL;
    NB_CUDA(cudaSetDevice(device));
    nb_ctx& c = sl.ctx;
    c.lay = static_layout();
    if (c.lay.total > kStaticScratchBytes) return NB_E_NOMEM;  // (cannot happen: the constants above are sized to fit)
    void* dev_ptr = nullptr;
    NB_CUDA(cudaGetSymbolAddress(&dev_ptr, g_static_scratch));  // NOT &g_static_scratch: that is a host address
    if (!dev_ptr || (reinterpret_cast<uintptr_t>(dev_ptr) & 255u)) {
        snprintf(g_errbuf, sizeof(g_errbuf), "cudaGetSymbolAddress(g_static_scratch) gave an unusable address");
        return NB_E_CUDA;
    }
    c.ws = static_cast<unsigned char*>(dev_ptr);
    c.ws_owned = false;
    c.device = device;
    NB_CUDA(cudaDeviceGetAttribute(&c.num_sms, cudaDevAttrMultiProcessorCount, device));
    // function attributes are per process (nb_create sets the same ones)
    NB_CUDA(cudaFuncSetAttribute(reduce_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)((size_t)kGatherWarps * (kMaxNbrCap + kMaxChunks) * sizeof(int32_t))));
    NB_CUDA(cudaFuncSetAttribute(reduce_gather_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)((size_t)kMaxNbrCap * sizeof(int32_t))));
    for (int k = 0; k < kNumShapes; ++k) {  // plain criterion, no potential: variant 0
        const int rc = force_dispatch(0, k, &c.ctas_per_sm[0][k], nullptr, nullptr, nullptr);
        if (rc != NB_OK) return rc;
    }
    c.n_max = kStaticMaxN;
    c.n_i_max = kStaticMaxNi;
    c.cap = kStaticMaxCap;
    c.opt_order_rows = 0;   // no ordering buffers in the array
    c.opt_fuse_pred = 0;    // always the predictor pass into the array's packed records
    sl.ready = true;
    return NB_OK;
}

}  // namespace

extern "C" int nb_regular_force_static(int device, int64_t n, const double* x0, const double* v0, const double* a0,
                                       const double* j0, const double* m, const double* t0, int32_t n_i,
                                       const int32_t* i_idx, const double* r_s, double t, int32_t nbr_cap, double* acc,
                                       double* jerk, int32_t* nbr_count, int32_t* nbr_list, int32_t* n_overflow,
                                       void* stream) {
    if (n < 1 || n_i < 0 || nbr_cap < 1 || !n_overflow) return NB_E_INVAL;
    if (n > kStaticMaxN || n_i > kStaticMaxNi || nbr_cap > kStaticMaxCap) return NB_E_LIMIT;
    StaticSlot* sl = nullptr;
    int rc = static_setup(device, &sl);
    if (rc != NB_OK) return rc;
    nb_ctx* c = &sl->ctx;
    NB_CUDA(cudaSetDevice(device));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // the array keeps the last call's contents: what must start at zero is cleared here, on the caller's stream
    NB_CUDA(cudaMemsetAsync(c->ws + c->lay.slot_off, 0, c->lay.ctl_off + c->lay.ctl_bytes - c->lay.slot_off, st));
    c->cap = nbr_cap;
    rc = nb_set_j(c, n, x0, v0, a0, j0, m, t0);  // registers the pointers; the prediction is now stale ...
    if (rc != NB_OK) return rc;
    // ... so this predicts all n particles into the array first, then runs force, gather and fix-up kernels
    return nb_regular_force_ex(c, n_i, i_idx, r_s, nullptr, t, acc, jerk, nullptr, nbr_count, nbr_list, n_overflow,
                               stream);
}

extern "C" int nb_static_limits(int64_t limits[4]) {
    if (!limits) return NB_E_INVAL;
    limits[0] = kStaticMaxN;
    limits[1] = kStaticMaxNi;
    limits[2] = kStaticMaxCap;
    limits[3] = (int64_t)kStaticScratchBytes;
    return NB_OK;
}
