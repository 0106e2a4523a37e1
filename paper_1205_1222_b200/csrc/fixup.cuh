// fixup.cuh -- the fp64 fix-up pass: rows of eq. (9), (10) whose sum is dominated by cancellation
// are evaluated again with fp64 pair arithmetic, so that the per-particle bound (1e-6 |acc|, 1e-5 |jerk|) holds for
// every row and not only for the typical one.  Which rows: fixflag.cuh (queued by force_kernel / the gather kernels;
// a few per 10^4 at the paper's workloads).  The paper's own answer to the same problem is footnote 2, PAPER.md:154:
// "there remain options using the 'two-float' method for the coordinates and the accumulator".
//
// The neighbour decisions are NOT taken again: a pair is left out of the fp64 sums iff the fp32 test of force_kernel's
// near path (geom_hi + geom_lo [+ rmin2_velocity], the same device functions on the same fp32 records) calls it a
// neighbour, so the result stays the sum over exactly the complement of the emitted list.  (A pair force_kernel took
// on its far path is never a neighbour by that test either: the far threshold carries a 2^-10 margin, force.cuh.)
//
// Mapping: the queued rows are taken R at a time (R = 8, or 4, 2, 1 when fewer than five rows are queued: the idle
// warps of a CTA then share a row); a work item is (group of R rows, j-chunk), and there are as many chunks as fill one
// wave of the grid.  The 256 threads of a CTA predict a tile of 256 j straight from the registered fp64 state into
// shared memory (the Horner form of predict.cuh; fp64 x_p, v_p, m and the fp32 record the neighbour test needs), then
// every warp runs its row over its share of the tile, lanes striding over j.  Lane sums are fp64, reduced by a fixed
// xor-shuffle tree; the warps that share a row are added in order, the chunks of a row in a fixed order by the CTA that
// finishes last (atomic ticket): deterministic for a given device.
// The pass always runs (one launch); with nothing queued every CTA returns at once.
#pragma once
#include "fixflag.cuh"
#include "force.cuh"
#include "record.cuh"

namespace nbreg {

constexpr int kFixWarps = 8;                 // rows per group = warps per CTA
constexpr int kFixThreads = kFixWarps * 32;  // = j per tile
constexpr int kFixMaxGrid = 1024;

struct FixupArgs {
    RawState raw;
    int32_t n;
    const int32_t* i_idx;
    const double* r_s;
    const double* dtr;       // VEL: regular time-step per row (eq. (3)), else null
    double* acc;
    double* jerk;
    int32_t* count;          // [1] queued rows (zero between calls; re-zeroed here)
    const int32_t* rows;     // [count] the caller's rows
    double* part;            // [(group, chunk)][kFixWarps][6] partial sums of the j-chunks
    int32_t* tickets;        // [groups] chunks of the group that are done (zero between calls)
    int32_t* done;           // [1] CTAs of this launch that are done (zero between calls)
    int32_t* stat_last;      // [1] rows the last call recomputed
    unsigned long long* stat_total;  // [1] rows recomputed since nb_create
};

struct RawJ {  // one particle's registered fp64 state
    double x[3], v[3], a[3], j[3], m, t0;
};
__device__ __forceinline__ RawJ load_raw(const RawState& r, int32_t j) {
    RawJ w;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        w.x[k] = __ldg(r.x0 + 3 * (size_t)j + k);
        w.v[k] = __ldg(r.v0 + 3 * (size_t)j + k);
        w.a[k] = __ldg(r.a0 + 3 * (size_t)j + k);
        w.j[k] = __ldg(r.j0 + 3 * (size_t)j + k);
    }
    w.m = __ldg(r.m + j);
    w.t0 = __ldg(r.t0 + j);
    return w;
}

template <bool VEL>
__global__ void __launch_bounds__(kFixThreads) fixup_kernel(FixupArgs a) {
    __shared__ double sx[3][kFixThreads], sv[3][kFixThreads], sm[kFixThreads];
    __shared__ float sh[3][kFixThreads], sl[3][kFixThreads], sw[3][kFixThreads];
    __shared__ double sred[kFixWarps][6];
    __shared__ int s_last;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    pdl_wait();
    const int32_t n_fix = *reinterpret_cast<volatile int32_t*>(a.count);
    if (n_fix == 0) {  // the usual case
        if (blockIdx.x == 0 && tid == 0) *a.stat_last = 0;
        return;
    }
    // Rows per CTA: a predicted tile serves up to eight rows, one per warp; with fewer than five rows queued (a small
    // active block: the call is short and this pass must be too) the idle warps take a share of the tile instead.
    // R is a function of n_fix alone: the same rows give the same bits.
    const int R = n_fix >= 5 ? 8 : n_fix >= 3 ? 4 : n_fix == 2 ? 2 : 1;
    const int nsub = kFixWarps / R, rs = warp % R, sub = warp / R;  // this warp: row slot, and which share of each tile
    const int32_t groups = (n_fix + R - 1) / R;
    const int32_t n_tiles = (a.n + kFixThreads - 1) / kFixThreads;
    // j-chunks per group: as many items as fit ONE wave of the grid (a few more than the grid would make a second,
    // almost empty wave: 63 groups x 5 chunks on 296 CTAs took twice as long as 63 x 4)
    int32_t C = min(max((int32_t)gridDim.x / groups, 1), n_tiles);
    const int32_t tpc = (n_tiles + C - 1) / C;
    C = (n_tiles + tpc - 1) / tpc;
    const int64_t items = (int64_t)groups * C;

    for (int64_t item = blockIdx.x; item < items; item += gridDim.x) {
        const int32_t g = (int32_t)(item / C), c = (int32_t)(item % C);
        const int32_t f = g * R + rs;
        const bool live = f < n_fix;  // warp-uniform
        // the item's first tile: its loads are issued before the row's chain of dependent loads below, not after it
        RawJ first{};
        {
            const int32_t j = c * tpc * kFixThreads + tid;
            if (j < a.n) first = load_raw(a.raw, j);
        }
        // ---- this warp's row: predicted in fp64, and its fp32 record exactly as force_kernel's i-setup forms it
        int32_t orow = 0, i = 0;
        double xi[3] = {0.0, 0.0, 0.0}, vi[3] = {0.0, 0.0, 0.0};
        IState I{};
        if (live) {
            orow = a.rows[f];
            i = a.i_idx[orow];
            const double dt = a.raw.t - __ldg(a.raw.t0 + i);
            float h[3], l[3], w[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double x = __ldg(a.raw.x0 + 3 * (size_t)i + k), v = __ldg(a.raw.v0 + 3 * (size_t)i + k);
                const double ac = __ldg(a.raw.a0 + 3 * (size_t)i + k), jk = __ldg(a.raw.j0 + 3 * (size_t)i + k);
                xi[k] = x + dt * (v + dt * (0.5 * ac + dt * ((1.0 / 6.0) * jk)));
                vi[k] = v + dt * (ac + dt * (0.5 * jk));
                h[k] = __double2float_rn(xi[k]);
                l[k] = __double2float_rn(xi[k] - (double)h[k]);
                w[k] = __double2float_rn(vi[k]);
            }
            I.nxh = -h[0]; I.nyh = -h[1]; I.nzh = -h[2];
            I.nxl = -l[0]; I.nyl = -l[1]; I.nzl = -l[2];
            I.nvx = -w[0]; I.nvy = -w[1]; I.nvz = -w[2];
            const double rs2 = a.r_s[orow];
            I.h2 = fmaxf(__double2float_rn(rs2 * rs2), 1.17549435e-38f);
            I.dtr = VEL ? __double2float_rn(a.dtr[orow]) : 0.f;
        }
        double s[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        const double h2_near = 1.01 * (double)I.h2;
        const int32_t t_end = min((c + 1) * tpc, n_tiles);
        for (int32_t t = c * tpc; t < t_end; ++t) {
            __syncthreads();  // the previous tile has been read by every warp
            {
                const int32_t j = t * kFixThreads + tid;
                if (j < a.n) {
                    const RawJ w = (t == c * tpc) ? first : load_raw(a.raw, j);
                    const double dt = a.raw.t - w.t0;
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        const double xp = w.x[k] + dt * (w.v[k] + dt * (0.5 * w.a[k] + dt * ((1.0 / 6.0) * w.j[k])));
                        const double vp = w.v[k] + dt * (w.a[k] + dt * (0.5 * w.j[k]));
                        const float xh = __double2float_rn(xp);
                        sx[k][tid] = xp;
                        sv[k][tid] = vp;
                        sh[k][tid] = xh;
                        sl[k][tid] = __double2float_rn(xp - (double)xh);
                        sw[k][tid] = __double2float_rn(vp);
                    }
                    sm[tid] = w.m;
                }
            }
            __syncthreads();
            if (!live) continue;
            const int32_t jn = min(kFixThreads, a.n - t * kFixThreads);
            for (int32_t jj = sub * 32 + lane; jj < jn; jj += 32 * nsub) {
                const int32_t j = t * kFixThreads + jj;
                if (j == i) continue;
                const double Rx = sx[0][jj] - xi[0], Ry = sx[1][jj] - xi[1], Rz = sx[2][jj] - xi[2];
                const double r2 = Rx * Rx + Ry * Ry + Rz * Rz;
                // The neighbour test of force_kernel's near path, on the same fp32 words (both halves hold j).  With the
                // plain criterion it is needed only close to r_s: the fp32 r^2 of the two-float difference is within
                // ~1e-6 of the fp64 one, so a pair with r^2 >= 1.01 r_s^2 cannot be a neighbour by it.
                if (VEL || r2 < h2_near) {
                    const float4 q0 = make_float4(sh[0][jj], sh[0][jj], sh[1][jj], sh[1][jj]);
                    const float4 q1 = make_float4(sh[2][jj], sh[2][jj], 0.f, 0.f);
                    const float4 q2 = make_float4(sw[0][jj], sw[0][jj], sw[1][jj], sw[1][jj]);
                    const float2 vz = make_float2(sw[2][jj], sw[2][jj]);
                    const float2 xl = make_float2(sl[0][jj], sl[0][jj]);
                    const float4 q4 = make_float4(sl[1][jj], sl[1][jj], sl[2][jj], sl[2][jj]);
                    PairGeom gm;
                    geom_hi(q0, q1, I, gm);
                    geom_lo(xl, q4, I, gm);
                    const float2 rm = VEL ? rmin2_velocity(q2, vz, I, gm) : gm.r2;
                    if (rm.x < I.h2) continue;  // neighbour: listed by force_kernel, not summed
                }
                // eq. (9), (10) in fp64
                const double Vx = sv[0][jj] - vi[0], Vy = sv[1][jj] - vi[1], Vz = sv[2][jj] - vi[2];
                if (r2 == 0.0) continue;  // coincident (reading R4)
                const double ri = rsqrt(r2), ri2 = ri * ri;
                const double mri3 = sm[jj] * ri * ri2;
                const double al = -3.0 * (Rx * Vx + Ry * Vy + Rz * Vz) * ri2;
                s[0] += mri3 * Rx;
                s[1] += mri3 * Ry;
                s[2] += mri3 * Rz;
                s[3] += mri3 * (Vx + al * Rx);
                s[4] += mri3 * (Vy + al * Ry);
                s[5] += mri3 * (Vz + al * Rz);
            }
        }
        // ---- the warp's lanes (fixed xor tree), then the warps that share the row (in order of their share)
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
            for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(0xffffffffu, s[k], off);
        }
        __syncthreads();  // sred of the previous item has been read
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 6; ++k) sred[warp][k] = s[k];
        }
        __syncthreads();
        double v = 0.0;  // lanes 0-5 of the row's first warp: one component each
        if (sub == 0 && lane < 6)
            for (int u = 0; u < nsub; ++u) v += sred[rs + u * R][lane];
        if (C == 1) {
            if (live && sub == 0 && lane < 6) {
                if (lane < 3) a.acc[(size_t)orow * 3 + lane] = v;
                else a.jerk[(size_t)orow * 3 + lane - 3] = v;
            }
            continue;
        }
        if (live && sub == 0 && lane < 6) a.part[((size_t)item * kFixWarps + rs) * 6 + lane] = v;
        __threadfence();
        __syncthreads();
        if (tid == 0) s_last = (atomicAdd(a.tickets + g, 1) == C - 1);
        __syncthreads();
        if (s_last) {  // every chunk of this group is in: lanes stride over the chunks, then the fixed shuffle tree
            __threadfence();
            if (live && sub == 0) {
                double w[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
                for (int32_t cc = lane; cc < C; cc += 32) {
                    const double* ps = a.part + (((size_t)g * C + cc) * kFixWarps + rs) * 6;
#pragma unroll
                    for (int k = 0; k < 6; ++k) w[k] += __ldcg(ps + k);
                }
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
                    for (int k = 0; k < 6; ++k) w[k] += __shfl_xor_sync(0xffffffffu, w[k], off);
                }
                if (lane < 3) {
                    a.acc[(size_t)orow * 3 + lane] = (lane == 0) ? w[0] : (lane == 1) ? w[1] : w[2];
                    a.jerk[(size_t)orow * 3 + lane] = (lane == 0) ? w[3] : (lane == 1) ? w[4] : w[5];
                }
            }
            if (tid == 0) a.tickets[g] = 0;
        }
    }
    // ---- the last CTA to finish leaves the queue empty for the next call
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(a.done, 1) == (int32_t)gridDim.x - 1) {
            *a.count = 0;
            *a.done = 0;
            *a.stat_last = n_fix;
            *a.stat_total += (unsigned long long)n_fix;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Option "ovf_first_in_j": a reproducible list for overflowed j-split rows.
//
// The list of a row keeps nbr_cap of its neighbours when it overflows (reading R7).  A row one CTA ran over the whole
// j-range keeps the first nbr_cap in ascending j; the CTAs of a j-split row reserve list slots with an atomic, so WHICH
// nbr_cap neighbours it keeps depends on the order in which they arrive and can differ from run to run (the paper's
// ring buffer at least is deterministic, PAPER.md:383-388, and PAPER.md:203 cares about reproducibility).  With the
// option on, the gather kernels queue the overflowed j-split rows and this kernel rewrites their lists: one warp per
// row walks the j-particles in ascending order, 32 at a time, repeats force_kernel's fp32 neighbour test (the same
// device functions on the same fp32 records: the packed records if the context holds a prediction, else predicted on
// the spot), and compacts the hits with ballot + popc until nbr_cap entries are stored.  Counts, overflow flag and forces
// are untouched.  Off by default: overflow is the exception (the caller sizes nbr_cap), and the walk costs a warp
// ~N / 32 iterations per overflowed row.
struct OverflowListArgs {
    RawState raw;
    const float4* packed;      // pair-interleaved predicted records, or null: predict from raw
    int32_t n;
    int32_t cap;
    const int32_t* i_idx;
    const double* r_s;
    const double* dtr;         // VEL, else null
    int32_t* nbr_list;
    int32_t* count;            // [1] queued rows (zero between calls; re-zeroed here)
    const int32_t* rows;       // [count] caller's rows
    int32_t* done;             // [1] CTAs of this launch that are done (zero between calls)
};

constexpr int kOvfWarps = 4;

template <bool VEL>
__global__ void __launch_bounds__(kOvfWarps * 32) overflow_list_kernel(OverflowListArgs a) {
    const int lane = threadIdx.x & 31;
    pdl_wait();
    const int32_t n_rows = *reinterpret_cast<volatile int32_t*>(a.count);
    if (n_rows == 0) return;
    const uint32_t lt_mask = (1u << lane) - 1u;
    for (int32_t f = blockIdx.x * kOvfWarps + (threadIdx.x >> 5); f < n_rows; f += gridDim.x * kOvfWarps) {
        const int32_t orow = a.rows[f];
        const int32_t i = a.i_idx[orow];
        auto record = [&](int32_t j) {
            if (!a.packed) return predict_record(a.raw, j);
            const float* rec = reinterpret_cast<const float*>(a.packed + (size_t)(j >> 1) * kQuadsPerPair) + (j & 1);
            PredRecord r;
            r.xh = __ldg(rec); r.yh = __ldg(rec + 2); r.zh = __ldg(rec + 4); r.m = 0.f;
            r.vx = __ldg(rec + 8); r.vy = __ldg(rec + 10); r.vz = __ldg(rec + 12);
            r.xl = __ldg(rec + 14); r.yl = __ldg(rec + 16); r.zl = __ldg(rec + 18);
            return r;
        };
        const PredRecord ri = record(i);
        IState I{};
        I.nxh = -ri.xh; I.nyh = -ri.yh; I.nzh = -ri.zh;
        I.nxl = -ri.xl; I.nyl = -ri.yl; I.nzl = -ri.zl;
        I.nvx = -ri.vx; I.nvy = -ri.vy; I.nvz = -ri.vz;
        const double rs = a.r_s[orow];
        I.h2 = fmaxf(__double2float_rn(rs * rs), 1.17549435e-38f);
        I.dtr = VEL ? __double2float_rn(a.dtr[orow]) : 0.f;
        int32_t* list = a.nbr_list + (size_t)orow * a.cap;
        int32_t pos = 0;
        for (int32_t base = 0; base < a.n && pos < a.cap; base += 32) {
            const int32_t j = base + lane;
            bool nb = false;
            if (j < a.n && j != i) {
                const PredRecord rj = record(j);
                const float4 q0 = make_float4(rj.xh, rj.xh, rj.yh, rj.yh);
                const float4 q1 = make_float4(rj.zh, rj.zh, 0.f, 0.f);
                const float4 q2 = make_float4(rj.vx, rj.vx, rj.vy, rj.vy);
                const float2 vz = make_float2(rj.vz, rj.vz);
                const float2 xl = make_float2(rj.xl, rj.xl);
                const float4 q4 = make_float4(rj.yl, rj.yl, rj.zl, rj.zl);
                PairGeom gm;
                geom_hi(q0, q1, I, gm);
                geom_lo(xl, q4, I, gm);
                const float2 rm = VEL ? rmin2_velocity(q2, vz, I, gm) : gm.r2;
                nb = rm.x < I.h2;
            }
            const uint32_t hits = __ballot_sync(0xffffffffu, nb);
            const int32_t at = pos + __popc(hits & lt_mask);
            if (nb && at < a.cap) list[at] = j;
            pos += __popc(hits);
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(a.done, 1) == (int32_t)gridDim.x - 1) {
            *a.count = 0;
            *a.done = 0;
        }
    }
}

}  // namespace nbreg
