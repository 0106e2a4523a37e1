// corrector.cuh -- the regular corrector of step (vii), and the neighbour-radius update eq. (1),
// PAPER.md:37, on the device, so that a whole regular step stays on the GPU:
//   "Execute the regular corrector.  Since the neighbour list L_i has been updated, the force polynomials should be
//    corrected to reflect the difference between the old and new list."
// The paper prints no formula, readings R16-R18, state what is computed:
//   1. F_R(L_old) = F_R(L_new) + sum_{j in L_new} f_ij - sum_{j in L_old} f_ij   (eq. (7) + (9) = total for any list):
//      the regular force at the end of the step with respect to the list the step was integrated with.  Only the
//      members of the symmetric difference are evaluated (in_list below): a member of both lists is never summed,
//      because its term can exceed the result by any factor (a hard binary companion near pericentre: 1e16 in the
//      jerk at config 4) and "+ term - term" in fp64 would leave its rounding error behind (measured: it did).
//   2. the cubic Hermite force polynomial through (F0, dF0) and (F1, dF1) (the "Hermite formulation ... for the case
//      of two force polynomials"): second and third derivative, and the dt^4, dt^5 terms of x and the
//      dt^3, dt^4 terms of v the predictor left out.
//   3. eq. (1): R_s_new = R_s_old (n_p / n_i)^(1/3), n_i = 0 counted as 1.
// One WARP per row, as in irregular.cuh (same gather of the particle-major predicted records); lanes 0..2 then do
// the fp64 arithmetic of one component each.
#pragma once
#include "irregular.cuh"

namespace nbreg {

struct CorrectorArgs {
    RawState raw;              // corrector_kernel<true>: the registered fp64 state and the time to predict to
    const float4* gather;      // particle-major predicted records
    int32_t n, n_i;
    const int32_t* i_idx;      // [n_i]
    const double* dt_r;        // [n_i] length of the regular step that ends now
    const double* fr0;         // [n_i][3] regular force at the start of the step (old list)
    const double* frd0;        // [n_i][3] its derivative
    const double* acc;         // [n_i][3] regular force now, NEW list (nb_regular_force)
    const double* jerk;        // [n_i][3]
    const int32_t* new_count;  // [n_i]
    const int32_t* new_list;   // [n_i][new_stride]
    int32_t new_stride;
    const int32_t* old_count;  // [n_i]
    const int32_t* old_list;   // [n_i][old_stride]
    int32_t old_stride;
    const double* r_s;         // [n_i] or null
    const double* n_p;         // [n_i] or null
    double* f1;                // [n_i][3] regular force now, OLD list
    double* fd1;               // [n_i][3]
    double* d2;                // [n_i][3] second derivative at the end of the step
    double* d3;                // [n_i][3] third derivative
    double* dx;                // [n_i][3] corrector increments
    double* dv;                // [n_i][3]
    double* r_s_new;           // [n_i] or null
};

// One member of a list: its fp32 pair term, added with `sign` to the lane's fp64 sums.
template <bool ACT>
__device__ __forceinline__ void signed_pair(const PredRecord& pi, const RawState& raw, const float4* gather, int32_t n,
                                            int32_t i, int32_t j, double sign, double s[6]) {
    if (j == i || j < 0 || j >= n) return;
    const PredRecord pj = ACT ? predict_record(raw, j) : load_record(gather, j);
    const float dx = (pj.xh - pi.xh) + (pj.xl - pi.xl);
    const float dy = (pj.yh - pi.yh) + (pj.yl - pi.yl);
    const float dz = (pj.zh - pi.zh) + (pj.zl - pi.zl);
    const float dvx = pj.vx - pi.vx, dvy = pj.vy - pi.vy, dvz = pj.vz - pi.vz;
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (r2 == 0.f) return;  // coincident: singular term skipped (reading R4)
    const float rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
    float ri = rsqrtf(r2);
    ri = ri * fmaf(-0.5f * r2 * ri, ri, 1.5f);  // one Newton step: the terms that do not cancel are few and near r_s
    const float ri2 = ri * ri;
    const float mri3 = pj.m * ri * ri2;
    const float al = -3.f * rv * ri2;
    s[0] += sign * (double)(mri3 * dx);
    s[1] += sign * (double)(mri3 * dy);
    s[2] += sign * (double)(mri3 * dz);
    s[3] += sign * (double)(mri3 * fmaf(al, dx, dvx));
    s[4] += sign * (double)(mri3 * fmaf(al, dy, dvy));
    s[5] += sign * (double)(mri3 * fmaf(al, dz, dvz));
}

// Is j a member of list[0, len)?  Called by the whole warp, each lane with its own j: the list passes through the
// warp 32 entries at a time and every lane compares its j with all of them (shuffle broadcast): len/32 x 32 compares
// per lane, no shared memory, no ordering assumed (the lists of j-split rows are not sorted).
__device__ __forceinline__ bool in_list(int32_t j, const int32_t* list, int32_t len, int lane) {
    bool found = false;
    for (int32_t base = 0; base < len; base += 32) {  // warp-uniform
        const int32_t o = (base + lane < len) ? list[base + lane] : -1;
#pragma unroll
        for (int k = 0; k < 32; ++k) found |= (__shfl_sync(0xffffffffu, o, k) == j);
    }
    return found;
}

// The same question for a list in strictly ascending order (what nb_regular_force writes, R11): binary search,
// <= log2(len) + 1 loads per lane from a row that sits in L1 after its first pass, against len shuffles.
__device__ __forceinline__ bool in_sorted_list(int32_t j, const int32_t* list, int32_t len) {
    int32_t lo = 0, hi = len;
    while (lo < hi) {
        const int32_t mid = (lo + hi) >> 1;
        if (list[mid] < j) lo = mid + 1; else hi = mid;
    }
    return lo < len && list[lo] == j;
}

// Is list[0, len) strictly ascending?  (warp-uniform result)
__device__ __forceinline__ bool is_ascending(const int32_t* list, int32_t len, int lane) {
    bool ok = true;
    for (int32_t e = lane; e + 1 < len; e += 32) ok &= list[e] < list[e + 1];
    return __all_sync(0xffffffffu, ok);
}

// ACT: the gathered particles are predicted on the spot from the fp64 state (record.cuh, the paper's PRED_ACT mode,
// PAPER.md:140), for a small block whose context holds no prediction at t -- e.g. right after a force call that
// predicted inside the force kernel: the regular step of a small block then runs without any prediction pass.
template <bool ACT>
__global__ void __launch_bounds__(kIrrWarps * 32) corrector_kernel(CorrectorArgs a) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * kIrrWarps + (threadIdx.x >> 5);
    if (row >= a.n_i) return;  // warp-uniform
    const int32_t i = a.i_idx[row];
    const PredRecord pi = ACT ? predict_record(a.raw, i) : load_record(a.gather, i);
    const int32_t n_new = a.new_count[row];
    const int32_t len_new = min(n_new, a.new_stride);
    const int32_t len_old = min(a.old_count[row], a.old_stride);
    const int32_t* lnew = a.new_list + (size_t)row * a.new_stride;
    const int32_t* lold = a.old_list + (size_t)row * a.old_stride;

    double s[6] = {0., 0., 0., 0., 0., 0.};
    const bool old_sorted = is_ascending(lold, len_old, lane), new_sorted = is_ascending(lnew, len_new, lane);
    for (int32_t base = 0; base < len_new; base += 32) {  // members of L_new that are not in L_old: +
        const int32_t e = base + lane;
        const int32_t j = (e < len_new) ? lnew[e] : -2;
        const bool common = old_sorted ? in_sorted_list(j, lold, len_old) : in_list(j, lold, len_old, lane);
        if (!common && j >= 0) signed_pair<ACT>(pi, a.raw, a.gather, a.n, i, j, 1.0, s);
    }
    for (int32_t base = 0; base < len_old; base += 32) {  // members of L_old that are not in L_new: -
        const int32_t e = base + lane;
        const int32_t j = (e < len_old) ? lold[e] : -2;
        const bool common = new_sorted ? in_sorted_list(j, lnew, len_new) : in_list(j, lnew, len_new, lane);
        if (!common && j >= 0) signed_pair<ACT>(pi, a.raw, a.gather, a.n, i, j, -1.0, s);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(0xffffffffu, s[k], off);
    }
    if (lane < 3) {
        const int64_t o = row * 3 + lane;
        const double df = (lane == 0) ? s[0] : (lane == 1) ? s[1] : s[2];
        const double dfd = (lane == 0) ? s[3] : (lane == 1) ? s[4] : s[5];
        const double f1 = a.acc[o] + df, fd1 = a.jerk[o] + dfd;  // 1. regular force with respect to the old list
        const double f0 = a.fr0[o], fd0 = a.frd0[o];
        const double h = a.dt_r[row], rh = 1.0 / h;
        // 2. F(tau) = f0 + fd0 tau + A tau^2/2 + B tau^3/6 through (f1, fd1) at tau = h
        const double u = (f1 - f0) * rh;                   // mean slope
        const double A = (6.0 * u - 4.0 * fd0 - 2.0 * fd1) * rh;
        const double B = (6.0 * (fd0 + fd1) - 12.0 * u) * rh * rh;
        const double h3 = h * h * h;
        a.f1[o] = f1;
        a.fd1[o] = fd1;
        a.d2[o] = A + h * B;
        a.d3[o] = B;
        a.dv[o] = h3 * (A * (1.0 / 6.0) + h * B * (1.0 / 24.0));
        a.dx[o] = h3 * h * (A * (1.0 / 24.0) + h * B * (1.0 / 120.0));
    }
    if (lane == 3 && a.r_s_new) {  // 3. eq. (1)
        const double ni = (double)max(n_new, 1);
        a.r_s_new[row] = a.r_s[row] * cbrt(a.n_p[row] / ni);
    }
}

}  // namespace nbreg
