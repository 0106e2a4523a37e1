// irregular.cuh -- the irregular force of step (iv): eq. (7), (8), PAPER.md:94-98,
//   F_I,i = sum_{j in L_i} m_j R_ij / r^3,   dF_I,i/dt = sum_{j in L_i} m_j [V_ij / r^3 - 3 (R_ij.V_ij) R_ij / r^5],
// over the members of each active particle's neighbour list: the job of the paper's GPUIRR library
// (PAPER.md:130-140), which its authors left on the CPU in 2011 because the work is fine-grained and every j has
// to be gathered "from non-contiguous addresses indicated by the neighbour list".
//
// Here: one WARP per row.  The lanes stride over the row's list (coalesced index loads), each lane gathers its j
// from the particle-major predicted records (nbreg_common.cuh) -- which at N <= 2^20 stay resident in the 126 MB L2 --
// and evaluates the pair in fp32 on "two-float" coordinate differences, always with the low words (PAPER.md:138:
// "full single precision ... may not be accurate enough during close encounters. Thus, we employ the so-called
// 'two-float' technique").  A lane holds at most cap/32 terms in fp32 ("single precision turned out to be
// sufficient since we do not accumulate too many terms"); the 32 lane sums are added in fp64 by a
// fixed xor-shuffle tree, so the result is deterministic.  An entry equal to i (the paper's device lists may contain
// self) or coincident with i is skipped.
#pragma once
#include "nbreg_common.cuh"
#include "record.cuh"

namespace nbreg {

struct IrregularArgs {
    RawState raw;              // irregular_kernel<true> only
    const float4* gather;      // particle-major predicted records, 3 float4 per particle (nbreg_common.cuh)
    int32_t n;                 // j-particles (entries outside [0, n) are ignored)
    int32_t n_i;
    int32_t list_stride;       // ints per row of nbr_list
    const int32_t* i_idx;      // [n_i]
    const int32_t* nbr_count;  // [n_i]; min(count, list_stride) entries are used
    const int32_t* nbr_list;   // [n_i][list_stride]
    double* acc;               // [n_i][3]
    double* jerk;              // [n_i][3]
};

constexpr int kIrrWarps = 8;

template <bool ACT>
__global__ void __launch_bounds__(kIrrWarps * 32) irregular_kernel(IrregularArgs a) {
    const int lane = threadIdx.x & 31;
    const int64_t row = (int64_t)blockIdx.x * kIrrWarps + (threadIdx.x >> 5);
    if (row >= a.n_i) return;  // warp-uniform
    const int32_t i = a.i_idx[row];
    const PredRecord pi = ACT ? predict_record(a.raw, i) : load_record(a.gather, i);
    const int32_t len = min(a.nbr_count[row], a.list_stride);
    const int32_t* list = a.nbr_list + (size_t)row * a.list_stride;

    float ax = 0.f, ay = 0.f, az = 0.f, jx = 0.f, jy = 0.f, jz = 0.f;
    for (int32_t e = lane; e < len; e += 32) {
        const int32_t j = list[e];
        if (j == i || j < 0 || j >= a.n) continue;
        const PredRecord pj = ACT ? predict_record(a.raw, j) : load_record(a.gather, j);
        // two-float differences: (xh_j - xh_i) + (xl_j - xl_i)
        const float dx = (pj.xh - pi.xh) + (pj.xl - pi.xl);
        const float dy = (pj.yh - pi.yh) + (pj.yl - pi.yl);
        const float dz = (pj.zh - pi.zh) + (pj.zl - pi.zl);
        const float dvx = pj.vx - pi.vx, dvy = pj.vy - pi.vy, dvz = pj.vz - pi.vz;
        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        if (r2 == 0.f) continue;  // coincident: singular term skipped (reading R4)
        const float rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
        float ri, ri2;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(ri) : "f"(r2));
        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(ri2) : "f"(r2));
        const float mri3 = pj.m * ri * ri2;
        const float al = -3.f * rv * ri2;
        ax = fmaf(mri3, dx, ax);
        ay = fmaf(mri3, dy, ay);
        az = fmaf(mri3, dz, az);
        jx = fmaf(mri3, fmaf(al, dx, dvx), jx);
        jy = fmaf(mri3, fmaf(al, dy, dvy), jy);
        jz = fmaf(mri3, fmaf(al, dz, dvz), jz);
    }
    double s[6] = {(double)ax, (double)ay, (double)az, (double)jx, (double)jy, (double)jz};
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k] += __shfl_xor_sync(0xffffffffu, s[k], off);
    }
    if (lane < 3) {
        a.acc[row * 3 + lane] = (lane == 0) ? s[0] : (lane == 1) ? s[1] : s[2];
        a.jerk[row * 3 + lane] = (lane == 0) ? s[3] : (lane == 1) ? s[4] : s[5];
    }
}

}  // namespace nbreg
