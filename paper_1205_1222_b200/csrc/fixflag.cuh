// fixflag.cuh -- which rows go to the fp64 fix-up pass (fixup.cuh), decided where a row's final sums are known: at the
// end of force_kernel for a row one CTA ran over the whole j-range, in the gather kernels for a j-split row.
//
// Why: the pair arithmetic is fp32 ("single precision ... sufficiently accurate ... because all the
// close interactions are skipped"; north_star prescribes it), so every term m_j R/r^3 carries a relative rounding
// error of a few 1e-7, random from pair to pair.  The row's absolute error is therefore ~ eps sqrt(sum_j |term_j|^2),
// whatever the sum itself comes to; a row whose terms cancel (a particle near the cluster centre; a row whose jerk
// happens to be small) can miss the per-particle bound 1e-6 |acc| / 1e-5 |jerk| although every term is accurate.  The
// paper keeps "options using the 'two-float' method for the coordinates and the accumulator" for such cases
// (footnote 2); here the few rows concerned are recomputed in fp64.
//
// The estimate of sum_j |term_j|^2 costs nothing in the j-loop: a tile's fp32 partial sum is the sum of ~256 terms of
// mixed direction, so the squared norms of the tile partials, which the kernel forms anyway when it flushes them into
// the fp64 running sums (S6), add up to that scale (plus |sum|^2 / tiles from the coherent part, which is harmless).
#pragma once
#include "nbreg_common.cuh"

namespace nbreg {

struct FixupFlag {
    int32_t* count;   // [1] rows queued so far in this call (zero between calls: fixup_kernel consumes and re-zeroes it)
    int32_t* rows;    // [n_i_max] the caller's rows that were queued, in arrival order
    float2* escale;   // [n_i_max] per caller's row: (sum_T |acc_T|^2, sum_T |jerk_T|^2), kept for nb_get_error_scale
    float ca2, cj2;   // C_a^2, C_j^2 (both 0: never queue)
    float inv_tiles;  // 1 / (number of j-tiles a row's sums were flushed from)
};

// q = sum_T |p_T|^2 over the T tile partials p_T of a row, whose sum is s.  The part of q that is NOT error scale is the
// coherent one: if every tile contributed its share s / T, q would be |s|^2 / T (a smooth field; it dominates when there
// are few tiles).  What is left, q - |s|^2 / T = sum_T |p_T - s / T|^2, estimates sum_j |term_j|^2.  A row is queued iff
//     C^2 (q - |s|^2 / T) > |s|^2,   i.e.   C^2 q > |s|^2 (1 + C^2 / T),
// for acc or for jerk.
__device__ __forceinline__ void fixup_flag(const FixupFlag& f, int32_t orow, float qa, float qj, double ax, double ay,
                                           double az, double jx, double jy, double jz) {
    f.escale[orow] = make_float2(qa, qj);
    const double a2 = ax * ax + ay * ay + az * az, j2 = jx * jx + jy * jy + jz * jz;
    const double ca2 = f.ca2, cj2 = f.cj2, it = f.inv_tiles;
    if (ca2 * (double)qa > a2 * (1.0 + ca2 * it) || cj2 * (double)qj > j2 * (1.0 + cj2 * it))
        f.rows[atomicAdd(f.count, 1)] = orow;
}

}  // namespace nbreg
