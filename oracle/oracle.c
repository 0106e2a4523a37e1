/* oracle.c -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, obviously-correct fp64 CPU statement of the hot path of arXiv 1205.1222
 * (Nitadori & Aarseth, "Accelerating NBODY6 with GPUs"): the Ahmad-Cohen regular force.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 * It shares no code, header, table or helper with paper_1205_1222_b200/csrc (the CUDA path).
 *
 * What it computes, and where the paper says so:
 *   oracle_predict           step (iii) "Predict all particles"; CXVPRED call PAPER.md:551-552.
 *                            The paper prints no formula; BASELINE.json north_star fixes it:
 *                            x + v dt + a dt^2/2 + jerk dt^3/6, v + a dt + jerk dt^2/2   (reading R8).
 *   oracle_regular_force     eq. (9) regular force, eq. (10) its time derivative, eq. (11) neighbour list,
 *                            PAPER.md:102-108, with the plain criterion eq. (2) |R_ij| < h_i
 *                            (north_star: sum over r_ij >= r_s,i, list r_ij < r_s,i; reading R1/R2).
 *                            R_ij = R_j - R_i.  Masked direct sum in j order, nothing clever.
 *   oracle_force_given_lists same sums, "neighbour" := membership in a given list (for rows whose GPU list
 *                            differs from the oracle's only by pairs inside the 1e-6 boundary band, north_star).
 *
 *   oracle_regular_force_ex  the two variants the paper's own kernel has (Listing B2): the
 *                            velocity neighbour criterion eq. (3), PAPER.md:69-73,
 *                            R_min = min(|R_ij|, |R_ij + dtr_i V_ij|) < h_i (lines 17-19, 22, 26 of the listing), and
 *                            the potential sum "fo.pot += mrinv1": pot_i = sum m_j / r_ij over
 *                            the same non-neighbours as eq. (9) (sign as in the listing: positive).
 *
 *   oracle_irregular_force   step (iv), eq. (7), (8): force and its time derivative from the
 *                            members of a given neighbour list (the job of the paper's GPUIRR library,
 *                            PAPER.md:130-140).  Same pair term as eq. (9), (10), summed over j in L_i.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC oracle.c -o liboracle.so -lm
 * (-ffp-contract=off: no FMA contraction, so the arithmetic is exactly what is written.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Hermite predictor, Horner form.  Arrays are [n][3] row-major; t0 is [n].  dt_j = t - t0[j], any sign. */
void oracle_predict(int64_t n, const double* x0, const double* v0, const double* a0, const double* j0,
                    const double* t0, double t, double* xp, double* vp) {
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < n; ++j) {
        double dt = t - t0[j];
        for (int c = 0; c < 3; ++c) {
            int64_t q = 3 * j + c;
            xp[q] = x0[q] + dt * (v0[q] + dt * (a0[q] / 2.0 + dt * (j0[q] / 6.0)));
            vp[q] = v0[q] + dt * (a0[q] + dt * (j0[q] / 2.0));
        }
    }
}

/* One (i, j) term of eq. (9) and eq. (10) added into acc[3], jerk[3]. */
static inline void pair_term(const double R[3], const double V[3], double r2, double mj, double acc[3],
                             double jerk[3]) {
    double rv = R[0] * V[0] + R[1] * V[1] + R[2] * V[2];
    double ri2 = 1.0 / r2;
    double mri3 = mj * ri2 * sqrt(ri2);
    double al = 3.0 * rv * ri2;
    for (int c = 0; c < 3; ++c) {
        acc[c] += mri3 * R[c];
        jerk[c] += mri3 * (V[c] - al * R[c]);
    }
}

/* Regular force, jerk and neighbour list of n_i active particles against all n predicted particles.
 *   xp, vp [n][3], m [n]; i_idx [n_i] 0-based; r_s [n_i].
 *   acc, jerk [n_i][3]; count [n_i] = TRUE number of neighbours (no cap);
 *   list [n_i][list_stride] (may be NULL): first min(count, list_stride) neighbours in ascending j.
 * Conventions (DESIGN.md readings): neighbour iff r^2 < r_s^2 strictly, on squares (R2); self excluded by
 * index, never listed or counted (R3); a coincident distinct particle (r^2 = 0) is a neighbour if r_s > 0 and
 * is skipped entirely if r_s = 0 (R4); no softening (R6). */
void oracle_regular_force(int64_t n, const double* xp, const double* vp, const double* m, int64_t n_i,
                          const int32_t* i_idx, const double* r_s, double* acc, double* jerk, int32_t* count,
                          int32_t* list, int64_t list_stride) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < n_i; ++q) {
        int64_t i = i_idx[q];
        double h2 = r_s[q] * r_s[q];
        double a[3] = {0.0, 0.0, 0.0}, jk[3] = {0.0, 0.0, 0.0};
        int32_t cnt = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double R[3], V[3];
            for (int c = 0; c < 3; ++c) {
                R[c] = xp[3 * j + c] - xp[3 * i + c];
                V[c] = vp[3 * j + c] - vp[3 * i + c];
            }
            double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
            if (r2 < h2) { /* neighbour: listed, NOT summed */
                if (list && cnt < list_stride) list[q * list_stride + cnt] = (int32_t)j;
                ++cnt;
            } else if (r2 == 0.0) {
                continue; /* R4: singular term with r_s = 0 is skipped */
            } else {
                pair_term(R, V, r2, m[j], a, jk);
            }
        }
        for (int c = 0; c < 3; ++c) {
            acc[3 * q + c] = a[c];
            jerk[3 * q + c] = jk[c];
        }
        count[q] = cnt;
    }
}

static int cmp_i32(const void* a, const void* b) {
    int32_t x = *(const int32_t*)a, y = *(const int32_t*)b;
    return (x > y) - (x < y);
}

/* Same sums with the neighbour set GIVEN: j is excluded iff j is in lists[q][0..counts[q]) (or j == i, or
 * coincident).  lists rows need not be sorted. */
void oracle_force_given_lists(int64_t n, const double* xp, const double* vp, const double* m, int64_t n_i,
                              const int32_t* i_idx, const int32_t* lists, const int32_t* counts,
                              int64_t list_stride, double* acc, double* jerk) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < n_i; ++q) {
        int64_t i = i_idx[q];
        int64_t len = counts[q] < list_stride ? counts[q] : list_stride;
        int32_t* sorted = (int32_t*)malloc((size_t)(len > 0 ? len : 1) * sizeof(int32_t));
        for (int64_t s = 0; s < len; ++s) sorted[s] = lists[q * list_stride + s];
        qsort(sorted, (size_t)len, sizeof(int32_t), cmp_i32);
        double a[3] = {0.0, 0.0, 0.0}, jk[3] = {0.0, 0.0, 0.0};
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            int32_t key = (int32_t)j;
            if (len > 0 && bsearch(&key, sorted, (size_t)len, sizeof(int32_t), cmp_i32)) continue;
            double R[3], V[3];
            for (int c = 0; c < 3; ++c) {
                R[c] = xp[3 * j + c] - xp[3 * i + c];
                V[c] = vp[3 * j + c] - vp[3 * i + c];
            }
            double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
            if (r2 == 0.0) continue;
            pair_term(R, V, r2, m[j], a, jk);
        }
        for (int c = 0; c < 3; ++c) {
            acc[3 * q + c] = a[c];
            jerk[3 * q + c] = jk[c];
        }
        free(sorted);
    }
}

/* Eq. (9), (10), (11) with the VELOCITY criterion eq. (3) and the potential of Listing B2.
 *   dtr [n_i] (may be NULL = all zero): the regular time-step of row q; neighbour iff
 *       min(|R|^2, |R + dtr V|^2) < r_s^2      (Listing B2: "if (fminf(r2, r2p) < ip.h2)"),
 *   compared on squares, strictly.  dtr = 0 gives oracle_regular_force exactly.
 *   pot [n_i] (may be NULL): sum over the summed (non-neighbour) pairs of m_j / r   ("fo.pot += mrinv1").
 * Everything else as oracle_regular_force (self by index, coincident pairs, true count, ascending list). */
void oracle_regular_force_ex(int64_t n, const double* xp, const double* vp, const double* m, int64_t n_i,
                             const int32_t* i_idx, const double* r_s, const double* dtr, double* acc, double* jerk,
                             double* pot, int32_t* count, int32_t* list, int64_t list_stride) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t q = 0; q < n_i; ++q) {
        int64_t i = i_idx[q];
        double h2 = r_s[q] * r_s[q];
        double dt = dtr ? dtr[q] : 0.0;
        double a[3] = {0.0, 0.0, 0.0}, jk[3] = {0.0, 0.0, 0.0}, phi = 0.0;
        int32_t cnt = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double R[3], V[3], Rp[3];
            for (int c = 0; c < 3; ++c) {
                R[c] = xp[3 * j + c] - xp[3 * i + c];
                V[c] = vp[3 * j + c] - vp[3 * i + c];
                Rp[c] = R[c] + dt * V[c];
            }
            double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
            double r2p = Rp[0] * Rp[0] + Rp[1] * Rp[1] + Rp[2] * Rp[2];
            double rmin2 = r2p < r2 ? r2p : r2;
            if (rmin2 < h2) {
                if (list && cnt < list_stride) list[q * list_stride + cnt] = (int32_t)j;
                ++cnt;
            } else if (r2 == 0.0) {
                continue;
            } else {
                pair_term(R, V, r2, m[j], a, jk);
                phi += m[j] / sqrt(r2);
            }
        }
        for (int c = 0; c < 3; ++c) {
            acc[3 * q + c] = a[c];
            jerk[3 * q + c] = jk[c];
        }
        if (pot) pot[q] = phi;
        count[q] = cnt;
    }
}

/* Irregular force, eq. (7), (8): for row q, i = i_idx[q],
 *   acc = sum over j in L_q of m_j R_ij / r^3,   jerk = sum of m_j [V_ij / r^3 - 3 (R_ij . V_ij) R_ij / r^5],
 * L_q = lists[q*list_stride .. + min(counts[q], list_stride)), summed in list order.  An entry equal to i (the
 * paper's device lists may contain self) or coincident with i (r = 0) is skipped.
 * acc_scale, jerk_scale [n_i] (may be NULL): sums of the natural MAGNITUDES of the terms, sum m/r^2 and
 * sum 4 m |V|/r^3 (= m (|V|/r^3 + 3 |R||V||R|/r^5): R.V is bounded by |R||V|, and a rounded evaluation of R.V errs
 * in proportion to |R||V|, not to |R.V|): the yardstick for the rounding error of a sum whose terms cancel. */
void oracle_irregular_force(int64_t n, const double* xp, const double* vp, const double* m, int64_t n_i,
                            const int32_t* i_idx, const int32_t* lists, const int32_t* counts, int64_t list_stride,
                            double* acc, double* jerk, double* acc_scale, double* jerk_scale) {
    (void)n;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t q = 0; q < n_i; ++q) {
        int64_t i = i_idx[q];
        int64_t len = counts[q] < list_stride ? counts[q] : list_stride;
        double a[3] = {0.0, 0.0, 0.0}, jk[3] = {0.0, 0.0, 0.0}, sa = 0.0, sj = 0.0;
        for (int64_t e = 0; e < len; ++e) {
            int64_t j = lists[q * list_stride + e];
            if (j == i) continue;
            double R[3], V[3];
            for (int c = 0; c < 3; ++c) {
                R[c] = xp[3 * j + c] - xp[3 * i + c];
                V[c] = vp[3 * j + c] - vp[3 * i + c];
            }
            double r2 = R[0] * R[0] + R[1] * R[1] + R[2] * R[2];
            if (r2 == 0.0) continue;
            pair_term(R, V, r2, m[j], a, jk);
            double r = sqrt(r2);
            double vn = sqrt(V[0] * V[0] + V[1] * V[1] + V[2] * V[2]);
            sa += m[j] / r2;
            sj += 4.0 * m[j] * vn / (r2 * r);
        }
        for (int c = 0; c < 3; ++c) {
            acc[3 * q + c] = a[c];
            jerk[3 * q + c] = jk[c];
        }
        if (acc_scale) acc_scale[q] = sa;
        if (jerk_scale) jerk_scale[q] = sj;
    }
}
