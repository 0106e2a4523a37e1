/* nbreg.h -- C ABI of the B200-native Ahmad-Cohen regular-force path (after arXiv 1205.1222).
 *
 * The library is the GPU counterpart of the paper's GPUNB library: "GPUNB receives positions, velocities,
 * masses and time-steps of the attracting particles (j-particles) and positions, velocities and neighbour
 * radii of the attracted (active) particles (i-particles), and it returns regular forces, their time
 * derivatives and neighbour lists" (section 3.1; calls GPUNB_OPEN / GPUNB_SEND / GPUNB_REGF /
 * GPUNB_CLOSE at PAPER.md:460,557,595,714).  Differences from GPUNB_REGF: the active block is given as
 * indices + r_s + t (not pre-packed XI, VI, H2I), and the Hermite predictor of step (iii) (the
 * host routine CXVPRED at PAPER.md:551-552) runs on the device.
 *
 * Conventions
 *   - Units G = 1.  R_ij = R_j - R_i, V_ij likewise.  acc = + sum m_j R_ij / r^3.
 *   - "dev" pointers are CUDA device pointers OWNED BY THE CALLER (e.g. PyTorch tensors); "host" pointers are
 *     ordinary host memory (pinned memory makes the copies asynchronous and fast).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-pointer calls only
 *     ENQUEUE work on `stream` and return; they never synchronise the host.
 *   - [n][3] arrays are row-major (x, y, z contiguous per particle).  Indices are 0-based int32.
 *   - Every function returns NB_OK (0) or a negative NB_E_* code.  Argument and state errors (NB_E_INVAL, NB_E_STATE,
 *     NB_E_NOMEM) are found before anything is enqueued.  A call enqueues several kernels; if a later launch fails
 *     (NB_E_CUDA) the work already enqueued is NOT rolled back and the outputs are undefined.  nb_regular_force_host
 *     synchronises its internal streams before it returns, on the error paths too.
 *     nb_strerror() gives the text; for NB_E_CUDA it includes the CUDA error string of the last failure.
 *   - A context is not thread-safe and owns ONE workspace: issue its calls from one thread at a time and keep them
 *     on one stream (or order streams yourself); use one context per concurrent stream.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with NB_E_CUDA.
 */
#ifndef NBREG_H_
#define NBREG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NB_OK 0
#define NB_E_INVAL (-1) /* null pointer, n > n_max, n_i > n_i_max, negative size, cap <= 0, bad option   */
#define NB_E_STATE (-2) /* call out of order: force/predict before nb_set_j, get_predicted before predict */
#define NB_E_NOMEM (-3) /* workspace too small, or a device allocation failed                            */
#define NB_E_CUDA (-4)  /* CUDA runtime / launch error                                                     */
#define NB_E_LIMIT (-5) /* size beyond the fixed limits of nb_regular_force_static                         */

typedef struct nb_ctx nb_ctx;

/* Library version: major * 10000 + minor * 100 + patch. */
int nb_version(void);

/* Text for a return code.  The pointer stays valid until the next failing call on the same thread. */
const char* nb_strerror(int code);

/* Bytes of device workspace nb_create needs for up to n_max j-particles, active blocks of up to n_i_max rows
 * and neighbour lists of nbr_cap entries per row (1 <= nbr_cap <= 8192).  Holds the packed predicted j-records
 * (40 B per j, pair-interleaved, plus a 48 B particle-major copy for nb_irregular_force / nb_regular_correct) and, for
 * the row blocks whose j-range is split over several CTAs, 64 B of partial sums per (row, j-chunk): at
 * most 128 MB, plus ~40 B per row for list-slot counters, the queues of the fix-up passes, the error scales and the row
 * ordering.  nb_create clears the counters once; every call leaves them cleared.  Returns 0 if an argument is invalid. */
size_t nb_workspace_bytes(int64_t n_max, int64_t n_i_max, int32_t nbr_cap);

/* cf. GPUNB_OPEN(NTOT).  Creates a context on CUDA device `device`.
 * dev_workspace: dev pointer to >= nb_workspace_bytes(...) bytes, 256-byte aligned, owned by the caller and
 * kept alive until nb_destroy; or NULL, in which case the library allocates (and later frees) it itself. */
int nb_create(nb_ctx** out, int device, int64_t n_max, int64_t n_i_max, int32_t nbr_cap, void* dev_workspace,
              size_t workspace_bytes);

/* cf. GPUNB_CLOSE.  Frees only what the library allocated itself.  NULL is allowed. */
int nb_destroy(nb_ctx* ctx);

/* cf. GPUNB_SEND(NN, BODY, X, XDOT), plus CXVPRED's inputs T0, X0, X0DOT, F, FDOT.
 * Registers the j-particle state WITHOUT copying: the context keeps the six dev pointers until the next
 * nb_set_j; the arrays must stay alive and unchanged while calls that read them are in flight.
 *   x0, v0, a0, j0: dev double[n][3]  position, velocity, acceleration, jerk at the particle's own time t0
 *                                     (physical values, no 1/2 or 1/6 folded in)
 *   m, t0:          dev double[n]     mass; time of the last force evaluation
 * Invalidates any earlier prediction.  1 <= n <= n_max. */
int nb_set_j(nb_ctx* ctx, int64_t n, const double* x0, const double* v0, const double* a0, const double* j0,
             const double* m, const double* t0);

/* Step (iii): predict all n particles to time t,
 *   x_p = x0 + v0 dt + a0 dt^2/2 + j0 dt^3/6,  v_p = v0 + a0 dt + j0 dt^2/2,  dt = t - t0[j]  (any sign),
 * in fp64, and store them as packed records in the workspace: position as a double-single pair of floats
 * (hi = fl32(x_p), lo = fl32(x_p - hi)), velocity and mass as fl32.  Enqueues one kernel on `stream`. */
int nb_predict_j(nb_ctx* ctx, double t, void* stream);

/* Test hook: write the fp64 predicted state at the time of the last prediction PASS (nb_predict_j, or the pass a
 * force / irregular / corrector call ran first) to xp, vp: dev double[n][3].  Same kernel and arithmetic as
 * nb_predict_j.  A call that predicted inside its own kernel (small blocks: options "fuse_pred", "irr_pred") leaves
 * no prediction in the context: this function then returns NB_E_STATE, or the state of an older pass if the context
 * still holds one -- call nb_predict_j(t) first to be sure of t. */
int nb_get_predicted(nb_ctx* ctx, double* xp, double* vp, void* stream);

/* Step (vi), eq. (9), (10), (11), with the plain neighbour criterion eq. (2), PAPER.md:65-67:
 * for each row q (particle i = i_idx[q], radius r_s[q]) over all j != i,
 *   neighbour  iff |R_ij|^2 <  r_s^2 : j goes to the list, nothing is summed;
 *   otherwise                        : acc += m_j R_ij / r^3,  jerk += m_j [V_ij / r^3 - 3 (R_ij.V_ij) R_ij / r^5].
 * If t differs from the time of the last prediction, nb_predict_j(t) runs first on the same stream (the fused
 * call), or, for a small block, the prediction runs inside the force kernel (option "fuse_pred").  Differences are formed from the double-single positions, pair arithmetic is fp32 with rsqrt, partial
 * sums are flushed to fp64 every j-tile; outputs are fp64.
 *   n_i:        0 <= n_i <= n_i_max (0 is a no-op that only zeroes n_overflow)
 *   i_idx:      dev int32[n_i]   0-based indices into the j arrays; duplicates allowed
 *   r_s:        dev double[n_i]  neighbour radius; 0 is legal (empty list, everything summed)
 *   acc, jerk:  dev double[n_i][3]
 *   nbr_count:  dev int32[n_i]   TRUE number of neighbours (may exceed nbr_cap: overflow, not an error)
 *   nbr_list:   dev int32[n_i][nbr_cap]  row q valid in [0, min(count, nbr_cap)), ascending j; the self index
 *               is never listed or counted; entries past the count are left untouched.  An overflowed row
 *               (count > nbr_cap) holds nbr_cap of its neighbours: the first ones in j if the row ran in one
 *               CTA, otherwise whichever reserved a slot first -- which may differ between two runs -- unless option
 *               "ovf_first_in_j" is set (reading R7/R15 in DESIGN.md)
 *   n_overflow: dev int32[1]     number of rows with count > nbr_cap
 * The pair within 1e-6 (relative) of r_s may fall on either side of the test (fp32 squares). */
int nb_regular_force(nb_ctx* ctx, int32_t n_i, const int32_t* i_idx, const double* r_s, double t, double* acc,
                     double* jerk, int32_t* nbr_count, int32_t* nbr_list, int32_t* n_overflow, void* stream);

/* The two variants of the paper's own kernel (Listing B2), selected by non-NULL pointers:
 *   dtr: dev double[n_i] or NULL.  Regular time-step of each row for the VELOCITY neighbour criterion eq. (3),
 *        j is a neighbour iff min(|R_ij|^2, |R_ij + dtr V_ij|^2) < r_s^2 ("fminf(r2, r2p) < ip.h2",
 *        PAPER.md:381); everything else (what is summed, what is listed) follows from that as in
 *        nb_regular_force.  dtr = 0 reproduces nb_regular_force exactly; NULL selects the plain-criterion kernel.
 *   pot: dev double[n_i] or NULL.  pot[q] = sum of m_j / r_ij over the summed (non-neighbour) pairs
 *        ("fo.pot += mrinv1"; positive, as in the listing).
 * All other arguments, conventions and return codes as nb_regular_force. */
int nb_regular_force_ex(nb_ctx* ctx, int32_t n_i, const int32_t* i_idx, const double* r_s, const double* dtr,
                        double t, double* acc, double* jerk, double* pot, int32_t* nbr_count, int32_t* nbr_list,
                        int32_t* n_overflow, void* stream);

/* Step (iv), eq. (7), (8), PAPER.md:94-98 (the job of the paper's GPUIRR library): the IRREGULAR
 * force and its time derivative of n_i active particles, summed over the members of their neighbour lists,
 *   acc = sum_{j in L} m_j R_ij / r^3,   jerk = sum_{j in L} m_j [V_ij / r^3 - 3 (R_ij.V_ij) R_ij / r^5],
 * on the state predicted to time t (if t differs from the last prediction, either nb_predict_j(t) runs first on the
 * same stream -- all particles are predicted, the paper's PRED_ALL mode -- or, for a small block, the gathered
 * particles are predicted on the spot, PRED_ACT: see nb_irregular_force_act and option "irr_pred").  Coordinate differences are two-float
 * (PAPER.md:138), pair arithmetic fp32, the sum fp64 over 32 fp32 lane sums.
 *   i_idx:       dev int32[n_i]               0-based particle indices
 *   nbr_count:   dev int32[n_i]               list lengths; min(count, list_stride) entries are used
 *   nbr_list:    dev int32[n_i][list_stride]  e.g. the nbr_list / nbr_cap of nb_regular_force.  Entries equal to the
 *                                             row's own particle, outside [0, n), or coincident with it are skipped
 *   acc, jerk:   dev double[n_i][3]
 * Enqueues one kernel (plus the predictor if needed) on `stream`. */
int nb_irregular_force(nb_ctx* ctx, int32_t n_i, const int32_t* i_idx, const int32_t* nbr_count,
                       const int32_t* nbr_list, int32_t list_stride, double t, double* acc, double* jerk,
                       void* stream);

/* The same sums with the prediction FUSED into the gather: the paper's PRED_ACT mode ("When N_act,I is
 * small, predicting all the N particles is not efficient.  Thus, at some point (cf. NPACT ...) we switch to predict
 * only the necessary particles in this block-step").  Every gathered particle is predicted on the spot from the
 * fp64 state registered with nb_set_j (the predictor's formula, split and roundings, so both modes evaluate the same
 * fp32 records and return the same bits); no prediction pass runs and the context's predicted records are neither
 * used nor changed.  One kernel.  Costs 112 B instead of 48 B per gathered particle: for small blocks only (turn-
 * around measured in DESIGN.md section 5.6).  Arguments and return codes as nb_irregular_force. */
int nb_irregular_force_act(nb_ctx* ctx, int32_t n_i, const int32_t* i_idx, const int32_t* nbr_count,
                           const int32_t* nbr_list, int32_t list_stride, double t, double* acc, double* jerk,
                           void* stream);

/* Step (vii), PAPER.md:110 ("Execute the regular corrector.  Since the neighbour list L_i has been updated, the
 * force polynomials should be corrected to reflect the difference between the old and new list"), and the
 * neighbour-radius update eq. (1), for the n_i rows of a regular step that ends at time t.  The paper
 * prints no corrector formula; readings R16-R18 of DESIGN.md state what is computed, per row q, i = i_idx[q]:
 *   1. f1, fd1 = acc, jerk + sum_{j in L_new} f_ij - sum_{j in L_old} f_ij: the regular force and its derivative at
 *      t with respect to the OLD list (the one the step was integrated with); f_ij = the pair terms of eq. (7), (8) on
 *      the state predicted to t (if t differs from the last prediction: all particles are predicted first, or, for a
 *      small block, the gathered ones on the spot -- the switch of nb_irregular_force, option "irr_pred"), fp32 on two-float
 *      differences, summed in fp64;
 *   2. the cubic Hermite polynomial F(tau) through (fr0, frd0) at tau = 0 and (f1, fd1) at tau = dt_r:
 *      d3 = F''' = [12 (fr0 - f1) + 6 dt (frd0 + fd1)] / dt^3,  d2 = F''(dt_r) = [-6 (fr0 - f1) - dt (4 frd0 + 2 fd1)] /
 *      dt^2 + dt d3 (physical derivatives, at the END of the step), and the terms the predictor left out:
 *      dx = F''(0) dt^4/24 + F''' dt^5/120,  dv = F''(0) dt^3/6 + F''' dt^4/24  (to be ADDED to the predicted x, v);
 *   3. r_s_new = r_s (n_p / max(nbr_count, 1))^(1/3)   (eq. (1); nbr_count is the TRUE count of the new list).
 * All pointers are dev pointers owned by the caller; [n_i][3] arrays are row-major double.
 *   i_idx       int32[n_i]                 dt_r     double[n_i], > 0 (0 gives inf/nan in that row, no error)
 *   fr0, frd0   double[n_i][3]  regular force and derivative at the START of the step (old list)
 *   acc, jerk   double[n_i][3]  regular force and derivative at t, NEW list (outputs of nb_regular_force)
 *   nbr_count, nbr_list, list_stride    the new list (outputs of nb_regular_force, list_stride = nbr_cap)
 *   old_count, old_list, old_stride     the list of the step that ends; min(count, stride) entries of each list
 *                                       are used: for a row that overflowed in either list f1, fd1 miss the entries
 *                                       that were dropped (flagged by count > stride, as everywhere)
 *   r_s, n_p    double[n_i]     old radius and predicted neighbour number; both NULL skips step 3
 *   f1, fd1, d2, d3, dx, dv     double[n_i][3] outputs;   r_s_new  double[n_i] output or NULL
 * Enqueues one kernel (plus the predictor if needed) on `stream`.  NB_E_INVAL for a null required pointer, a
 * stride < 1 or n_i out of range; NB_E_STATE before nb_set_j. */
typedef struct nb_corrector_io {
    const int32_t* i_idx;
    const double* dt_r;
    const double* fr0;
    const double* frd0;
    const double* acc;
    const double* jerk;
    const int32_t* nbr_count;
    const int32_t* nbr_list;
    const int32_t* old_count;
    const int32_t* old_list;
    const double* r_s;
    const double* n_p;
    double* f1;
    double* fd1;
    double* d2;
    double* d3;
    double* dx;
    double* dv;
    double* r_s_new;
    int32_t list_stride;
    int32_t old_stride;
} nb_corrector_io;
int nb_regular_correct(nb_ctx* ctx, int32_t n_i, const nb_corrector_io* io, double t, void* stream);

/* End-to-end convenience with HOST buffers: copies the j-state and the active block to device buffers the
 * context owns (allocated on first use, sized by n_max / n_i_max / nbr_cap), runs nb_set_j + nb_regular_force
 * on an internal stream -- in up to 8 row chunks, so that the copy of one chunk's outputs back to the host runs on
 * a second stream while the next chunk is computed -- and synchronises when acc, jerk, nbr_count, nbr_list and
 * n_overflow have arrived.  Of nbr_list only the columns that hold entries are copied (up to the longest stored
 * list of each chunk, rounded up to 32): entries past a row's count are left untouched in the host array too.  All pointers are host pointers with the shapes documented above. */
int nb_regular_force_host(nb_ctx* ctx, int64_t n, const double* x0, const double* v0, const double* a0,
                          const double* j0, const double* m, const double* t0, int32_t n_i, const int32_t* i_idx,
                          const double* r_s, double t, double* acc, double* jerk, int32_t* nbr_count,
                          int32_t* nbr_list, int32_t* n_overflow);

/* The same call returning the neighbour lists in CSR form, which is what a host integrator stores anyway and a
 * fraction of the bytes of the dense [n_i][nbr_cap] rectangle (config 5: ~100 of 512 columns used): the stored entries
 * min(count, nbr_cap) of all rows back to back, packed on the device (exclusive scan + one warp per row) before they
 * travel.
 *   nbr_offset:  host int64[n_i + 1]   row q's entries are nbr_packed[nbr_offset[q] .. nbr_offset[q + 1]), ascending j
 *   nbr_packed:  host int32[packed_capacity]
 * If the entries do not fit packed_capacity the call returns NB_E_NOMEM after filling acc, jerk, nbr_count, n_overflow
 * and nbr_offset (nbr_offset[n_i] is the capacity to come back with); nbr_packed then holds the leading row chunks
 * that did fit.  Everything else as nb_regular_force_host. */
int nb_regular_force_host_csr(nb_ctx* ctx, int64_t n, const double* x0, const double* v0, const double* a0,
                              const double* j0, const double* m, const double* t0, int32_t n_i, const int32_t* i_idx,
                              const double* r_s, double t, double* acc, double* jerk, int32_t* nbr_count,
                              int64_t* nbr_offset, int32_t* nbr_packed, int64_t packed_capacity, int32_t* n_overflow);

/* The fp64 fix-up pass (footnote 2: "options using the 'two-float' method for the coordinates and the
 * accumulator").  The pair arithmetic of nb_regular_force[_ex] is fp32, so a row's absolute error is
 * ~ eps sqrt(sum_j |term_j|^2) whatever its sum comes to; rows whose terms cancel would miss the per-particle bound
 * (1e-6 |acc|, 1e-5 |jerk|).  The force kernel estimates that scale per row for free (squared norms of its per-tile
 * partial sums: q_a, q_j); a row with C_a sqrt(q_a) > |acc| or C_j sqrt(q_j) > |jerk| is evaluated again in fp64 by one
 * more kernel of the same call, over exactly the complement of the list the fp32 kernel emitted (its neighbour tests
 * are repeated bit for bit).  Options: "fixup" 0 | 1 (default 1); "fixup_ca_milli", "fixup_cj_milli" = 1000 C_a, 1000 C_j.
 *
 * nb_get_error_scale: test hook.  escale: dev float[n_i][2] = (q_a, q_j) of rows 0 .. n_i-1 of the last force call.
 * nb_fixup_stats: stats (HOST int64[2]) = rows the last force call recomputed in fp64, rows recomputed since nb_create.
 *                 Synchronises `stream`. */
int nb_get_error_scale(nb_ctx* ctx, int32_t n_i, float* escale, void* stream);
int nb_fixup_stats(nb_ctx* ctx, int64_t stats[2], void* stream);

/* The regular-force call (step (vi), eq. (9)-(11), after predicting all n particles to t, step (iii),
 * PAPER.md:93) for callers that MUST NOT ALLOCATE: code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc.  No context and no workspace: all scratch (packed predicted records, partial sums of j-split rows,
 * counters and queues) lives in one file-scope device array of 8 MiB inside the library, which every GPU that loads the
 * library holds until the process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating routine.
 *   LIMITS: n <= 65536, n_i <= 4096, nbr_cap <= 512 (nb_static_limits reports them: {n, n_i, nbr_cap, scratch bytes});
 *           beyond them the call returns NB_E_LIMIT and enqueues nothing -- use nb_create + nb_regular_force instead.
 *   device: CUDA device ordinal; the array of THAT device is used (set up at the first call for the device: symbol
 *           address, kernel attributes -- make that first call outside a graph capture).
 *   x0, v0, a0, j0: dev double[n][3]; m, t0: dev double[n]  (16-byte aligned), as nb_set_j
 *   i_idx, r_s, acc, jerk, nbr_count, nbr_list ([n_i][nbr_cap]), n_overflow: dev, as nb_regular_force
 * Same kernels, same arithmetic, same fp64 fix-up pass as nb_regular_force (plain criterion, rows in the order given);
 * only the launch plan may differ (fewer j-chunks fit the array), i.e. the sums agree to rounding, lists and counts
 * exactly.  ALL CALLS ON A DEVICE SHARE THE ARRAY, which keeps the last call's contents: the call clears what must start
 * at zero, on `stream`; calls that overlap on the GPU (two streams, two threads) race -- keep them on one stream. */
int nb_regular_force_static(int device, int64_t n, const double* x0, const double* v0, const double* a0,
                            const double* j0, const double* m, const double* t0, int32_t n_i, const int32_t* i_idx,
                            const double* r_s, double t, int32_t nbr_cap, double* acc, double* jerk,
                            int32_t* nbr_count, int32_t* nbr_list, int32_t* n_overflow, void* stream);
int nb_static_limits(int64_t limits[4]);

/* Tuning knobs (tests and benchmarks).  key:
 *   "j_split"   force the number of j-chunks per row for ALL row blocks (0 = automatic; 1 = never split)
 *   "i_block"   force the rows per CTA: 32, 64, 128, 256 or 512 (0 = automatic)
 *   "order_rows" 1 (default): large enough blocks are processed in Morton order of the predicted positions
 *               (results go to the caller's rows all the same); 0: always in the order given; 2: always ordered
 *   "fuse_pred" 1 (default): a regular-force call that finds no prediction at t, uses the plain criterion without
 *               potential and has at most 128 rows predicts inside the force kernel instead of running
 *               nb_predict_j first, when n >= 262144 (every j is predicted by the CTA that uses it; the context
 *               then holds no prediction at t); 0: never; 2: also for smaller n.  Results are identical bit for bit
 *   "irr_pred"  how nb_irregular_force gets its predicted particles when the context holds no prediction at t:
 *               0 (default): rows <= n / 96 predict what they gather (as nb_irregular_force_act), larger blocks
 *               predict all n first; 1: always predict all; 2: always fused.  Results are identical bit for bit
 *   "gather_copy" 0 (default): the predictor writes the particle-major copy of the records (for nb_irregular_force and
 *               nb_regular_correct) only from the first such call of the context on; 1: from the start
 *   "fixup", "fixup_ca_milli", "fixup_cj_milli": the fp64 fix-up pass, see nb_get_error_scale above
 *   "ovf_first_in_j" 0 (default): an overflowed row whose j-range was split over several CTAs keeps whichever nbr_cap
 *               neighbours reserved a list slot first (may differ from run to run); 1: one more kernel rewrites the lists
 *               of such rows as the FIRST nbr_cap neighbours in ascending j, as rows run by one CTA keep them anyway:
 *               reproducible lists, at ~n/32 warp iterations per overflowed row
 *   "pdl"       1 (default): the kernels of a call are chained by programmatic dependent launch; 0: ordinary launches
 *               (process-wide; a debugging aid)
 * Returns NB_E_INVAL for an unknown key or value. */
int nb_set_option(nb_ctx* ctx, const char* key, int64_t value);

/* What the last nb_regular_force enqueued: info[0] rows per CTA, [1] i per thread, [2] j-chunks per split row
 * block (1 = nothing split), [3] CTAs of the force kernel, [4] row blocks whose j-range was split (the "tail"
 * that fills the last wave of CTAs; all blocks for a small active block), [5] kernels
 * launched by that call (predictor included), [6] j per shared-memory tile, [7] CTAs per SM the force kernel
 * can hold. */
int nb_last_launch_info(const nb_ctx* ctx, int64_t info[8]);

/* The launch planner alone (host only, no device needed): the plan nb_regular_force would use for n
 * j-particles and n_i rows on a GPU with num_sms SMs holding ctas_per_sm[k] CTAs of shape k (rows per CTA 256,
 * 128, 64, 32, 512).  info as in nb_last_launch_info, except info[5] = j-tiles per chunk. */
int nb_plan(int64_t n, int32_t n_i, int32_t num_sms, const int32_t ctas_per_sm[5], int64_t i_block, int64_t j_split,
            int64_t info[8]);

#ifdef __cplusplus
}
#endif
#endif /* NBREG_H_ */
