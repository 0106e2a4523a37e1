// record.cuh -- one particle's predicted record, fetched from the particle-major copy the predictor wrote
// (load_record) or predicted on the spot from the registered fp64 state (predict_record): used by the kernels that
// gather particles by index (irregular.cuh, corrector.cuh) and by the force kernel's fused-prediction variant.
#pragma once
#include "nbreg_common.cuh"

namespace nbreg {

// The registered fp64 state (nb_set_j) and the time to predict to: what the fused-prediction variant gathers from.
struct RawState {
    const double *x0, *v0, *a0, *j0, *m, *t0;
    double t;
};

struct PredRecord {  // one particle's share of a packed pair record
    float xh, yh, zh, m, xl, yl, zl, vx, vy, vz;
};

// Gather one particle: three 16-byte loads from its 48-byte particle-major record (two sectors).  This kernel sits on
// the L1/TEX sector rate for scattered accesses (profiles/r1_irregular_kernel_ncu_full.md), so what counts is
// the number of sector accesses per gathered particle: 3 here, 5 from the pair-interleaved records of the
// regular-force kernel, 10 with scalar loads.
__device__ __forceinline__ PredRecord load_record(const float4* gather, int32_t j) {
    const float4* rec = gather + (size_t)j * kGatherQuads;
    const float4 g0 = __ldg(rec), g1 = __ldg(rec + 1), g2 = __ldg(rec + 2);
    PredRecord r;
    r.xh = g0.x; r.yh = g0.y; r.zh = g0.z; r.m = g0.w;
    r.xl = g1.x; r.yl = g1.y; r.zl = g1.z; r.vx = g1.w;
    r.vy = g2.x; r.vz = g2.y;
    return r;
}

// The paper's PRED_ACT mode ("When N_act,I is small, predicting all the N particles is not efficient.
// Thus ... we switch to predict only the necessary particles in this block-step"): gather a particle's fp64 state
// (14 scalar loads, 112 B) and predict it on the spot -- the Horner form, the two-float split and the roundings of
// predict.cuh, so that both modes feed the pair arithmetic the same record.  No prediction pass, no dependence on
// the context's predicted records: one launch for a small irregular block.
__device__ __forceinline__ PredRecord predict_record(const RawState& s, int32_t j) {
    const double dt = s.t - __ldg(s.t0 + j);
    float h[3], l[3], w[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double x = __ldg(s.x0 + 3 * (size_t)j + c), v = __ldg(s.v0 + 3 * (size_t)j + c);
        const double acc = __ldg(s.a0 + 3 * (size_t)j + c), jrk = __ldg(s.j0 + 3 * (size_t)j + c);
        const double xp = x + dt * (v + dt * (0.5 * acc + dt * ((1.0 / 6.0) * jrk)));
        const double vp = v + dt * (acc + dt * (0.5 * jrk));
        h[c] = __double2float_rn(xp);
        l[c] = __double2float_rn(xp - (double)h[c]);
        w[c] = __double2float_rn(vp);
    }
    PredRecord r;
    r.xh = h[0]; r.yh = h[1]; r.zh = h[2]; r.m = __double2float_rn(__ldg(s.m + j));
    r.xl = l[0]; r.yl = l[1]; r.zl = l[2]; r.vx = w[0]; r.vy = w[1]; r.vz = w[2];
    return r;
}

}  // namespace nbreg
