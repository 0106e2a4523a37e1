// predict.cuh -- S1, the Hermite j-predictor (step (iii) "Predict all particles"; the paper runs it
// on the host as CXVPRED, and prints no formula: BASELINE.json north_star fixes
//   x_p = x0 + v0 dt + a0 dt^2/2 + j0 dt^3/6,   v_p = v0 + a0 dt + j0 dt^2/2,   dt = t - t0[j]).
// HBM-bound: reads 112 B and writes 40 B per particle (SURVEY 8(a) S1 budgets 112 + 48).  One thread per PAIR of
// particles so that every global access is a 16-byte vector: 3 x double2 per [2][3] block of each state array,
// 5 x float4 out.  The particle-major copy for the kernels that gather single particles (irregular.cuh, corrector.cuh;
// 48 B per particle more) is written only when such a consumer exists (GATHER): the regular-force path alone never
// pays for it.
#pragma once
#include "nbreg_common.cuh"

namespace nbreg {

struct PredictArgs {
    int64_t n;        // real particles
    int64_t n_pairs;  // packed pairs to write (n_pad / 2)
    const double* x0;
    const double* v0;
    const double* a0;
    const double* j0;
    const double* m;
    const double* t0;
    double t;
    float4* packed;
    float4* gather;    // GATHER: [n][3] particle-major copy of the predicted records (nbreg_common.cuh)
    float* tile_vmax;  // [n_pad / 256] upper bound of |v_p| over each block of 256 consecutive particles
    double* xp_out;  // fp64 outputs (test hook), used only when WRITE_F64
    double* vp_out;
};

__device__ __forceinline__ void load6(const double* base, int64_t p, double (&out)[6]) {
    const double2* q = reinterpret_cast<const double2*>(base + 6 * p);
    double2 a = __ldg(q), b = __ldg(q + 1), c = __ldg(q + 2);
    out[0] = a.x; out[1] = a.y; out[2] = b.x; out[3] = b.y; out[4] = c.x; out[5] = c.y;
}

__device__ __forceinline__ void load3(const double* base, int64_t j, double (&out)[6], int off) {
    out[off + 0] = __ldg(base + 3 * j + 0);
    out[off + 1] = __ldg(base + 3 * j + 1);
    out[off + 2] = __ldg(base + 3 * j + 2);
}

// The kernel also leaves, per block of 256 consecutive particles (= kJPad, a multiple of every j-tile), an upper
// bound of the predicted speed: the velocity neighbour criterion eq. (3) needs |V_ij| bounded to
// decide that a far pair cannot come within r_s during dtr (force.cuh).
template <bool WRITE_F64, bool GATHER>
__global__ void __launch_bounds__(256) predict_kernel(PredictArgs a) {
    pdl_wait();
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = p < a.n_pairs;
    const int64_t j0 = 2 * p;
    float xh[6], xl[6], vf[6], mf[2];
#pragma unroll
    for (int k = 0; k < 6; ++k) vf[k] = 0.f;
    if (!active) {
        // nothing to predict; the thread still takes part in the speed reduction below
    } else if (j0 >= a.n) {  // padding pair: massless, far away, at rest
#pragma unroll
        for (int k = 0; k < 6; ++k) { xh[k] = kFarAway; xl[k] = 0.f; vf[k] = 0.f; }
        mf[0] = mf[1] = 0.f;
    } else {
        double x[6], v[6], acc[6], jrk[6], mm[2], tt[2];
        const bool both = (j0 + 1 < a.n);
        if (both) {
            load6(a.x0, p, x); load6(a.v0, p, v); load6(a.a0, p, acc); load6(a.j0, p, jrk);
            double2 m2 = __ldg(reinterpret_cast<const double2*>(a.m + j0));
            double2 t2 = __ldg(reinterpret_cast<const double2*>(a.t0 + j0));
            mm[0] = m2.x; mm[1] = m2.y; tt[0] = t2.x; tt[1] = t2.y;
        } else {  // odd n: last pair holds one real particle and one dummy
            load3(a.x0, j0, x, 0); load3(a.v0, j0, v, 0); load3(a.a0, j0, acc, 0); load3(a.j0, j0, jrk, 0);
            mm[0] = __ldg(a.m + j0); tt[0] = __ldg(a.t0 + j0);
#pragma unroll
            for (int k = 3; k < 6; ++k) { x[k] = (double)kFarAway; v[k] = 0.0; acc[k] = 0.0; jrk[k] = 0.0; }
            mm[1] = 0.0; tt[1] = a.t;
        }
        double xp[6], vp[6];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double dt = a.t - tt[h];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const int k = 3 * h + c;
                // Horner form of the Taylor series, fp64
                xp[k] = x[k] + dt * (v[k] + dt * (0.5 * acc[k] + dt * ((1.0 / 6.0) * jrk[k])));
                vp[k] = v[k] + dt * (acc[k] + dt * (0.5 * jrk[k]));
                xh[k] = __double2float_rn(xp[k]);
                xl[k] = __double2float_rn(xp[k] - (double)xh[k]);
                vf[k] = __double2float_rn(vp[k]);
            }
            mf[h] = __double2float_rn(mm[h]);
        }
        if (WRITE_F64) {
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                if (k < 3 || both) {
                    a.xp_out[6 * p + k] = xp[k];
                    a.vp_out[6 * p + k] = vp[k];
                }
            }
        }
    }
    if (!WRITE_F64) {
        // speed bound of this thread's pair, rounded up; max over the 128 threads (4 warps) of each 256-particle block
        __shared__ float warp_max[8];
        const float s0 = vf[0] * vf[0] + vf[1] * vf[1] + vf[2] * vf[2];
        const float s1 = vf[3] * vf[3] + vf[4] * vf[4] + vf[5] * vf[5];
        float vm = sqrtf(fmaxf(s0, s1)) * 1.000001f;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) vm = fmaxf(vm, __shfl_xor_sync(0xffffffffu, vm, off));
        if ((threadIdx.x & 31) == 0) warp_max[threadIdx.x >> 5] = vm;
        __syncthreads();
        if ((threadIdx.x & 127) == 0 && active) {
            const int w = threadIdx.x >> 5;
            a.tile_vmax[p >> 7] = fmaxf(fmaxf(warp_max[w], warp_max[w + 1]), fmaxf(warp_max[w + 2], warp_max[w + 3]));
        }
    }
    if (!WRITE_F64 && active) {
        float4* o = a.packed + kQuadsPerPair * p;
        o[0] = make_float4(xh[0], xh[3], xh[1], xh[4]);
        o[1] = make_float4(xh[2], xh[5], mf[0], mf[1]);
        o[2] = make_float4(vf[0], vf[3], vf[1], vf[4]);
        o[3] = make_float4(vf[2], vf[5], xl[0], xl[3]);
        o[4] = make_float4(xl[1], xl[4], xl[2], xl[5]);
        if (GATHER && j0 < a.n) {  // particle-major copy: the pair's two records are contiguous (96 B)
            float4* g = a.gather + kGatherQuads * j0;
            g[0] = make_float4(xh[0], xh[1], xh[2], mf[0]);
            g[1] = make_float4(xl[0], xl[1], xl[2], vf[0]);
            g[2] = make_float4(vf[1], vf[2], 0.f, 0.f);
            if (j0 + 1 < a.n) {
                g[3] = make_float4(xh[3], xh[4], xh[5], mf[1]);
                g[4] = make_float4(xl[3], xl[4], xl[5], vf[3]);
                g[5] = make_float4(vf[4], vf[5], 0.f, 0.f);
            }
        }
    }
}

}  // namespace nbreg
