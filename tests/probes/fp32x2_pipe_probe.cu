// fp32x2_pipe_probe.cu -- what the B200 FP32 pipe sustains for the packed instructions force_kernel is made of.
//
// TEST INFRASTRUCTURE (built and run by tests/test_gpu_pipe_probe.py; not part of the library).
// bounds force_kernel by the FP32 pipe: 25 packed f32x2 instructions per two pairs, nominal 128 lanes per clock per SM.
// This probe measures, with the kernel's own occupancy (32 warps per SM, one wave), how many lane-operations per clock
// per SM a stream of independent packed instructions really retires:
//   ffma2_3reg   d = a * b + d, a, b, d distinct 64-bit registers per chain (the shape of the kernel's sums)
//   ffma2_shared d = a * b + d with a and b common to all chains (operand reuse possible)
//   fadd2, fmul2 two-operand packed instructions
//   mix          the kernel's own proportion: 9 FADD2 : 5 FMUL2 : 11 FFMA2 ... per 25, independent chains
//   mix_mufu     the same plus 4 MUFU (2 rsqrt, 2 rcp) per 25, as in the kernel's common path
//   ffma_scalar  the unpacked FFMA for reference
// Output: one JSON object on stdout: lanes per clock per SM for each stream (nominal 128).
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>

constexpr int kChains = 8;
constexpr int kIters = 1 << 13;
constexpr int kThreads = 128;
constexpr int kCtasPerSm = 8;

__device__ __forceinline__ float rsq(float x) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp(float x) { float y; asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

template <int MODE>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) probe(float* out, long long* cycles, float seed) {
    float2 d[kChains], a[kChains], b[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        d[k] = make_float2(seed + k, seed - k);
        a[k] = make_float2(1.0f + 1e-7f * (threadIdx.x + k), 1.0f - 1e-7f * k);
        b[k] = make_float2(1e-9f * (k + 1), -1e-9f * (k + 2));
    }
    const float2 sa = a[0], sb = b[0];
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
        if (MODE == 0) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) d[k] = __ffma2_rn(a[k], b[k], d[k]);
        } else if (MODE == 1) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) d[k] = __ffma2_rn(sa, sb, d[k]);
        } else if (MODE == 2) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) d[k] = __fadd2_rn(d[k], b[k]);
        } else if (MODE == 3) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) d[k] = __fmul2_rn(d[k], a[k]);
        } else if (MODE == 4 || MODE == 5) {
            // 25 packed instructions: 9 FADD2, 5 FMUL2, 11 FFMA2 (force_kernel's common path), on 8 independent chains
#pragma unroll
            for (int k = 0; k < 8; ++k) d[k] = __fadd2_rn(d[k], b[k]);
            d[0] = __fadd2_rn(d[0], b[1]);
#pragma unroll
            for (int k = 0; k < 5; ++k) d[k] = __fmul2_rn(d[k], a[k]);
#pragma unroll
            for (int k = 0; k < 8; ++k) d[k] = __ffma2_rn(a[k], b[k], d[k]);
#pragma unroll
            for (int k = 0; k < 3; ++k) d[k] = __ffma2_rn(a[k + 1], b[k + 2], d[k]);
            if (MODE == 5) {  // 4 MUFU per 25, results folded back so they are not dead
                a[6].x = rsq(a[6].x); a[6].y = rsq(a[6].y);
                a[7].x = rcp(a[7].x); a[7].y = rcp(a[7].y);
            }
        } else {
#pragma unroll
            for (int k = 0; k < kChains; ++k) {
                d[k].x = fmaf(a[k].x, b[k].x, d[k].x);
                d[k].y = fmaf(a[k].y, b[k].y, d[k].y);
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += d[k].x + d[k].y + a[k].x;
    out[blockIdx.x * kThreads + threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int MODE>
double run(int sms, double lane_ops_per_thread_iter, float* out, long long* cyc, long long* h) {
    const int grid = sms * kCtasPerSm;
    probe<MODE><<<grid, kThreads>>>(out, cyc, 1.0f);  // warm-up
    probe<MODE><<<grid, kThreads>>>(out, cyc, 1.0f);
    cudaMemcpy(h, cyc, grid * sizeof(long long), cudaMemcpyDeviceToHost);
    double mean = 0;
    for (int i = 0; i < grid; ++i) mean += (double)h[i];
    mean /= grid;
    // lane-operations one SM retires: CTAs per SM x threads x iterations x lane-ops per thread-iteration
    return (double)kCtasPerSm * kThreads * kIters * lane_ops_per_thread_iter / mean;
}

int main() {
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    const int grid = sms * kCtasPerSm;
    float* out;
    long long *cyc, *h = (long long*)malloc(grid * sizeof(long long));
    cudaMalloc(&out, (size_t)grid * kThreads * sizeof(float));
    cudaMalloc(&cyc, grid * sizeof(long long));
    // a packed instruction is 2 lane-operations per thread
    const double r0 = run<0>(sms, 2.0 * kChains, out, cyc, h);
    const double r1 = run<1>(sms, 2.0 * kChains, out, cyc, h);
    const double r2 = run<2>(sms, 2.0 * kChains, out, cyc, h);
    const double r3 = run<3>(sms, 2.0 * kChains, out, cyc, h);
    const double r4 = run<4>(sms, 2.0 * 25, out, cyc, h);
    const double r5 = run<5>(sms, 2.0 * 25, out, cyc, h);
    const double r6 = run<6>(sms, 2.0 * kChains, out, cyc, h);
    if (cudaDeviceSynchronize() != cudaSuccess) return 1;
    printf("{\"sms\": %d, \"warps_per_sm\": %d, \"nominal_lanes_per_clk_per_sm\": 128, \"ffma2_3reg\": %.2f, "
           "\"ffma2_shared\": %.2f, \"fadd2\": %.2f, \"fmul2\": %.2f, \"mix\": %.2f, \"mix_mufu\": %.2f, "
           "\"ffma_scalar\": %.2f}\n",
           sms, kCtasPerSm * kThreads / 32, r0, r1, r2, r3, r4, r5, r6);
    return 0;
}
