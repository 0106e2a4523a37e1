// fp32x2_pipe_probe.cu -- what the B200 FP32 pipes sustain for the packed instructions force_kernel is made of.
//
// TEST INFRASTRUCTURE (built and run by tests/test_gpu_pipe_probe.py; not part of the library).
// bounds force_kernel by the FP32 pipe: 25 packed f32x2 instructions per two pairs (6 FADD2, 6 FMUL2, 13 FFMA2 in the
// SASS of the common path) plus 4 MUFU.  This probe measures, with the kernel's own occupancy (32 warps per SM, one wave of CTAs), how many
// lane-operations per clock per SM streams of independent packed instructions really retire, alone and mixed:
// probe<A, M, F, U> issues per loop iteration A FADD2, M FMUL2, F FFMA2 and U pairs of MUFU (rsqrt + rcp) on 8
// independent chains per thread (the loop is unrolled so that loop overhead is < 4 % of the issue slots).
// "ffma2_3reg": multiplicands distinct per chain (three distinct 64-bit register operands, the shape of the kernel's
// sums); "ffma2_shared": multiplicands common to all chains.
// Output: one JSON object on stdout, lanes per clock per SM for each stream (one packed instruction = 2 lane-ops per
// thread; nominal FP32 rate 128 lanes per clock per SM).
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>

constexpr int kChains = 8;
constexpr int kIters = 1 << 11;
constexpr int kThreads = 128;
constexpr int kCtasPerSm = 8;

__device__ __forceinline__ float rsq(float x) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp(float x) { float y; asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// A, M, F: FADD2, FMUL2, FFMA2 per round over the 8 chains; R rounds per loop iteration; U: MUFU pairs per round;
// SHARED: common multiplicands; SCALAR: unpacked instructions instead
template <int A, int M, int F, int U, int R, bool SHARED, bool SCALAR>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) probe(float* out, long long* cycles, float seed) {
    float2 d[kChains], a[kChains], b[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        d[k] = make_float2(seed + k, seed - k);
        a[k] = make_float2(1.0f + 1e-7f * (threadIdx.x + k), 1.0f - 1e-7f * k);
        b[k] = make_float2(1e-9f * (k + 1), -1e-9f * (k + 2));
    }
    const float2 sa = a[0], sb = b[0];
    float mu = 1.0f + 1e-3f * threadIdx.x, mv = 2.0f;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
#pragma unroll
            for (int k = 0; k < A; ++k) {
                const int c = k & 7;
                if (SCALAR) { d[c].x = __fadd_rn(d[c].x, b[c].x); d[c].y = __fadd_rn(d[c].y, b[c].y); }
                else d[c] = __fadd2_rn(d[c], b[c]);
            }
#pragma unroll
            for (int k = 0; k < M; ++k) {
                const int c = (k + 3) & 7;
                if (SCALAR) { d[c].x = __fmul_rn(d[c].x, a[k & 7].x); d[c].y = __fmul_rn(d[c].y, a[k & 7].y); }
                else d[c] = __fmul2_rn(d[c], a[k & 7]);
            }
#pragma unroll
            for (int k = 0; k < F; ++k) {
                const int c = (k + 5) & 7, e = k & 7;
                if (SCALAR) { d[c].x = __fmaf_rn(a[e].x, b[e].x, d[c].x); d[c].y = __fmaf_rn(a[e].y, b[e].y, d[c].y); }
                else d[c] = SHARED ? __ffma2_rn(sa, sb, d[c]) : __ffma2_rn(a[e], b[e], d[c]);
            }
#pragma unroll
            for (int k = 0; k < U; ++k) { mu = rsq(mu); mv = rcp(mv); }
        }
    }
    const long long t1 = clock64();
    float s = mu + mv;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += d[k].x + d[k].y + a[k].x;
    out[blockIdx.x * kThreads + threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

static int g_sms;
static float* g_out;
static long long* g_cyc;

// SM clock during the run: clock64 ticks per second of globaltimer, measured by one spinning thread
__global__ void clock_rate_kernel(double* hz) {
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long c0 = clock64();
    do {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    } while (g1 - g0 < 2000000ull);  // 2 ms
    const long long c1 = clock64();
    *hz = (double)(c1 - c0) / ((double)(g1 - g0) * 1e-9);
}

static double g_hz;

// lanes per clock per SM = FP32 lane-operations of the whole launch / (kernel time x SM clock x SMs); the time is taken
// with CUDA events around the second of two launches (every CTA of the grid is resident at once: one wave)
template <int A, int M, int F, int U, int R, bool SHARED, bool SCALAR>
double run() {
    const int grid = g_sms * kCtasPerSm;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    probe<A, M, F, U, R, SHARED, SCALAR><<<grid, kThreads>>>(g_out, g_cyc, 1.0f);  // warm-up
    cudaEventRecord(e0);
    probe<A, M, F, U, R, SHARED, SCALAR><<<grid, kThreads>>>(g_out, g_cyc, 1.0f);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double lane_ops = (double)grid * kThreads * kIters * 2.0 * (A + M + F) * R;
    return lane_ops / (ms * 1e-3 * g_hz * g_sms);
}

int main() {
    cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, 0);
    const int grid = g_sms * kCtasPerSm;
    cudaMalloc(&g_out, (size_t)grid * kThreads * sizeof(float));
    cudaMalloc(&g_cyc, grid * sizeof(long long));
    double* d_hz;
    cudaMalloc(&d_hz, sizeof(double));
    clock_rate_kernel<<<1, 1>>>(d_hz);
    cudaMemcpy(&g_hz, d_hz, sizeof(double), cudaMemcpyDeviceToHost);
    printf("{\"sms\": %d, \"warps_per_sm\": %d, \"sm_clock_mhz\": %.0f, \"nominal_lanes_per_clk_per_sm\": 128", g_sms,
           kCtasPerSm * kThreads / 32, g_hz * 1e-6);
    printf(", \"ffma2_3reg\": %.2f", run<0, 0, 8, 0, 8, false, false>());
    printf(", \"ffma2_shared\": %.2f", run<0, 0, 8, 0, 8, true, false>());
    printf(", \"fadd2\": %.2f", run<8, 0, 0, 0, 8, false, false>());
    printf(", \"fmul2\": %.2f", run<0, 8, 0, 0, 8, false, false>());
    printf(", \"fadd2_ffma2_1to1\": %.2f", run<4, 0, 4, 0, 8, true, false>());
    printf(", \"mix_6_6_13\": %.2f", run<6, 6, 13, 0, 3, false, false>());
    printf(", \"mix_6_6_13_shared\": %.2f", run<6, 6, 13, 0, 3, true, false>());
    printf(", \"mix_6_6_13_mufu4\": %.2f", run<6, 6, 13, 2, 3, false, false>());
    printf(", \"mix_6_6_13_shared_mufu4\": %.2f", run<6, 6, 13, 2, 3, true, false>());
    printf(", \"ffma_scalar\": %.2f", run<0, 0, 8, 0, 8, false, true>());
    printf(", \"fadd_scalar\": %.2f", run<8, 0, 0, 0, 8, false, true>());
    printf(", \"mix_6_6_13_scalar\": %.2f", run<6, 6, 13, 0, 3, false, true>());
    printf("}\n");
    return cudaDeviceSynchronize() == cudaSuccess ? 0 : 1;
}
