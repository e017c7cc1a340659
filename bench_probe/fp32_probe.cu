// fp32_probe.cu -- FP32 FMA-pipe probe for the roofline denominator: a bench-side helper (beside bench.py) built into its own
// library (libfp32probe.so), NOT part of liblinmin.so or of include/linmin.h.
// MEASURED_PEAKS.json carries HBM and bf16 tensor figures only; the path here is bound by plain FP32
// arithmetic, so bench.py measures what the FMA pipe sustains: every thread runs
// independent dependent-free FMA chains from registers, as scalar FFMA and as packed FFMA2.
#include <cuda_runtime.h>

namespace {

template <bool PACKED>
__global__ void __launch_bounds__(256) fp32_probe_kernel(float *sink, int iters, float seed) {
    // 16 independent accumulator pairs per thread: enough to cover the FMA latency at 8 warps per scheduler
    float2 acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = make_float2(seed + (float)i, seed - (float)i);
    const float2 m = make_float2(1.0f + 1e-7f * seed, 1.0f - 1e-7f * seed), c = make_float2(1e-9f, -1e-9f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            if (PACKED) {
                unsigned long long d, a, b, e;
                asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(acc[i].x), "f"(acc[i].y));
                asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(m.x), "f"(m.y));
                asm("mov.b64 %0, {%1, %2};" : "=l"(e) : "f"(c.x), "f"(c.y));
                asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(e));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(acc[i].x), "=f"(acc[i].y) : "l"(d));
            } else {
                acc[i].x = fmaf(acc[i].x, m.x, c.x);
                acc[i].y = fmaf(acc[i].y, m.y, c.y);
            }
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += acc[i].x + acc[i].y;
    if (s == 123.456f) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true: keeps the chains alive
}

// Returns TFLOP/s (2 flops per FMA) of scalar FFMA and of packed FFMA2 streams on the device of `stream`.
cudaError_t probe_fp32(int sm_count, cudaStream_t stream, double *ffma_tflops, double *ffma2_tflops) {
    float *sink = nullptr;
    cudaError_t e = cudaMalloc((void **)&sink, sizeof(float) * 256);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sm_count * 8, block = 256, iters = 4096;
    double out[2] = {0.0, 0.0};
    for (int packed = 0; packed < 2; ++packed) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(e0, stream);
            if (packed) fp32_probe_kernel<true><<<grid, block, 0, stream>>>(sink, iters, 0.5f);
            else fp32_probe_kernel<false><<<grid, block, 0, stream>>>(sink, iters, 0.5f);
            cudaEventRecord(e1, stream);
            e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) break;
            float ms = 0.0f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        const double flops = 2.0 * 32.0 * (double)iters * (double)grid * (double)block;
        out[packed] = flops / ((double)best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    if (e == cudaSuccess) e = cudaGetLastError();
    *ffma_tflops = out[0]; *ffma2_tflops = out[1];
    return e;
}

}  // namespace

// host pointers; synchronous; a few milliseconds of work on `stream` (a cudaStream_t, NULL = default stream).
// Returns 0 or a cudaError_t.
extern "C" int fp32_probe_peak(void *stream, double *ffma_tflops, double *ffma2_tflops) {
    if (!ffma_tflops || !ffma2_tflops) return (int)cudaErrorInvalidValue;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = probe_fp32(sms, (cudaStream_t)stream, ffma_tflops, ffma2_tflops);
    return (int)e;
}
