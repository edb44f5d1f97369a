// bench_probe.cu -- FP32 FMA issue-rate probe of bench.py: the measured denominator of the ALU roofline
// ("measured on the box in the same session").  Bench harness only: it is
// built into bench_probe.so beside bench.py, not into libsph.so, and no step of the path runs here.
#include <cuda_runtime.h>

namespace {

#define PROBE_ACC 16    // independent accumulators per thread (ILP covers the 4-cycle FMA latency)
#define PROBE_INNER 256 // FMAs per accumulator per outer iteration

__global__ void __launch_bounds__(256) k_probe_scalar(int iters, float a, float b, float *out)
{
    float acc[PROBE_ACC];
#pragma unroll
    for (int i = 0; i < PROBE_ACC; i++) acc[i] = (float)(threadIdx.x + i);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int k = 0; k < PROBE_INNER; k++) {
#pragma unroll
            for (int i = 0; i < PROBE_ACC; i++) acc[i] = fmaf(acc[i], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PROBE_ACC; i++) s += acc[i];
    if (s == 12345.678f) out[0] = s; // keeps the chain live, practically never taken
}

__global__ void __launch_bounds__(256) k_probe_packed(int iters, float a, float b, float *out)
{
    unsigned long long acc[PROBE_ACC / 2], pa, pb;
    asm("mov.b64 %0, {%1, %1};" : "=l"(pa) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(pb) : "f"(b));
#pragma unroll
    for (int i = 0; i < PROBE_ACC / 2; i++) {
        float x = (float)(threadIdx.x + i);
        asm("mov.b64 %0, {%1, %1};" : "=l"(acc[i]) : "f"(x));
    }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int k = 0; k < PROBE_INNER; k++) {
#pragma unroll
            for (int i = 0; i < PROBE_ACC / 2; i++)
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(acc[i]) : "l"(pa), "l"(pb));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PROBE_ACC / 2; i++) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(acc[i]));
        s += lo + hi;
    }
    if (s == 12345.678f) out[0] = s;
}

} // namespace

// Runs a register-only chain of fused multiply-adds on every SM (about iters x 4096 FMAs per thread) on the given
// stream and returns the achieved rate in TFLOP/s (2 flop per FMA) in *tflops_host; packed != 0 uses the two-wide
// fma.rn.f32x2 form of sm_100.  Returns 0, or a cudaError_t value.  Synchronises the stream.
extern "C" int bench_fp32_peak(void *cuda_stream, int iters, int packed, double *tflops_host)
{
    if (!tflops_host || iters < 1) return (int)cudaErrorInvalidValue;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return (int)e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return (int)e;
    float *dummy = nullptr; // never written (see the kernels)
    if ((e = cudaMalloc((void **)&dummy, 256)) != cudaSuccess) return (int)e;
    const int blocks = sms * 8, threads = 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int rep = 0; rep < 2; rep++) { // first launch warms up
        cudaEventRecord(e0, st);
        if (packed) k_probe_packed<<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, dummy);
        else k_probe_scalar<<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, dummy);
        cudaEventRecord(e1, st);
        cudaStreamSynchronize(st);
    }
    float ms = 0.f;
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(dummy);
    if (e != cudaSuccess) return (int)e;
    const double fmas = (double)blocks * threads * (double)iters * PROBE_INNER * PROBE_ACC;
    *tflops_host = 2.0 * fmas / ((double)ms * 1e-3) * 1e-12;
    return 0;
}
