// sph_probe.cu -- FP32 FMA issue-rate probe: the measured counterpart of the derived ALU roofline
// denominator.  Measurement support only; no step of the path runs here.
#include "sph_internal.cuh"

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

extern "C" int sph_fp32_peak(sph_ctx *ctx, int iters, int packed, double *tflops_host)
{
    if (!ctx || !tflops_host || iters < 1) return SPH_E_ARG;
    cudaStream_t st = ctx->stream;
    float *dummy = reinterpret_cast<float *>(ctx->cnt); // never written (see the kernels)
    const int blocks = ctx->device_sms * 8, threads = 256;
    cudaEvent_t e0, e1;
    SPH_CUDA(ctx, cudaEventCreate(&e0));
    SPH_CUDA(ctx, cudaEventCreate(&e1));
    for (int rep = 0; rep < 2; rep++) { // first launch warms up
        SPH_CUDA(ctx, cudaEventRecord(e0, st));
        if (packed) k_probe_packed<<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, dummy);
        else k_probe_scalar<<<blocks, threads, 0, st>>>(iters, 0.999f, 0.001f, dummy);
        SPH_CUDA(ctx, cudaEventRecord(e1, st));
        SPH_CUDA(ctx, cudaStreamSynchronize(st));
    }
    SPH_CUDA(ctx, cudaGetLastError());
    float ms = 0.f;
    SPH_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    double fmas = (double)blocks * threads * (double)iters * PROBE_INNER * PROBE_ACC;
    *tflops_host = 2.0 * fmas / ((double)ms * 1e-3) * 1e-12;
    ctx->launches += 2;
    return SPH_OK;
}
