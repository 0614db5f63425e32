// gsvox_probe.cu — live measurement of the ALU rooflines the hot path is bound by (SURVEY.md
// 8(d): "measure both with an FMA-chain and an ex2-chain microbenchmark in the same run").
// Three register-only kernels, each thread running kChains independent dependency chains:
//   FFMA   scalar fp32 fused multiply-add            (2 flops / lane-instruction)
//   FFMA2  packed fma.rn.f32x2 (sm_100 family)       (4 flops / lane-instruction)
//   EX2    MUFU ex2.approx.ftz.f32                    (1 result / lane-instruction)
// Grid = SM count x 8 CTAs of 256 threads; timed with CUDA events on the caller's stream.
// Bench-only: built into libgsvox_probe.so (include/gsvox_probe.h), not into the product library.
#include "gsvox_internal.cuh"
#include "../../include/gsvox_probe.h"
#undef GSVOX_CUDA
#define GSVOX_CUDA(call) do { if ((call) != cudaSuccess) { (void)cudaGetLastError(); return GSVOX_ECUDA; } } while (0)

namespace gsvox {

constexpr int kProbeThreads = 256;
constexpr int kChains = 8;
constexpr int kProbeIters = 4096;

__global__ void __launch_bounds__(kProbeThreads) k_probe_ffma(float* sink, float a, float b)
{
    float v[kChains];
    #pragma unroll
    for (int c = 0; c < kChains; ++c) v[c] = (float)(threadIdx.x + c);
    for (int i = 0; i < kProbeIters; ++i) {
        #pragma unroll
        for (int c = 0; c < kChains; ++c) v[c] = fmaf(v[c], a, b);
    }
    float s = 0.f;
    #pragma unroll
    for (int c = 0; c < kChains; ++c) s += v[c];
    if (s == 123.456f) sink[0] = s;          // never true for the arguments used; keeps the chains alive
}

__global__ void __launch_bounds__(kProbeThreads) k_probe_ffma2(float* sink, float a, float b)
{
    unsigned long long v[kChains], pa, pb;
    asm("mov.b64 %0, {%1, %1};" : "=l"(pa) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(pb) : "f"(b));
    #pragma unroll
    for (int c = 0; c < kChains; ++c) {
        float lo = (float)(threadIdx.x + c), hi = lo + 0.5f;
        asm("mov.b64 %0, {%1, %2};" : "=l"(v[c]) : "f"(lo), "f"(hi));
    }
    for (int i = 0; i < kProbeIters; ++i) {
        #pragma unroll
        for (int c = 0; c < kChains; ++c)
            asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v[c]) : "l"(pa), "l"(pb));
    }
    float s = 0.f;
    #pragma unroll
    for (int c = 0; c < kChains; ++c) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v[c]));
        s += lo + hi;
    }
    if (s == 123.456f) sink[0] = s;
}

__global__ void __launch_bounds__(kProbeThreads) k_probe_ex2(float* sink, float a)
{
    float v[kChains];
    #pragma unroll
    for (int c = 0; c < kChains; ++c) v[c] = a * (float)(threadIdx.x + c);
    for (int i = 0; i < kProbeIters; ++i) {
        #pragma unroll
        for (int c = 0; c < kChains; ++c) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(v[c]));
    }
    float s = 0.f;
    #pragma unroll
    for (int c = 0; c < kChains; ++c) s += v[c];
    if (s == 123.456f) sink[0] = s;
}

}  // namespace gsvox

using namespace gsvox;

extern "C" int gsvox_probe_peaks(void* scratch, double* fp32_tflops, double* fp32x2_tflops,
                                 double* ex2_tera_per_s, int32_t* sm_count, void* stream)
{
    if (!scratch) return GSVOX_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    GSVOX_CUDA(cudaGetDevice(&dev));
    GSVOX_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = sms * 8;
    cudaEvent_t e0, e1;
    GSVOX_CUDA(cudaEventCreate(&e0));
    GSVOX_CUDA(cudaEventCreate(&e1));
    float* sink = (float*)scratch;
    const double lane_inst = (double)grid * kProbeThreads * kChains * (double)kProbeIters;
    double best[3] = { 0.0, 0.0, 0.0 };
    for (int kind = 0; kind < 3; ++kind) {
        for (int rep = 0; rep < 6; ++rep) {                    // first rep warms up; best of the rest
            cudaEventRecord(e0, st);
            if (kind == 0)      k_probe_ffma<<<grid, kProbeThreads, 0, st>>>(sink, 0.999f, 0.001f);
            else if (kind == 1) k_probe_ffma2<<<grid, kProbeThreads, 0, st>>>(sink, 0.999f, 0.001f);
            else                k_probe_ex2<<<grid, kProbeThreads, 0, st>>>(sink, -0.001f);
            cudaEventRecord(e1, st);
            cudaError_t e = cudaEventSynchronize(e1);
            if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); (void)cudaGetLastError(); return GSVOX_ECUDA; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            const double per_s = lane_inst / (ms * 1e-3);
            if (rep > 0 && per_s > best[kind]) best[kind] = per_s;
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    GSVOX_CUDA(cudaGetLastError());
    if (fp32_tflops)    *fp32_tflops = 2.0 * best[0] / 1e12;
    if (fp32x2_tflops)  *fp32x2_tflops = 4.0 * best[1] / 1e12;
    if (ex2_tera_per_s) *ex2_tera_per_s = best[2] / 1e12;
    if (sm_count)       *sm_count = sms;
    return GSVOX_OK;
}
