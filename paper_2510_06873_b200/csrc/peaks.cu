// peaks.cu — scalar-pipe roofline denominators ("both to be re-measured by an FMA microbenchmark because
// MEASURED_PEAKS has no scalar-pipe entry").  Dependent-free FMA chains on every SM, timed with CUDA events:
//   kind 0  fp32  FFMA        (2 flop per lane-instruction)
//   kind 1  fp32  FFMA2       (fma.rn.f32x2: 4 flop per lane-instruction, sm_100)
//   kind 2  fp64  DFMA
// bench.py --peaks calls metad_fma_peak and uses the measured numbers as the "alu" roofline peaks.
#include <stdio.h>
#include "common.cuh"

#define PK_CHAINS 8
#define PK_THREADS 256

__global__ void __launch_bounds__(PK_THREADS)
k_peak_f32(int iters, float a, float b, float *out) {
    float x[PK_CHAINS];
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) x[k] = (float)(threadIdx.x + k) * 1e-3f;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < PK_CHAINS; ++k) x[k] = fmaf(x[k], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) s += x[k];
    if (s == 123.456f) out[0] = s;                  // never true: keeps the chains alive
}

__global__ void __launch_bounds__(PK_THREADS)
k_peak_f32x2(int iters, float a, float b, float *out) {
    unsigned long long x[PK_CHAINS], aa, bb;
    asm("mov.b64 %0, {%1,%1};" : "=l"(aa) : "f"(a));
    asm("mov.b64 %0, {%1,%1};" : "=l"(bb) : "f"(b));
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) {
        const float v = (float)(threadIdx.x + k) * 1e-3f;
        asm("mov.b64 %0, {%1,%2};" : "=l"(x[k]) : "f"(v), "f"(-v));
    }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < PK_CHAINS; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[k]) : "l"(aa), "l"(bb));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) { float lo, hi; asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x[k])); s += lo + hi; }
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(PK_THREADS)
k_peak_f64(int iters, double a, double b, double *out) {
    double x[PK_CHAINS];
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) x[k] = (double)(threadIdx.x + k) * 1e-3;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int k = 0; k < PK_CHAINS; ++k) x[k] = fma(x[k], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; ++k) s += x[k];
    if (s == 123.456) out[0] = s;
}

extern "C" int metad_fma_peak(int kind, double *h_tflops, double *h_ms) {
    if (kind < 0 || kind > 2 || !h_tflops) { metad_set_error("kind must be 0 (fp32), 1 (fp32x2) or 2 (fp64)"); return METAD_ERR_ARG; }
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    void *d_out = nullptr;
    CUDA_TRY(cudaMalloc(&d_out, 64));
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    const int blocks = sms * 8;                     // 2,048 threads per SM: every scheduler has 16 warps to pick from
    const int iters = kind == 2 ? 2048 : 16384;     // ~1-2 ms per launch
    double best = 0.0, best_ms = 0.0;
    for (int rep = 0; rep < 6; ++rep) {             // first repetitions warm the clocks up; best of the rest
        cudaEventRecord(e0, 0);
        if (kind == 0) k_peak_f32<<<blocks, PK_THREADS>>>(iters, 0.999f, 1e-3f, (float *)d_out);
        else if (kind == 1) k_peak_f32x2<<<blocks, PK_THREADS>>>(iters, 0.999f, 1e-3f, (float *)d_out);
        else k_peak_f64<<<blocks, PK_THREADS>>>(iters, 0.999, 1e-3, (double *)d_out);
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaFree(d_out); CUDA_TRY(e); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fl = (double)blocks * PK_THREADS * (double)iters * 8.0 * PK_CHAINS * (kind == 1 ? 4.0 : 2.0);
        const double tf = fl / (ms * 1e-3) / 1e12;
        if (rep >= 2 && tf > best) { best = tf; best_ms = ms; }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    *h_tflops = best;
    if (h_ms) *h_ms = best_ms;
    return METAD_OK;
}
