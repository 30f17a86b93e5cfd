// noalloc.cu — metad_bias_noalloc: the hill sum V(s), dV/ds (a5) as ONE entry point that allocates nothing.
//
// For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it): no
// context, no cudaMalloc / cudaFree, no allocating library routine.  The caller passes the hill arrays, the CV point and the
// outputs; the per-block partial sums and the ticket of the fixed-order "last block finishes" reduction — what k_bias_sum
// (bias.cu) keeps in the context's scratch — live in a file-scope __device__ array of a fixed size.  Every GPU that loads
// this library holds those METAD_NOALLOC_SCRATCH_BYTES until the process exits.
//
// The array bounds the problem: one row of partials per block, one block per NA_CHUNK hills, so at most
// METAD_NOALLOC_MAX_HILLS hills per call.  Every call shares the array and it keeps the last call's contents: the ticket is
// cleared on the caller's stream before each launch, the partial rows a launch reads are the rows that launch wrote.  Two
// calls that overlap on the GPU (different streams, no ordering between them) race on it.
#include <mutex>
#include <stdio.h>
#include "common.cuh"

#define NA_THREADS 256
#define NA_CHUNK 2048                                   // hills per block (8 per thread)
#define NA_MAX_BLOCKS (METAD_NOALLOC_MAX_HILLS / NA_CHUNK)
#define NA_ROW (1 + METAD_MAX_CV)                       // V, dV/ds_0..3
#define NA_HEAD 256                                     // bytes in front of the partial rows: the ticket
#define NA_SCRATCH_BYTES (NA_HEAD + NA_MAX_BLOCKS * NA_ROW * 8)
static_assert(NA_SCRATCH_BYTES == METAD_NOALLOC_SCRATCH_BYTES, "include/metad.h states the size of the scratch array");
static_assert(METAD_NOALLOC_MAX_HILLS % NA_CHUNK == 0, "whole blocks");

// In host code this name is a host-side stand-in, NOT a device address: the launch below gets the address from
// cudaGetSymbolAddress (noalloc_scratch()).  Device code of this file could name it directly.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_SCRATCH_BYTES];

struct NaParams {
    int D, H, ld;
    double inv_sigma[METAD_MAX_CV];
    double period[METAD_MAX_CV];                        // 0: not periodic (reading W)
};

// restated from bias.cu (no code path of the context library is touched): s - c at the nearest periodic image
__device__ __forceinline__ double na_pdiff(double s, double c, double P) {
    double d = s - c;
    if (P > 0.0) d -= P * rint(d / P);
    return d;
}

__global__ void __launch_bounds__(NA_THREADS)
k_bias_sum_noalloc(NaParams p, const double *__restrict__ centers, const double *__restrict__ heights,
                   const double *__restrict__ cv, unsigned char *__restrict__ scratch, double *__restrict__ V,
                   double *__restrict__ dVds) {
    __shared__ double red[NA_ROW * 32];
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch);
    double *partials = reinterpret_cast<double *>(scratch + NA_HEAD);
    double s[METAD_MAX_CV];
#pragma unroll
    for (int d = 0; d < METAD_MAX_CV; ++d) s[d] = d < p.D ? cv[d] : 0.0;
    double acc[NA_ROW];
#pragma unroll
    for (int d = 0; d < NA_ROW; ++d) acc[d] = 0.0;
    const int k0 = blockIdx.x * NA_CHUNK, k1 = min(p.H, k0 + NA_CHUNK);
    for (int k = k0 + threadIdx.x; k < k1; k += NA_THREADS) {
        double e = 0.0, t[METAD_MAX_CV];
#pragma unroll
        for (int d = 0; d < METAD_MAX_CV; ++d) {
            if (d < p.D) {
                t[d] = na_pdiff(s[d], centers[(size_t)d * p.ld + k], p.period[d]) * p.inv_sigma[d];
                e += t[d] * t[d];
            }
        }
        const double g = heights[k] * exp(-0.5 * e);
        acc[0] += g;
#pragma unroll
        for (int d = 0; d < METAD_MAX_CV; ++d)
            if (d < p.D) acc[1 + d] -= g * t[d] * p.inv_sigma[d];
    }
    block_reduce<NA_ROW>(acc, red);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int d = 0; d < NA_ROW; ++d) partials[blockIdx.x * NA_ROW + d] = acc[d];
    }
    if (last_block_ticket(ticket)) {                    // fixed-order sum of the rows THIS launch wrote (0 .. gridDim.x - 1)
        double t[NA_ROW];
#pragma unroll
        for (int d = 0; d < NA_ROW; ++d) t[d] = 0.0;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) {
#pragma unroll
            for (int d = 0; d < NA_ROW; ++d) t[d] += partials[b * NA_ROW + d];
        }
        block_reduce<NA_ROW>(t, red);
        if (threadIdx.x == 0) {
            *V = t[0];
            for (int d = 0; d < p.D; ++d) dVds[d] = t[1 + d];
        }
    }
}

// Device address of the scratch array on the CURRENT device: resolved once per device, with that device current.
#define NA_MAX_DEVICES 64
static int noalloc_scratch(unsigned char **out) {
    static std::mutex mu;
    static unsigned char *addr[NA_MAX_DEVICES];         // zero-initialised: not resolved yet
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) { metad_set_error("metad_bias_noalloc: device ordinal out of range"); return METAD_ERR_ARG; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        unsigned char *p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_noalloc_scratch));
        if (!p) { metad_set_error("metad_bias_noalloc: cudaGetSymbolAddress returned a null address"); return METAD_ERR_CUDA; }
        addr[dev] = p;
    }
    *out = addr[dev];
    return METAD_OK;
}

extern "C" int metad_bias_noalloc(const double *d_centers, int ld_centers, const double *d_heights, int nhills, int ncv,
                                  const double *h_sigma, const double *h_period, const double *d_cv, double *d_V,
                                  double *d_dVds, void *cuda_stream) {
    char msg[256];
    if (!d_cv || !d_V || !d_dVds || !h_sigma) { metad_set_error("metad_bias_noalloc: null argument"); return METAD_ERR_ARG; }
    if (ncv < 1 || ncv > METAD_MAX_CV) {
        snprintf(msg, sizeof(msg), "metad_bias_noalloc: ncv = %d outside 1..%d", ncv, METAD_MAX_CV);
        metad_set_error(msg); return METAD_ERR_ARG;
    }
    if (nhills < 0 || nhills > METAD_NOALLOC_MAX_HILLS) {
        snprintf(msg, sizeof(msg), "metad_bias_noalloc: nhills = %d exceeds METAD_NOALLOC_MAX_HILLS = %d (the fixed scratch array "
                 "holds one row of partial sums per %d hills)", nhills, METAD_NOALLOC_MAX_HILLS, NA_CHUNK);
        metad_set_error(msg); return METAD_ERR_ARG;
    }
    if (nhills > 0 && (!d_centers || !d_heights || ld_centers < nhills)) {
        metad_set_error("metad_bias_noalloc: hill arrays missing or ld_centers < nhills"); return METAD_ERR_ARG;
    }
    NaParams p;
    p.D = ncv; p.H = nhills; p.ld = ld_centers;
    for (int d = 0; d < METAD_MAX_CV; ++d) {
        const double sg = d < ncv ? h_sigma[d] : 1.0;
        if (!(sg > 0.0)) { metad_set_error("metad_bias_noalloc: sigma must be positive"); return METAD_ERR_ARG; }
        p.inv_sigma[d] = 1.0 / sg;
        p.period[d] = (d < ncv && h_period) ? h_period[d] : 0.0;
        if (!(p.period[d] >= 0.0)) { metad_set_error("metad_bias_noalloc: period must be >= 0"); return METAD_ERR_ARG; }
    }
    unsigned char *scratch = nullptr;
    int r = noalloc_scratch(&scratch);
    if (r) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the ticket must start at zero whatever an earlier (possibly failed) launch left behind; a memset node, no allocation
    CUDA_TRY(cudaMemsetAsync(scratch, 0, NA_HEAD, st));
    const int nb = nhills > 0 ? (nhills + NA_CHUNK - 1) / NA_CHUNK : 1;
    k_bias_sum_noalloc<<<nb, NA_THREADS, 0, st>>>(p, d_centers, d_heights, d_cv, scratch, d_V, d_dVds);
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
