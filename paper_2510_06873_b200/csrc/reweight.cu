// reweight.cu — NEXT-2: batched bias evaluation and free-energy reconstruction by reweighting
// (PAPER.md:85-87):  P(s) = < delta[s - s(R)] e^{beta V_b} > / < e^{beta V_b} >,  F = -(1/beta) log P,
// averages over the frames of the biased trajectory (reading Z: delta = uniform bins).
//   k_bias_batch      V_b at T points: thread per point, the hill array streamed through shared memory
//                     in tiles (the FP64 exp is the work: T x H evaluations, pure ALU, no HBM re-reads)
//   k_vmax            max of V over the frames (order-independent)
//   k_reweight_hist   w = e^{(V - Vmax)/kT} as 2^-40 fixed point, integer atomics into the bins: the
//                     sums do not depend on the order of the atomics => run-to-run bit-identical
//   k_reweight_finish P = bin / (total x bin volume), F = -kT log P (+inf for empty bins)
#include <math.h>
#include <string.h>
#include <algorithm>
#include "common.cuh"

#define RW_THREADS 256
#define RW_TILE 512

struct RwBias { int D, H, max_hills; double inv_sigma[METAD_MAX_CV], period[METAD_MAX_CV], inv_period[METAD_MAX_CV]; };
struct RwBins { int D, nb[2]; double lo[2], hi[2], h[2], period[2], vol; };

__global__ void __launch_bounds__(RW_THREADS)
k_bias_batch(RwBias bp, const double *__restrict__ centers, const double *__restrict__ heights,
             const int *__restrict__ nhills, const double *__restrict__ points, int T, double *__restrict__ V) {
    __shared__ double sc[METAD_MAX_CV][RW_TILE];
    __shared__ double sh[RW_TILE];
    const int H = nhills ? *nhills : bp.H;
    const int t = blockIdx.x * RW_THREADS + threadIdx.x;
    double s[METAD_MAX_CV];
#pragma unroll
    for (int d = 0; d < METAD_MAX_CV; ++d) s[d] = (d < bp.D && t < T) ? points[(size_t)t * bp.D + d] : 0.0;
    double acc = 0.0;
    for (int base = 0; base < H; base += RW_TILE) {
        const int nh = min(RW_TILE, H - base);
        __syncthreads();
        for (int k = threadIdx.x; k < nh; k += RW_THREADS) {
            sh[k] = heights[base + k];
#pragma unroll
            for (int d = 0; d < METAD_MAX_CV; ++d)
                if (d < bp.D) sc[d][k] = centers[(size_t)d * bp.max_hills + base + k];
        }
        __syncthreads();
        for (int k = 0; k < nh; ++k) {
            double e = 0.0;
#pragma unroll
            for (int d = 0; d < METAD_MAX_CV; ++d) {
                if (d < bp.D) {
                    double x = s[d] - sc[d][k];
                    if (bp.period[d] > 0.0) x -= bp.period[d] * rint(x * bp.inv_period[d]);   // nearest image (reading W)
                    x *= bp.inv_sigma[d];
                    e += x * x;
                }
            }
            acc += sh[k] * exp(-0.5 * e);
        }
    }
    if (t < T) V[t] = acc;
}

// order-preserving map double -> uint64 (for an atomic max that does not care about the order of arrival)
__device__ __forceinline__ unsigned long long dkey(double x) {
    unsigned long long u = (unsigned long long)__double_as_longlong(x);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}
__host__ __device__ inline double dkey_inv(unsigned long long k) {
    unsigned long long u = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
#ifdef __CUDA_ARCH__
    return __longlong_as_double((long long)u);
#else
    double d; memcpy(&d, &u, sizeof(d)); return d;
#endif
}

__global__ void k_vmax(int T, const double *__restrict__ V, unsigned long long *__restrict__ key) {
    unsigned long long m = 0ull;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < T; t += gridDim.x * blockDim.x) m = max(m, dkey(V[t]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_down_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(key, m);
}

#define RW_FIXED 1099511627776.0   // 2^40

__global__ void k_reweight_hist(RwBins rb, int T, const double *__restrict__ traj, const double *__restrict__ V,
                                const unsigned long long *__restrict__ vmax_key, double inv_kT,
                                unsigned long long *__restrict__ hist /* [nb0*nb1] + total */) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const double vmax = dkey_inv(*vmax_key);
    const double w = exp((V[t] - vmax) * inv_kT);
    const unsigned long long q = (unsigned long long)(w * RW_FIXED + 0.5);
    int idx[2] = { 0, 0 };
    bool inside = true;
#pragma unroll
    for (int d = 0; d < 2; ++d) {
        if (d < rb.D) {
            double x = traj[(size_t)t * rb.D + d];
            if (rb.period[d] > 0.0) {
                x -= rb.period[d] * floor((x - rb.lo[d]) / rb.period[d]);
                if (x >= rb.lo[d] + rb.period[d]) x -= rb.period[d];
                if (x < rb.lo[d]) x += rb.period[d];
            }
            int b = (int)floor((x - rb.lo[d]) / rb.h[d]);
            if (rb.period[d] > 0.0 && b >= rb.nb[d]) b = rb.nb[d] - 1;
            if (b < 0 || b >= rb.nb[d] || !(x >= rb.lo[d])) inside = false;
            idx[d] = b;
        }
    }
    const int nbins = rb.nb[0] * rb.nb[1];
    atomicAdd(hist + nbins, q);
    if (inside) atomicAdd(hist + (size_t)idx[0] * rb.nb[1] + idx[1], q);
}

__global__ void k_reweight_finish(RwBins rb, const unsigned long long *__restrict__ hist, double kT,
                                  double *__restrict__ P, double *__restrict__ F) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    const int nbins = rb.nb[0] * rb.nb[1];
    if (b >= nbins) return;
    const double tot = (double)hist[nbins];
    const double p = tot > 0.0 ? (double)hist[b] / (tot * rb.vol) : 0.0;
    P[b] = p;
    F[b] = p > 0.0 ? -kT * log(p) : (double)INFINITY;
}

// ------------------------------------------------------------------------------------------------
static RwBias make_rwbias(const metad_ctx *c) {
    RwBias bp;
    bp.D = c->D; bp.H = 0; bp.max_hills = c->p.max_hills;
    for (int d = 0; d < METAD_MAX_CV; ++d) {
        bp.inv_sigma[d] = d < c->D ? 1.0 / c->p.sigma[d] : 1.0;
        bp.period[d] = d < c->D ? c->p.period[d] : 0.0;
        bp.inv_period[d] = bp.period[d] > 0.0 ? 1.0 / bp.period[d] : 0.0;
    }
    return bp;
}

int bias_batch(metad_ctx *c, const double *d_points, int T, double *d_V) {
    if (T == 0) return METAD_OK;
    k_bias_batch<<<div_up(T, RW_THREADS), RW_THREADS, 0, c->stream>>>(make_rwbias(c), c->d_centers, c->d_heights, c->d_nhills,
                                                                      d_points, T, d_V);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int reweight_run(metad_ctx *c, const double *d_traj, int T, const int *nbins, const double *lo, const double *hi,
                 double *d_P, double *d_F) {
    RwBins rb;
    rb.D = c->D; rb.vol = 1.0;
    for (int d = 0; d < 2; ++d) {
        const bool on = d < c->D;
        rb.nb[d] = on ? nbins[d] : 1;
        rb.lo[d] = on ? lo[d] : 0.0; rb.hi[d] = on ? hi[d] : 1.0;
        rb.h[d] = (rb.hi[d] - rb.lo[d]) / rb.nb[d];
        rb.period[d] = on ? c->p.period[d] : 0.0;
        if (on) rb.vol *= (rb.hi[d] - rb.lo[d]) / rb.nb[d];
    }
    const int nb = rb.nb[0] * rb.nb[1];
    double *d_V = nullptr;
    unsigned long long *d_hist = nullptr;     // [nb] bins, [nb] total, [nb + 1] key of max V
    CUDA_TRY(cudaMalloc((void **)&d_V, sizeof(double) * (size_t)(T > 0 ? T : 1)));
    CUDA_TRY(cudaMalloc((void **)&d_hist, sizeof(unsigned long long) * ((size_t)nb + 2)));
    CUDA_TRY(cudaMemsetAsync(d_hist, 0, sizeof(unsigned long long) * ((size_t)nb + 2), c->stream));
    int r = bias_batch(c, d_traj, T, d_V);
    if (r == METAD_OK && T > 0) {
        k_vmax<<<std::min(div_up(T, 256), 1024), 256, 0, c->stream>>>(T, d_V, d_hist + nb + 1);
        k_reweight_hist<<<div_up(T, 256), 256, 0, c->stream>>>(rb, T, d_traj, d_V, d_hist + nb + 1, 1.0 / c->p.kT, d_hist);
        c->launches += 2;
    }
    k_reweight_finish<<<div_up(nb, 256), 256, 0, c->stream>>>(rb, d_hist, c->p.kT, d_P, d_F);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    cudaStreamSynchronize(c->stream);
    cudaFree(d_V); cudaFree(d_hist);
    CUDA_TRY(e);
    return r;
}
