// reweight.cu — NEXT-2: batched bias evaluation and free-energy reconstruction by reweighting
// (PAPER.md:85-87):  P(s) = < delta[s - s(R)] e^{beta V_b} > / < e^{beta V_b} >,  F = -(1/beta) log P,
// averages over the frames of the biased trajectory (reading Z: delta = uniform bins).
//   k_bias_batch      V_b at T points: thread per point, the hill array streamed through shared memory
//                     in tiles (the FP64 exp is the work: T x H evaluations, pure ALU, no HBM re-reads)
//   k_reweight_binmax bin of every frame; largest V inside each bin (order-independent atomic max)
//   k_reweight_hist   w = e^{(V - Vmax_bin)/kT} as 2^-64 fixed point summed into a 128-bit integer per bin: the
//                     sums do not depend on the order of the atomics => run-to-run bit-identical, and a bin far
//                     below the most probable one keeps the full resolution of its own sum
//   k_reweight_finish bins combined in log space: P = W_b / (sum W x bin volume), F = -kT log P (+inf for empty bins)
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
__device__ __forceinline__ double dkey_inv(unsigned long long k) {
    unsigned long long u = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
    return __longlong_as_double((long long)u);
}

// bin of a frame (reading Z); nbins = the "outside" bin (frames beyond a non-periodic range: denominator only)
__device__ __forceinline__ int rw_bin(const RwBins &rb, const double *__restrict__ s) {
    int idx[2] = { 0, 0 };
    bool inside = true;
#pragma unroll
    for (int d = 0; d < 2; ++d) {
        if (d < rb.D) {
            double x = s[d];
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
    return inside ? idx[0] * rb.nb[1] + idx[1] : rb.nb[0] * rb.nb[1];
}

// Pass A: bin of every frame and the largest V inside each bin (atomic max on an order-preserving key).
__global__ void k_reweight_binmax(RwBins rb, int T, const double *__restrict__ traj, const double *__restrict__ V,
                                  int *__restrict__ bin_of, unsigned long long *__restrict__ vmax_key /* [nbins + 1] */) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const int b = rw_bin(rb, traj + (size_t)t * rb.D);
    bin_of[t] = b;
    atomicMax(vmax_key + b, dkey(V[t]));
}

// Pass B: the weight of a frame RELATIVE TO THE LARGEST ONE OF ITS OWN BIN, w = e^{(V - Vmax_bin)/kT} in (0, 1], as a 2^-64
// fixed-point number summed into a 128-bit integer per bin (low word by atomicAdd, the carry into the high word): an
// integer sum does not depend on the order of the atomics, so P and F are bit-identical from run to run; a bin holds up to
// 2^63 frames, and a bin 60 kT (or 600 kT) below the most probable one keeps the full 64-bit resolution of its own sum —
// nothing is quantised against the global maximum (the bins are combined in log space by k_reweight_finish).
__global__ void k_reweight_hist(int T, const double *__restrict__ V, const int *__restrict__ bin_of,
                                const unsigned long long *__restrict__ vmax_key, double inv_kT,
                                unsigned long long *__restrict__ sum_lo, unsigned long long *__restrict__ sum_hi) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const int b = bin_of[t];
    const double w = exp((V[t] - dkey_inv(vmax_key[b])) * inv_kT);           // <= 1, == 1 for the bin's top frame
    const double x = w * 18446744073709551616.0;                              // * 2^64, exact scaling
    if (x >= 18446744073709551616.0) { atomicAdd(sum_hi + b, 1ull); return; }
    const unsigned long long q = (unsigned long long)x;                       // truncation: deterministic
    const unsigned long long old = atomicAdd(sum_lo + b, q);
    if (old + q < old) atomicAdd(sum_hi + b, 1ull);                           // carry
}

// log of the (unnormalised) weight of every bin, log W_b = log(sum_b) + Vmax_b / kT; the normalisation
// log sum_b' W_b' (outside bin included) by a fixed-order log-sum-exp in one block; then
//     P_b = W_b / (sum W vol),   F_b = -kT log P_b   (formed in log space: finite whenever the bin holds a frame).
#define RW_FIN_THREADS 1024
__global__ void __launch_bounds__(RW_FIN_THREADS)
k_reweight_finish(RwBins rb, const unsigned long long *__restrict__ sum_lo, const unsigned long long *__restrict__ sum_hi,
                  const unsigned long long *__restrict__ vmax_key, double kT, double *__restrict__ P, double *__restrict__ F) {
    __shared__ double red[32];
    __shared__ double s_top, s_logtot;
    const int nbins = rb.nb[0] * rb.nb[1];
    const double inv_kT = 1.0 / kT;
    auto logw = [&](int b) -> double {
        const double sum = (double)sum_hi[b] + (double)sum_lo[b] * (1.0 / 18446744073709551616.0);
        return sum > 0.0 ? log(sum) + dkey_inv(vmax_key[b]) * inv_kT : -INFINITY;
    };
    // largest log W (fixed order)
    double m = -INFINITY;
    for (int b = threadIdx.x; b <= nbins; b += blockDim.x) m = fmax(m, logw(b));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_down_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = red[0];
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) t = fmax(t, red[w]);
        s_top = t;
    }
    __syncthreads();
    const double top = s_top;
    double acc[1] = { 0.0 };
    if (top > -INFINITY)
        for (int b = threadIdx.x; b <= nbins; b += blockDim.x) { const double l = logw(b); if (l > -INFINITY) acc[0] += exp(l - top); }
    block_reduce<1>(acc, red);
    if (threadIdx.x == 0) s_logtot = top > -INFINITY ? top + log(acc[0]) : -INFINITY;
    __syncthreads();
    const double logtot = s_logtot, logvol = log(rb.vol);
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) {
        const double l = logw(b);
        if (l > -INFINITY) {
            const double lp = l - logtot - logvol;
            P[b] = exp(lp);
            F[b] = -kT * lp;
        } else {
            P[b] = 0.0;
            F[b] = (double)INFINITY;
        }
    }
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
    // scratch of this call (not a per-step call): V per frame, bin per frame, per bin (+ the outside bin) the key of the
    // largest V and the two words of the 128-bit weight sum
    double *d_V = nullptr;
    int *d_bin = nullptr;
    unsigned long long *d_acc = nullptr;
    const size_t nacc = 3 * ((size_t)nb + 1);
    cudaError_t ea = cudaMalloc((void **)&d_V, sizeof(double) * (size_t)(T > 0 ? T : 1));
    if (ea == cudaSuccess) ea = cudaMalloc((void **)&d_bin, sizeof(int) * (size_t)(T > 0 ? T : 1));
    if (ea == cudaSuccess) ea = cudaMalloc((void **)&d_acc, sizeof(unsigned long long) * nacc);
    if (ea != cudaSuccess) { cudaFree(d_V); cudaFree(d_bin); cudaFree(d_acc); CUDA_TRY(ea); }
    unsigned long long *d_key = d_acc, *d_lo = d_acc + (nb + 1), *d_hi = d_acc + 2 * ((size_t)nb + 1);
    cudaMemsetAsync(d_acc, 0, sizeof(unsigned long long) * nacc, c->stream);      // key 0 sorts below every double
    int r = bias_batch(c, d_traj, T, d_V);
    if (r == METAD_OK && T > 0) {
        k_reweight_binmax<<<div_up(T, 256), 256, 0, c->stream>>>(rb, T, d_traj, d_V, d_bin, d_key);
        k_reweight_hist<<<div_up(T, 256), 256, 0, c->stream>>>(T, d_V, d_bin, d_key, 1.0 / c->p.kT, d_lo, d_hi);
        c->launches += 2;
    }
    k_reweight_finish<<<1, RW_FIN_THREADS, 0, c->stream>>>(rb, d_lo, d_hi, d_key, c->p.kT, d_P, d_F);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    cudaStreamSynchronize(c->stream);
    cudaFree(d_V); cudaFree(d_bin); cudaFree(d_acc);
    CUDA_TRY(e);
    return r;
}
