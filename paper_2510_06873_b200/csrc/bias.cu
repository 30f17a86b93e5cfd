// bias.cu — a5 hill sum, a5g grid-tabulated bias (bicubic Hermite), a7 on-device deposition.
// V_b(s) = sum_tau w_tau exp(-(s - s_tau)^2 / (2 sigma^2)); well-tempered heights per
// PAPER.md:43 / ref. [16] (reading I).  Everything fp64; hill count and step counter live on the device
// so that the whole step can sit inside a CUDA graph.
#include "common.cuh"
#include "cv_torsion.cuh"

#define BIAS_THREADS 256
#define BIAS_MAX_BLOCKS 592   // 4 x 148 SMs

struct BiasParams {
    int D, max_hills;
    double sigma[METAD_MAX_CV];
    double inv_sigma[METAD_MAX_CV];
    double period[METAD_MAX_CV];     // 0: not periodic (reading W)
};

struct GridParams {
    int n0, n1;
    double lo[2], hi[2], h[2], inv_h[2];
    double period[2];                // > 0: periodic dimension, n nodes at lo + i * period / n (reading X)
};

// s - c brought to the nearest periodic image (reading W); P = 0: plain difference
__device__ __forceinline__ double pdiff(double s, double c, double P) {
    double d = s - c;
    if (P > 0.0) d -= P * rint(d / P);
    return d;
}

// device scalars, one int array:  [0] = grid miss flag of this step, [1] = index of the hill
// deposited in this step (-1: none)
#define AUX_GRID_MISS 0
#define AUX_DEP_INDEX 1

// ------------------------------------------------------------------------------------------------
// a7: deposition (readings I, J, U).  One thread.  V = the bias at cv from the hills deposited before this step.
__device__ __forceinline__ void deposit_one(const BiasParams &bp, int stride, double w0, double kT, double gamma,
                                            const double *cv, double V, double *centers, double *heights, int *nhills,
                                            int *step, int *aux, unsigned int *sticky, double *traj, int traj_cap) {
    int st = *step + 1;
    *step = st;
    if (traj) {                                   // device-resident CV trajectory (reweighting input)
        if (st <= traj_cap) { for (int d = 0; d < bp.D; ++d) traj[(size_t)(st - 1) * bp.D + d] = cv[d]; }
        else atomicOr(sticky, (unsigned)METAD_DEV_TRAJ_FULL);
    }
    aux[AUX_DEP_INDEX] = -1;
    if (stride <= 0 || st % stride != 0) return;
    int H = *nhills;
    if (H >= bp.max_hills) { atomicOr(sticky, (unsigned)METAD_DEV_HILL_OVERFLOW); return; }
    double h = gamma > 1.0 ? w0 * exp(-V / ((gamma - 1.0) * kT)) : w0;
    for (int d = 0; d < bp.D; ++d) centers[(size_t)d * bp.max_hills + H] = cv[d];
    heights[H] = h;
    *nhills = H + 1;
    aux[AUX_DEP_INDEX] = H;
}

__global__ void k_deposit(BiasParams bp, int stride, double w0, double kT, double gamma, const double *__restrict__ cv,
                          const double *__restrict__ V, double *__restrict__ centers, double *__restrict__ heights,
                          int *__restrict__ nhills, int *__restrict__ step, int *__restrict__ aux,
                          unsigned int *__restrict__ sticky, double *__restrict__ traj, int traj_cap) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    deposit_one(bp, stride, w0, kT, gamma, cv, *V, centers, heights, nhills, step, aux, sticky, traj, traj_cap);
}

// deposition riding on the hill sum (metad_run / metad_step_host without a grid): the last block of k_bias_sum, which holds
// V, deposits in the same launch — every other block has finished reading the hill arrays by then (ticket), the new hill
// goes to slot H, which this launch never read
struct DepArgs { int on, stride, traj_cap; double w0, kT, gamma; int *step; unsigned int *sticky; double *traj; };

// ------------------------------------------------------------------------------------------------
// exact hill sum at one point: blocks stride over the hill array, fixed-order reduction.
__global__ void __launch_bounds__(BIAS_THREADS)
k_bias_sum(BiasParams bp, double *centers, double *heights, int *nhills, const double *__restrict__ cv,
           double *__restrict__ partials, unsigned int *__restrict__ ticket, double *__restrict__ V,
           double *__restrict__ dVds, int *aux, int grid_on, DepArgs dep) {
    __shared__ double red[(1 + METAD_MAX_CV) * 32];
    if (grid_on && aux[AUX_GRID_MISS] == 0) return;   // the grid lookup already produced V, dVds
    const int H = *nhills;
    double s[METAD_MAX_CV];
#pragma unroll
    for (int d = 0; d < METAD_MAX_CV; ++d) s[d] = d < bp.D ? cv[d] : 0.0;
    double acc[1 + METAD_MAX_CV];
#pragma unroll
    for (int d = 0; d <= METAD_MAX_CV; ++d) acc[d] = 0.0;
    for (int k = blockIdx.x * BIAS_THREADS + threadIdx.x; k < H; k += gridDim.x * BIAS_THREADS) {
        double e = 0.0, t[METAD_MAX_CV];
#pragma unroll
        for (int d = 0; d < METAD_MAX_CV; ++d) {
            if (d < bp.D) {
                t[d] = pdiff(s[d], centers[(size_t)d * bp.max_hills + k], bp.period[d]) * bp.inv_sigma[d];
                e += t[d] * t[d];
            }
        }
        double g = heights[k] * exp(-0.5 * e);
        acc[0] += g;
#pragma unroll
        for (int d = 0; d < METAD_MAX_CV; ++d)
            if (d < bp.D) acc[1 + d] -= g * t[d] * bp.inv_sigma[d];
    }
    block_reduce<1 + METAD_MAX_CV>(acc, red);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int d = 0; d <= METAD_MAX_CV; ++d) partials[blockIdx.x * (1 + METAD_MAX_CV) + d] = acc[d];
    }
    if (last_block_ticket(ticket)) {
        double t[1 + METAD_MAX_CV];
#pragma unroll
        for (int d = 0; d <= METAD_MAX_CV; ++d) t[d] = 0.0;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) {
#pragma unroll
            for (int d = 0; d <= METAD_MAX_CV; ++d) t[d] += partials[b * (1 + METAD_MAX_CV) + d];
        }
        block_reduce<1 + METAD_MAX_CV>(t, red);
        if (threadIdx.x == 0) {
            *V = t[0];
            for (int d = 0; d < bp.D; ++d) dVds[d] = t[1 + d];
            if (dep.on)
                deposit_one(bp, dep.stride, dep.w0, dep.kT, dep.gamma, cv, t[0], centers, heights, nhills, dep.step, aux,
                            dep.sticky, dep.traj, dep.traj_cap);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// grid lookup: bicubic Hermite on node values V, V_0, V_1, V_01 (reading M)
__device__ __forceinline__ void hermite(double t, double *h, double *dh) {
    double t2 = t * t, t3 = t2 * t;
    h[0] = 2 * t3 - 3 * t2 + 1; h[1] = -2 * t3 + 3 * t2; h[2] = t3 - 2 * t2 + t; h[3] = t3 - t2;
    dh[0] = 6 * t2 - 6 * t; dh[1] = -6 * t2 + 6 * t; dh[2] = 3 * t2 - 4 * t + 1; dh[3] = 3 * t2 - 2 * t;
}

// bicubic Hermite lookup at (s0, s1); returns true if the point is outside a non-periodic range (no result then)
__device__ __forceinline__ bool grid_lookup(const GridParams &gp, const double *__restrict__ table, double s0, double s1,
                                            double &V, double &dV0, double &dV1) {
    const double sv[2] = { s0, s1 };
    const int nn[2] = { gp.n0, gp.n1 };
    int i0[2], i1[2];
    double tt[2];
    bool miss = false;
#pragma unroll
    for (int d = 0; d < 2; ++d) {
        if (gp.period[d] > 0.0) {            // periodic: wrap into [lo, lo + P); node n coincides with node 0
            double x = sv[d] - gp.period[d] * floor((sv[d] - gp.lo[d]) / gp.period[d]);
            if (x >= gp.lo[d] + gp.period[d]) x -= gp.period[d];
            if (x < gp.lo[d]) x += gp.period[d];
            const double f = (x - gp.lo[d]) * gp.inv_h[d];
            const int i = max(min((int)floor(f), nn[d] - 1), 0);
            tt[d] = f - i; i0[d] = i; i1[d] = i + 1 == nn[d] ? 0 : i + 1;
        } else {
            if (!(sv[d] >= gp.lo[d]) || !(sv[d] <= gp.hi[d])) miss = true;
            const double f = (sv[d] - gp.lo[d]) * gp.inv_h[d];
            const int i = max(min((int)floor(f), nn[d] - 2), 0);
            tt[d] = f - i; i0[d] = i; i1[d] = i + 1;
        }
    }
    if (miss || !isfinite(sv[0]) || !isfinite(sv[1])) return true;
    double hx[4], dhx[4], hy[4], dhy[4];
    hermite(tt[0], hx, dhx);
    hermite(tt[1], hy, dhy);
    size_t plane = (size_t)gp.n0 * gp.n1;
    double v = 0.0, vx = 0.0, vy = 0.0;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            size_t o = (size_t)(a ? i1[0] : i0[0]) * gp.n1 + (b ? i1[1] : i0[1]);
            double f = table[o], f0 = table[plane + o] * gp.h[0], f1 = table[2 * plane + o] * gp.h[1],
                   f01 = table[3 * plane + o] * gp.h[0] * gp.h[1];
            v += f * hx[a] * hy[b] + f0 * hx[2 + a] * hy[b] + f1 * hx[a] * hy[2 + b] + f01 * hx[2 + a] * hy[2 + b];
            vx += f * dhx[a] * hy[b] + f0 * dhx[2 + a] * hy[b] + f1 * dhx[a] * hy[2 + b] + f01 * dhx[2 + a] * hy[2 + b];
            vy += f * hx[a] * dhy[b] + f0 * hx[2 + a] * dhy[b] + f1 * hx[a] * dhy[2 + b] + f01 * hx[2 + a] * dhy[2 + b];
        }
    V = v; dV0 = vx * gp.inv_h[0]; dV1 = vy * gp.inv_h[1];
    return false;
}

__global__ void k_bias_grid(GridParams gp, const double *__restrict__ table, const double *__restrict__ cv,
                            double *__restrict__ V, double *__restrict__ dVds, int *__restrict__ aux,
                            unsigned int *__restrict__ sticky) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double v, d0, d1;
    if (grid_lookup(gp, table, cv[0], cv[1], v, d0, d1)) {
        aux[AUX_GRID_MISS] = 1;
        atomicOr(sticky, (unsigned)METAD_DEV_GRID_RANGE);
        return;
    }
    aux[AUX_GRID_MISS] = 0;
    *V = v; dVds[0] = d0; dVds[1] = d1;
}

// table build: 16x16 node tile per block; hills staged through shared memory in chunks, the two
// 1-D Gaussian factors computed once per (hill, row) / (hill, column) of the tile (separable form).
#define GT 16
#define GCH 64
__global__ void __launch_bounds__(GT * GT)
k_grid_accumulate(GridParams gp, BiasParams bp, const double *__restrict__ centers, const double *__restrict__ heights,
                  int k0, const int *__restrict__ nhills_dev, int k1_host, double *__restrict__ table) {
    __shared__ double ex[GCH][GT], gx[GCH][GT], ey[GCH][GT], gy[GCH][GT];
    const int k1 = nhills_dev ? *nhills_dev : k1_host;
    const int tx = threadIdx.x % GT, ty = threadIdx.x / GT;
    const int i = blockIdx.x * GT + ty, j = blockIdx.y * GT + tx;   // node (i along s0, j along s1)
    double v = 0.0, v0 = 0.0, v1 = 0.0, v01 = 0.0;
    for (int base = k0; base < k1; base += GCH) {
        int nh = min(GCH, k1 - base);
        __syncthreads();
        // 2*GCH*GT factor evaluations spread over the 256 threads
        for (int q = threadIdx.x; q < 2 * GCH * GT; q += GT * GT) {
            int which = q / (GCH * GT), r = q % (GCH * GT), h = r / GT, t = r % GT;
            if (h < nh) {
                int k = base + h;
                if (which == 0) {
                    double x = gp.lo[0] + (blockIdx.x * GT + t) * gp.h[0];
                    double a = pdiff(x, centers[k], gp.period[0]) * bp.inv_sigma[0];
                    ex[h][t] = heights[k] * exp(-0.5 * a * a);
                    gx[h][t] = -a * bp.inv_sigma[0];
                } else {
                    double y = gp.lo[1] + (blockIdx.y * GT + t) * gp.h[1];
                    double b = pdiff(y, centers[(size_t)bp.max_hills + k], gp.period[1]) * bp.inv_sigma[1];
                    ey[h][t] = exp(-0.5 * b * b);
                    gy[h][t] = -b * bp.inv_sigma[1];
                }
            }
        }
        __syncthreads();
        for (int h = 0; h < nh; ++h) {
            double g = ex[h][ty] * ey[h][tx];
            double ga = gx[h][ty], gb = gy[h][tx];
            v += g; v0 += g * ga; v1 += g * gb; v01 += g * ga * gb;
        }
    }
    if (i < gp.n0 && j < gp.n1) {
        size_t plane = (size_t)gp.n0 * gp.n1, o = (size_t)i * gp.n1 + j;
        table[o] += v; table[plane + o] += v0; table[2 * plane + o] += v1; table[3 * plane + o] += v01;
    }
}

// per-step: add the hill deposited in this step (if any) to every node
__global__ void k_grid_add_last(GridParams gp, BiasParams bp, const double *__restrict__ centers,
                                const double *__restrict__ heights, const int *__restrict__ aux,
                                double *__restrict__ table) {
    const int k = aux[AUX_DEP_INDEX];
    if (k < 0) return;
    int o = blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= gp.n0 * gp.n1) return;
    int i = o / gp.n1, j = o % gp.n1;
    double a = pdiff(gp.lo[0] + i * gp.h[0], centers[k], gp.period[0]) * bp.inv_sigma[0];
    double b = pdiff(gp.lo[1] + j * gp.h[1], centers[(size_t)bp.max_hills + k], gp.period[1]) * bp.inv_sigma[1];
    double g = heights[k] * exp(-0.5 * (a * a + b * b));
    double ga = -a * bp.inv_sigma[0], gb = -b * bp.inv_sigma[1];
    size_t plane = (size_t)gp.n0 * gp.n1;
    table[o] += g; table[plane + o] += g * ga; table[2 * plane + o] += g * gb; table[3 * plane + o] += g * ga * gb;
}

// ------------------------------------------------------------------------------------------------
// Fused step for torsion-only contexts (a 22-atom molecule, two torsions): CV evaluation, bias (grid
// lookup, else the exact hill sum by the whole block in a fixed order), gather-form forces and deposition in ONE launch.
// Such a step is nothing but launch latency (6 dependent launches of ~2.3 us otherwise).  Used by metad_run /
// metad_step_host when params.lazy_neighbors is set and every CV is a torsion; the five stage calls stay available.
struct FusedTors { int D; int idx[METAD_MAX_CV][4]; int natoms; };

template <typename T>
__global__ void __launch_bounds__(256)
k_fused_torsion_step(FusedTors ft, const int *__restrict__ tors_atoms, const T *__restrict__ pos, BoxD bd, BiasParams bp,
                     GridParams gp, int grid_on, const double *__restrict__ table, double *__restrict__ centers,
                     double *__restrict__ heights, int *__restrict__ nhills, int *__restrict__ step, int *__restrict__ aux,
                     unsigned int *__restrict__ sticky, int stride, double w0, double kT, double gamma, double force_scale,
                     double *__restrict__ cv_out, double *__restrict__ V_out, double *__restrict__ dVds_out,
                     double *__restrict__ tors_grad, T *__restrict__ F, double *__restrict__ traj, int traj_cap, const DevGeom *__restrict__ dg) {
    if (dg) bd = dg->bd;                          // device-resident box (NPT): metad_*_dev
    __shared__ double s_cv[METAD_MAX_CV], s_g[METAD_MAX_CV][12], s_V, s_dV[METAD_MAX_CV];
    __shared__ int s_exact;
    __shared__ double red[(1 + METAD_MAX_CV) * 32];
    const int tid = threadIdx.x;
    if (tid < ft.D) {                                            // a2t: one thread per torsion
        double b[3][3];
        for (int k = 0; k < 3; ++k) {
            for (int a = 0; a < 3; ++a)
                b[k][a] = (double)pos[3 * (size_t)ft.idx[tid][k + 1] + a] - (double)pos[3 * (size_t)ft.idx[tid][k] + a];
            min_image_d(bd, b[k][0], b[k][1], b[k][2]);
        }
        double g[12];
        const double phi = torsion_eval(b[0], b[1], b[2], g);
        s_cv[tid] = phi; cv_out[tid] = phi;
        for (int k = 0; k < 12; ++k) { s_g[tid][k] = g[k]; tors_grad[12 * tid + k] = g[k]; }
        if (!isfinite(phi)) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
    }
    __syncthreads();
    if (tid == 0) {                                              // a5g: table lookup
        int exact = 1;
        if (grid_on) {
            double v, d0, d1;
            if (grid_lookup(gp, table, s_cv[0], s_cv[1], v, d0, d1)) { aux[AUX_GRID_MISS] = 1; atomicOr(sticky, (unsigned)METAD_DEV_GRID_RANGE); }
            else { aux[AUX_GRID_MISS] = 0; s_V = v; s_dV[0] = d0; s_dV[1] = d1; exact = 0; }
        }
        s_exact = exact;
    }
    __syncthreads();
    if (s_exact) {                                               // a5: exact hill sum, thread-strided, fixed-order reduction
        const int H = *nhills;
        double acc[1 + METAD_MAX_CV];
#pragma unroll
        for (int d = 0; d <= METAD_MAX_CV; ++d) acc[d] = 0.0;
        for (int k = tid; k < H; k += blockDim.x) {
            double e = 0.0, t[METAD_MAX_CV];
#pragma unroll
            for (int d = 0; d < METAD_MAX_CV; ++d) {
                if (d < bp.D) {
                    t[d] = pdiff(s_cv[d], centers[(size_t)d * bp.max_hills + k], bp.period[d]) * bp.inv_sigma[d];
                    e += t[d] * t[d];
                }
            }
            const double g = heights[k] * exp(-0.5 * e);
            acc[0] += g;
#pragma unroll
            for (int d = 0; d < METAD_MAX_CV; ++d)
                if (d < bp.D) acc[1 + d] -= g * t[d] * bp.inv_sigma[d];
        }
        block_reduce<1 + METAD_MAX_CV>(acc, red);
        if (tid == 0) { s_V = acc[0]; for (int d = 0; d < bp.D; ++d) s_dV[d] = acc[1 + d]; }
        __syncthreads();
    }
    if (tid < ft.natoms) {                                       // a6: gather form, thread per touched atom
        const int a = tors_atoms[tid];
        double f[3] = { 0.0, 0.0, 0.0 };
        for (int d = 0; d < ft.D; ++d)
            for (int k = 0; k < 4; ++k)
                if (ft.idx[d][k] == a) { f[0] += s_dV[d] * s_g[d][3 * k]; f[1] += s_dV[d] * s_g[d][3 * k + 1]; f[2] += s_dV[d] * s_g[d][3 * k + 2]; }
        F[3 * (size_t)a] += (T)(-force_scale * f[0]);
        F[3 * (size_t)a + 1] += (T)(-force_scale * f[1]);
        F[3 * (size_t)a + 2] += (T)(-force_scale * f[2]);
    }
    if (tid == 0) {                                              // a7: deposition (readings I, J, U)
        *V_out = s_V;
        for (int d = 0; d < bp.D; ++d) dVds_out[d] = s_dV[d];
        const int st = *step + 1;
        *step = st;
        if (traj) {
            if (st <= traj_cap) { for (int d = 0; d < bp.D; ++d) traj[(size_t)(st - 1) * bp.D + d] = s_cv[d]; }
            else atomicOr(sticky, (unsigned)METAD_DEV_TRAJ_FULL);
        }
        aux[AUX_DEP_INDEX] = -1;
        if (stride > 0 && st % stride == 0) {
            const int H = *nhills;
            if (H >= bp.max_hills) atomicOr(sticky, (unsigned)METAD_DEV_HILL_OVERFLOW);
            else {
                const double h = gamma > 1.0 ? w0 * exp(-s_V / ((gamma - 1.0) * kT)) : w0;
                for (int d = 0; d < bp.D; ++d) centers[(size_t)d * bp.max_hills + H] = s_cv[d];
                heights[H] = h;
                *nhills = H + 1;
                aux[AUX_DEP_INDEX] = H;
            }
        }
    }
}

__global__ void k_hills_import(int D, int max_hills, int count, const double *__restrict__ rowmajor,
                               const double *__restrict__ h_in, double *__restrict__ centers,
                               double *__restrict__ heights, int *__restrict__ nhills) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k == 0) *nhills = count;
    if (k >= count) return;
    for (int d = 0; d < D; ++d) centers[(size_t)d * max_hills + k] = rowmajor[(size_t)k * D + d];
    heights[k] = h_in[k];
}

__global__ void k_hills_export(int D, int max_hills, int capacity, const double *__restrict__ centers,
                               const double *__restrict__ heights, const int *__restrict__ nhills,
                               double *__restrict__ rowmajor, double *__restrict__ h_out) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= *nhills || k >= capacity) return;
    for (int d = 0; d < D; ++d) rowmajor[(size_t)k * D + d] = centers[(size_t)d * max_hills + k];
    h_out[k] = heights[k];
}

// ------------------------------------------------------------------------------------------------
static BiasParams make_bp(const metad_ctx *c) {
    BiasParams bp;
    bp.D = c->D; bp.max_hills = c->p.max_hills;
    for (int d = 0; d < METAD_MAX_CV; ++d) {
        bp.sigma[d] = d < c->D ? c->p.sigma[d] : 1.0;
        bp.inv_sigma[d] = 1.0 / bp.sigma[d];
        bp.period[d] = d < c->D ? c->p.period[d] : 0.0;
    }
    return bp;
}
static GridParams make_gp(const metad_ctx *c) {
    GridParams gp;
    gp.n0 = c->p.grid_n[0]; gp.n1 = c->p.grid_n[1];
    for (int d = 0; d < 2; ++d) {
        gp.lo[d] = c->p.grid_lo[d]; gp.hi[d] = c->p.grid_hi[d];
        int n = d == 0 ? gp.n0 : gp.n1;
        gp.period[d] = c->p.period[d];
        gp.h[d] = gp.period[d] > 0.0 ? (gp.hi[d] - gp.lo[d]) / n : (n > 1 ? (gp.hi[d] - gp.lo[d]) / (n - 1) : 1.0);
        gp.inv_h[d] = 1.0 / gp.h[d];
    }
    return gp;
}


int bias_eval(metad_ctx *c, const double *d_cv, double *d_V, double *d_dVds, bool with_deposit) {
    BiasParams bp = make_bp(c);
    DepArgs dep = { 0, c->p.stride, c->p.traj_capacity, c->p.w0, c->p.kT, c->p.bias_factor, c->d_step, c->d_sticky, c->d_traj };
    if (with_deposit) {
        if (c->grid_on) return METAD_ERR_STATE;            // the table update follows the deposit: separate launches
        dep.on = 1;
    }
    if (c->grid_on) {
        k_bias_grid<<<1, 32, 0, c->stream>>>(make_gp(c), c->d_table, d_cv, d_V, d_dVds, ctx_aux(c), c->d_sticky);
        c->launches++;
    }
    int nb = div_up(c->p.max_hills, BIAS_THREADS);
    if (nb > BIAS_MAX_BLOCKS) nb = BIAS_MAX_BLOCKS;
    if (nb < 1) nb = 1;
    k_bias_sum<<<nb, BIAS_THREADS, 0, c->stream>>>(bp, c->d_centers, c->d_heights, c->d_nhills, d_cv, c->d_bias_partials,
                                                  c->d_tickets + 8, d_V, d_dVds, ctx_aux(c), c->grid_on, dep);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int bias_deposit(metad_ctx *c, const double *d_cv, const double *d_V) {
    BiasParams bp = make_bp(c);
    k_deposit<<<1, 32, 0, c->stream>>>(bp, c->p.stride, c->p.w0, c->p.kT, c->p.bias_factor, d_cv, d_V, c->d_centers,
                                       c->d_heights, c->d_nhills, c->d_step, ctx_aux(c), c->d_sticky, c->d_traj,
                                       c->p.traj_capacity);
    c->launches++;
    if (c->grid_on) {
        int nn = c->p.grid_n[0] * c->p.grid_n[1];
        k_grid_add_last<<<div_up(nn, 256), 256, 0, c->stream>>>(make_gp(c), bp, c->d_centers, c->d_heights, ctx_aux(c),
                                                                c->d_table);
        c->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int bias_grid_rebuild(metad_ctx *c) {
    if (!c->grid_on) return METAD_OK;
    GridParams gp = make_gp(c);
    CUDA_TRY(cudaMemsetAsync(c->d_table, 0, sizeof(double) * 4 * (size_t)gp.n0 * gp.n1, c->stream));
    dim3 g(div_up(gp.n0, GT), div_up(gp.n1, GT));
    k_grid_accumulate<<<g, GT * GT, 0, c->stream>>>(gp, make_bp(c), c->d_centers, c->d_heights, 0, c->d_nhills, 0,
                                                    c->d_table);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int bias_set_hills_dev(metad_ctx *c, const double *d_rowmajor, const double *d_heights, int count) {
    k_hills_import<<<div_up(count > 0 ? count : 1, 256), 256, 0, c->stream>>>(c->D, c->p.max_hills, count, d_rowmajor,
                                                                            d_heights, c->d_centers, c->d_heights,
                                                                            c->d_nhills);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return bias_grid_rebuild(c);
}

int bias_get_hills_dev(metad_ctx *c, double *d_rowmajor, double *d_heights, int capacity) {
    k_hills_export<<<div_up(c->p.max_hills, 256), 256, 0, c->stream>>>(c->D, c->p.max_hills, capacity, c->d_centers,
                                                                     c->d_heights, c->d_nhills, d_rowmajor, d_heights);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}


// the whole step of a torsion-only context in one launch (+ the table update in grid mode)
int bias_fused_torsion_step(metad_ctx *c, const void *d_pos, void *d_F) {
    FusedTors ft;
    ft.D = c->D; ft.natoms = c->ntors_atoms;
    for (int d = 0; d < METAD_MAX_CV; ++d)
        for (int k = 0; k < 4; ++k) ft.idx[d][k] = d < c->D ? c->cv[d].tors[k] : 0;
    BiasParams bp = make_bp(c);
    GridParams gp = make_gp(c);
    if (c->prec == 32)
        k_fused_torsion_step<float><<<1, 256, 0, c->stream>>>(ft, c->d_tors_atoms, (const float *)d_pos, c->boxd, bp, gp, c->grid_on,
            c->d_table, c->d_centers, c->d_heights, c->d_nhills, c->d_step, ctx_aux(c), c->d_sticky, c->p.stride, c->p.w0, c->p.kT,
            c->p.bias_factor, c->p.force_scale, c->d_cv, c->d_V, c->d_dVds, c->d_tors_grad, (float *)d_F, c->d_traj, c->p.traj_capacity, c->dg);
    else
        k_fused_torsion_step<double><<<1, 256, 0, c->stream>>>(ft, c->d_tors_atoms, (const double *)d_pos, c->boxd, bp, gp, c->grid_on,
            c->d_table, c->d_centers, c->d_heights, c->d_nhills, c->d_step, ctx_aux(c), c->d_sticky, c->p.stride, c->p.w0, c->p.kT,
            c->p.bias_factor, c->p.force_scale, c->d_cv, c->d_V, c->d_dVds, c->d_tors_grad, (double *)d_F, c->d_traj, c->p.traj_capacity, c->dg);
    c->launches++;
    if (c->grid_on) {
        int nn = c->p.grid_n[0] * c->p.grid_n[1];
        k_grid_add_last<<<div_up(nn, 256), 256, 0, c->stream>>>(gp, bp, c->d_centers, c->d_heights, ctx_aux(c), c->d_table);
        c->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
