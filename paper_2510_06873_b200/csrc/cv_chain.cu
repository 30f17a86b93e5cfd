// cv_chain.cu — a4: radius of gyration of an ordered chain and native-contact fraction
// (BASELINE.json configs[1]; readings G, H).  Tiny kernels: ~1,000 atoms / ~5,000 pairs, all fp64,
// positions read from the caller's array in its own dtype.
#include "common.cuh"
#include "cv_torsion.cuh"

#define RG_THREADS 1024

struct RgScratch { double com[3]; double M; double rg; };   // stored after the unwrapped coords

// single block: unwrap by a block-wide prefix sum of minimum-image bond vectors, then COM and Rg.
template <typename T>
__global__ void __launch_bounds__(RG_THREADS)
k_rgyr(int nchain, const int *__restrict__ chain, const double *__restrict__ mass, const T *__restrict__ pos,
       BoxD bd, double *__restrict__ unwrapped, double *__restrict__ cv_out, unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg) {
    if (dg) bd = dg->bd;                          // device-resident box (NPT): metad_*_dev
    __shared__ double wsum[3][32];
    __shared__ double carry[3];
    __shared__ double red[4 * 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x < 3) carry[threadIdx.x] = 0.0;
    __syncthreads();
    for (int base = 0; base < nchain; base += RG_THREADS) {
        int k = base + threadIdx.x;
        double v[3] = { 0.0, 0.0, 0.0 };
        if (k < nchain) {
            int i = chain[k];
            if (k == 0) {
                v[0] = (double)pos[3 * i]; v[1] = (double)pos[3 * i + 1]; v[2] = (double)pos[3 * i + 2];
            } else {
                int p = chain[k - 1];
                v[0] = (double)pos[3 * i] - (double)pos[3 * p];
                v[1] = (double)pos[3 * i + 1] - (double)pos[3 * p + 1];
                v[2] = (double)pos[3 * i + 2] - (double)pos[3 * p + 2];
                min_image_d(bd, v[0], v[1], v[2]);
            }
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                double t = __shfl_up_sync(0xffffffffu, v[a], o);
                if (lane >= o) v[a] += t;
            }
            if (lane == 31) wsum[a][wid] = v[a];
        }
        __syncthreads();
        if (wid == 0) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                double w = wsum[a][lane], inc = w;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    double t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                wsum[a][lane] = inc - w;
            }
        }
        __syncthreads();
        double tot[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            v[a] += wsum[a][wid] + carry[a];
            if (k < nchain) unwrapped[3 * k + a] = v[a];
            tot[a] = v[a];
        }
        __syncthreads();
        if (threadIdx.x == RG_THREADS - 1) { carry[0] = tot[0]; carry[1] = tot[1]; carry[2] = tot[2]; }
        __syncthreads();
    }
    // centre of mass
    double s[4] = { 0.0, 0.0, 0.0, 0.0 };
    for (int k = threadIdx.x; k < nchain; k += RG_THREADS) {
        double mk = mass ? mass[k] : 1.0;
        s[0] += mk * unwrapped[3 * k]; s[1] += mk * unwrapped[3 * k + 1]; s[2] += mk * unwrapped[3 * k + 2];
        s[3] += mk;
    }
    block_reduce<4>(s, red);
    __shared__ double com[4];
    if (threadIdx.x == 0) { com[0] = s[0] / s[3]; com[1] = s[1] / s[3]; com[2] = s[2] / s[3]; com[3] = s[3]; }
    __syncthreads();
    double q[1] = { 0.0 };
    for (int k = threadIdx.x; k < nchain; k += RG_THREADS) {
        double mk = mass ? mass[k] : 1.0;
        double x = unwrapped[3 * k] - com[0], y = unwrapped[3 * k + 1] - com[1], z = unwrapped[3 * k + 2] - com[2];
        q[0] += mk * (x * x + y * y + z * z);
    }
    block_reduce<1>(q, red);
    if (threadIdx.x == 0) {
        double rg = sqrt(q[0] / com[3]);
        RgScratch *sc = reinterpret_cast<RgScratch *>(unwrapped + 3 * (size_t)nchain);
        sc->com[0] = com[0]; sc->com[1] = com[1]; sc->com[2] = com[2]; sc->M = com[3]; sc->rg = rg;
        *cv_out = rg;
        if (!isfinite(rg)) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
    }
}

template <typename T>
__global__ void k_rgyr_force(int nchain, const int *__restrict__ chain, const double *__restrict__ mass,
                             const double *__restrict__ unwrapped, double force_scale,
                             const double *__restrict__ dVds, T *__restrict__ F) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nchain) return;
    const RgScratch *sc = reinterpret_cast<const RgScratch *>(unwrapped + 3 * (size_t)nchain);
    if (!(sc->rg > 0.0)) return;
    double mk = mass ? mass[k] : 1.0;
    double a = -force_scale * dVds[0] * mk / (sc->M * sc->rg);
    int i = chain[k];
    F[3 * i] += (T)(a * (unwrapped[3 * k] - sc->com[0]));
    F[3 * i + 1] += (T)(a * (unwrapped[3 * k + 1] - sc->com[1]));
    F[3 * i + 2] += (T)(a * (unwrapped[3 * k + 2] - sc->com[2]));
}

__device__ __forceinline__ double switch_d(double x, int n, int m, double &dsw) {
    double xn1 = 1.0;
    for (int k = 0; k < n - 1; ++k) xn1 *= x;
    if (m == 2 * n) {
        double inv = 1.0 / (1.0 + xn1 * x);
        dsw = -(double)n * xn1 * inv * inv;
        return inv;
    }
    double e = x - 1.0;
    if (fabs(e) < 1e-6) {
        dsw = (double)n * (double)(n - m) / (2.0 * (double)m);
        return (double)n / (double)m + dsw * e;
    }
    double xm1 = 1.0;
    for (int k = 0; k < m - 1; ++k) xm1 *= x;
    double num = 1.0 - xn1 * x, den = 1.0 - xm1 * x;
    dsw = (-(double)n * xn1 * den + num * (double)m * xm1) / (den * den);
    return num / den;
}

template <typename T>
__global__ void __launch_bounds__(256)
k_contacts_cv(int npairs, const int *__restrict__ pairs, const double *__restrict__ pair_r0, int n, int m,
              double scale, const T *__restrict__ pos, BoxD bd, double *__restrict__ partials,
              unsigned int *__restrict__ ticket, double *__restrict__ cv_out, unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg) {
    if (dg) bd = dg->bd;                          // device-resident box (NPT): metad_*_dev
    __shared__ double red[32];
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    double v[1] = { 0.0 };
    if (p < npairs) {
        int i = pairs[2 * p], j = pairs[2 * p + 1];
        double dx = (double)pos[3 * j] - (double)pos[3 * i], dy = (double)pos[3 * j + 1] - (double)pos[3 * i + 1],
               dz = (double)pos[3 * j + 2] - (double)pos[3 * i + 2];
        min_image_d(bd, dx, dy, dz);
        double dsw;
        v[0] = switch_d(sqrt(dx * dx + dy * dy + dz * dz) / pair_r0[p], n, m, dsw);
    }
    block_reduce<1>(v, red);
    if (threadIdx.x == 0) partials[blockIdx.x] = v[0];
    if (last_block_ticket(ticket)) {
        double t[1] = { 0.0 };
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) t[0] += partials[b];
        block_reduce<1>(t, red);
        if (threadIdx.x == 0) {
            double r = scale * t[0];
            *cv_out = r;
            if (!isfinite(r)) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
        }
    }
}

// gather form: one WARP per atom that appears in any pair; csr lists its incident pairs, the lanes share them and a
// fixed shuffle tree sums the lane partials (deterministic; ~1,000 atoms with ~10 pairs each are pure latency otherwise).
template <typename T>
__global__ void k_contacts_force(int natoms_touched, const int *__restrict__ atoms, const int *__restrict__ csr_off,
                                 const int *__restrict__ csr_pair, const int *__restrict__ pairs,
                                 const double *__restrict__ pair_r0, int n, int m, double coef /* fs*scale */,
                                 const T *__restrict__ pos, BoxD bd, const double *__restrict__ dVds,
                                 T *__restrict__ F, const DevGeom *__restrict__ dg) {
    if (dg) bd = dg->bd;                          // device-resident box (NPT): metad_*_dev
    const int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (t >= natoms_touched) return;
    int a = atoms[t];
    double ax = 0.0, ay = 0.0, az = 0.0;
    for (int q = csr_off[t] + lane; q < csr_off[t + 1]; q += 32) {
        int p = csr_pair[q];
        int o = pairs[2 * p] == a ? pairs[2 * p + 1] : pairs[2 * p];
        double dx = (double)pos[3 * o] - (double)pos[3 * a], dy = (double)pos[3 * o + 1] - (double)pos[3 * a + 1],
               dz = (double)pos[3 * o + 2] - (double)pos[3 * a + 2];
        min_image_d(bd, dx, dy, dz);
        double r = sqrt(dx * dx + dy * dy + dz * dz), dsw;
        switch_d(r / pair_r0[p], n, m, dsw);
        double g = dsw / (pair_r0[p] * r);
        ax += g * dx; ay += g * dy; az += g * dz;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        ax += __shfl_down_sync(0xffffffffu, ax, o);
        ay += __shfl_down_sync(0xffffffffu, ay, o);
        az += __shfl_down_sync(0xffffffffu, az, o);
    }
    if (lane != 0) return;
    // dQ/dr_a = scale * sum g * (-d_a)  ->  F_a += +fs*scale*dVds * sum g*d_a
    double c = coef * dVds[0];
    F[3 * a] += (T)(c * ax);
    F[3 * a + 1] += (T)(c * ay);
    F[3 * a + 2] += (T)(c * az);
}


template <typename T>
static int chain_eval_t(metad_ctx *c, int dim, double *d_cv) {
    CvDev &d = c->cv[dim];
    const T *pos = (const T *)ctx_last_pos(c);
    if (d.kind == METAD_CV_RGYR) {
        k_rgyr<T><<<1, RG_THREADS, 0, c->stream>>>(d.nchain, d.d_chain, d.d_mass, pos, c->boxd, d.d_unwrapped, d_cv + dim,
                                                   c->d_sticky, c->dg);
    } else {
        int nb = div_up(d.npairs, 256);
        k_contacts_cv<T><<<nb, 256, 0, c->stream>>>(d.npairs, d.d_pairs, d.d_pair_r0, d.n, d.m, d.scale, pos, c->boxd,
                                                    c->d_partials + 3 * (size_t)c->nblocks_atoms, c->d_tickets + 2 + dim,
                                                    d_cv + dim, c->d_sticky, c->dg);
    }
    c->launches++;
    return METAD_OK;
}

int chain_eval(metad_ctx *c, int dim, const void *, double *d_cv) {
    return c->prec == 32 ? chain_eval_t<float>(c, dim, d_cv) : chain_eval_t<double>(c, dim, d_cv);
}

template <typename T>
static int chain_forces_t(metad_ctx *c, const double *d_dVds, void *d_F) {
    const T *pos = (const T *)ctx_last_pos(c);
    for (int dim = 0; dim < c->D; ++dim) {
        CvDev &d = c->cv[dim];
        if (d.kind == METAD_CV_RGYR) {
            k_rgyr_force<T><<<div_up(d.nchain, 128), 128, 0, c->stream>>>(d.nchain, d.d_chain, d.d_mass, d.d_unwrapped,
                                                                        c->p.force_scale, d_dVds + dim, (T *)d_F);
            c->launches++;
        } else if (d.kind == METAD_CV_CONTACTS) {
            k_contacts_force<T><<<div_up((long long)d.ncatoms * 32, 128), 128, 0, c->stream>>>(
                d.ncatoms, d.d_catoms, d.d_csr_off, d.d_csr_pair, d.d_pairs, d.d_pair_r0, d.n, d.m,
                c->p.force_scale * d.scale, pos, c->boxd, d_dVds + dim, (T *)d_F, c->dg);
            c->launches++;
        }
    }
    return METAD_OK;
}

int chain_forces(metad_ctx *c, const double *d_dVds, void *d_F) {
    return c->prec == 32 ? chain_forces_t<float>(c, d_dVds, d_F) : chain_forces_t<double>(c, d_dVds, d_F);
}


// ------------------------------------------------------------------------------------------------
// NEXT-1: torsion CVs (reading V).  One thread per torsion dimension evaluates the angle and
// keeps the gradient of its four atoms; the force kernel is gather form (thread per touched atom, fixed
// summation order over dimensions and slots, no atomics).
struct TorsTable { int kind[METAD_MAX_CV]; int idx[METAD_MAX_CV][4]; };

template <typename T>
__global__ void k_torsions_cv(int D, TorsTable tt, const T *__restrict__ pos, BoxD bd, double *__restrict__ grad,
                              double *__restrict__ cv_out, unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg) {
    if (dg) bd = dg->bd;                          // device-resident box (NPT): metad_*_dev
    const int d = threadIdx.x;
    if (d >= D || tt.kind[d] != METAD_CV_TORSION) return;
    double r[4][3], b[3][3];
    for (int k = 0; k < 4; ++k)
        for (int a = 0; a < 3; ++a) r[k][a] = (double)pos[3 * (size_t)tt.idx[d][k] + a];
    for (int k = 0; k < 3; ++k) {
        b[k][0] = r[k + 1][0] - r[k][0]; b[k][1] = r[k + 1][1] - r[k][1]; b[k][2] = r[k + 1][2] - r[k][2];
        min_image_d(bd, b[k][0], b[k][1], b[k][2]);
    }
    double g[12];
    const double phi = torsion_eval(b[0], b[1], b[2], g);
    for (int k = 0; k < 12; ++k) grad[12 * d + k] = g[k];
    cv_out[d] = phi;
    if (!isfinite(phi)) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
}

template <typename T>
__global__ void k_torsions_force(int D, TorsTable tt, int natoms_touched, const int *__restrict__ atoms,
                                 const double *__restrict__ grad, double force_scale, const double *__restrict__ dVds,
                                 T *__restrict__ F) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= natoms_touched) return;
    const int a = atoms[t];
    double f[3] = { 0.0, 0.0, 0.0 };
    for (int d = 0; d < D; ++d) {
        if (tt.kind[d] != METAD_CV_TORSION) continue;
        const double w = dVds[d];
        for (int k = 0; k < 4; ++k)
            if (tt.idx[d][k] == a) { f[0] += w * grad[12 * d + 3 * k]; f[1] += w * grad[12 * d + 3 * k + 1]; f[2] += w * grad[12 * d + 3 * k + 2]; }
    }
    F[3 * (size_t)a] += (T)(-force_scale * f[0]);
    F[3 * (size_t)a + 1] += (T)(-force_scale * f[1]);
    F[3 * (size_t)a + 2] += (T)(-force_scale * f[2]);
}

static TorsTable tors_table(const metad_ctx *c) {
    TorsTable tt;
    for (int d = 0; d < METAD_MAX_CV; ++d) {
        tt.kind[d] = d < c->D ? c->cv[d].kind : -1;
        for (int k = 0; k < 4; ++k) tt.idx[d][k] = d < c->D ? c->cv[d].tors[k] : 0;
    }
    return tt;
}

int torsion_eval_all(metad_ctx *c, double *d_cv) {
    if (!c->has_torsion) return METAD_OK;
    if (c->prec == 32)
        k_torsions_cv<float><<<1, 32, 0, c->stream>>>(c->D, tors_table(c), (const float *)ctx_last_pos(c), c->boxd, c->d_tors_grad, d_cv, c->d_sticky, c->dg);
    else
        k_torsions_cv<double><<<1, 32, 0, c->stream>>>(c->D, tors_table(c), (const double *)ctx_last_pos(c), c->boxd, c->d_tors_grad, d_cv, c->d_sticky, c->dg);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int torsion_forces(metad_ctx *c, const double *d_dVds, void *d_F) {
    if (!c->has_torsion) return METAD_OK;
    if (c->prec == 32)
        k_torsions_force<float><<<1, 32, 0, c->stream>>>(c->D, tors_table(c), c->ntors_atoms, c->d_tors_atoms, c->d_tors_grad, c->p.force_scale, d_dVds, (float *)d_F);
    else
        k_torsions_force<double><<<1, 32, 0, c->stream>>>(c->D, tors_table(c), c->ntors_atoms, c->d_tors_atoms, c->d_tors_grad, c->p.force_scale, d_dVds, (double *)d_F);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}


// ------------------------------------------------------------------------------------------------
// NEXT-3: lattice-parameter CVs (reading AB): s = |h_k|; the bias force acts on the box rows.
struct LatTable { int kind[METAD_MAX_CV]; int axis[METAD_MAX_CV]; double h[9]; };

__global__ void k_lattice_cv(int D, LatTable lt, double *__restrict__ cv_out, const DevGeom *__restrict__ dg) {
    if (dg) { for (int k = 0; k < 9; ++k) lt.h[k] = dg->box[k]; }   // device-resident box
    const int d = threadIdx.x;
    if (d >= D || lt.kind[d] != METAD_CV_LATTICE) return;
    const double *h = lt.h + 3 * lt.axis[d];
    cv_out[d] = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
}

__global__ void k_lattice_force(int D, LatTable lt, double force_scale, const double *__restrict__ dVds,
                                double *__restrict__ fbox, double *__restrict__ virial /* NULL: not wanted */, const DevGeom *__restrict__ dg) {
    if (dg) { for (int k = 0; k < 9; ++k) lt.h[k] = dg->box[k]; }   // device-resident box
    const int e = threadIdx.x;              // box element (row, component)
    if (e >= 9) return;
    const int row = e / 3;
    if (virial) {                           // d|h_k|/d eps_ab = h_a h_b / |h_k| (reading AD); e = (a, b)
        double w = 0.0;
        for (int d = 0; d < D; ++d) {
            if (lt.kind[d] != METAD_CV_LATTICE) continue;
            const double *h = lt.h + 3 * lt.axis[d];
            w += dVds[d] * h[e / 3] * h[e % 3] / sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
        }
        virial[e] += -force_scale * w;
    }
    double f = 0.0;
    for (int d = 0; d < D; ++d) {
        if (lt.kind[d] != METAD_CV_LATTICE || lt.axis[d] != row) continue;
        const double *h = lt.h + 3 * row;
        f += dVds[d] * h[e - 3 * row] / sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
    }
    fbox[e] = -force_scale * f;
}

static LatTable lat_table(const metad_ctx *c) {
    LatTable lt;
    for (int d = 0; d < METAD_MAX_CV; ++d) { lt.kind[d] = d < c->D ? c->cv[d].kind : -1; lt.axis[d] = d < c->D ? c->cv[d].n : 0; }
    const BoxD &b = c->boxd;
    const double h[9] = { b.ax, 0.0, 0.0, b.bx, b.by, 0.0, b.cx, b.cy, b.cz };
    for (int k = 0; k < 9; ++k) lt.h[k] = h[k];
    return lt;
}

int lattice_eval(metad_ctx *c, double *d_cv) {
    if (!c->has_lattice) return METAD_OK;
    k_lattice_cv<<<1, 32, 0, c->stream>>>(c->D, lat_table(c), d_cv, c->dg);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int lattice_forces(metad_ctx *c, const double *d_dVds) {
    if (!c->has_lattice) return METAD_OK;
    k_lattice_force<<<1, 32, 0, c->stream>>>(c->D, lat_table(c), c->p.force_scale, d_dVds, c->d_box_force,
                                            c->p.want_virial ? c->d_virial : nullptr, c->dg);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}


// ------------------------------------------------------------------------------------------------
// Bias virial of the chain / torsion CVs (reading AD), only launched with params.want_virial.  One block each; the
// sums are short (<= a few thousand terms) and taken in a fixed order.
__global__ void __launch_bounds__(256)
k_rgyr_virial(int nchain, const double *__restrict__ mass, const double *__restrict__ unwrapped, double force_scale,
              const double *__restrict__ dVds, double *__restrict__ virial) {
    __shared__ double red[9 * 32];
    const RgScratch *sc = reinterpret_cast<const RgScratch *>(unwrapped + 3 * (size_t)nchain);
    double w[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) w[q] = 0.0;
    for (int k = threadIdx.x; k < nchain; k += blockDim.x) {
        const double mk = mass ? mass[k] : 1.0;
        const double u[3] = { unwrapped[3 * k] - sc->com[0], unwrapped[3 * k + 1] - sc->com[1], unwrapped[3 * k + 2] - sc->com[2] };
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) w[3 * a + b] += mk * u[a] * u[b];
    }
    block_reduce<9>(w, red);
    if (threadIdx.x == 0 && sc->rg > 0.0) {
        const double f = -force_scale * dVds[0] / (sc->M * sc->rg);      // d Rg/d eps = sum m u u^T / (M Rg)
        for (int q = 0; q < 9; ++q) virial[q] += f * w[q];
    }
}

template <typename T>
__global__ void __launch_bounds__(256)
k_contacts_virial(int npairs, const int *__restrict__ pairs, const double *__restrict__ pair_r0, int n, int m,
                  double coef /* force_scale * scale */, const T *__restrict__ pos, BoxD bd, const double *__restrict__ dVds,
                  double *__restrict__ virial, const DevGeom *__restrict__ dg) {
    if (dg) bd = dg->bd;                          // device-resident box (NPT): metad_*_dev
    __shared__ double red[9 * 32];
    double w[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) w[q] = 0.0;
    for (int p = threadIdx.x; p < npairs; p += blockDim.x) {
        const int i = pairs[2 * p], j = pairs[2 * p + 1];
        double d[3] = { (double)pos[3 * j] - (double)pos[3 * i], (double)pos[3 * j + 1] - (double)pos[3 * i + 1],
                        (double)pos[3 * j + 2] - (double)pos[3 * i + 2] };
        min_image_d(bd, d[0], d[1], d[2]);
        const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double dsw;
        switch_d(r / pair_r0[p], n, m, dsw);
        const double g = dsw / (pair_r0[p] * r);
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) w[3 * a + b] += g * d[a] * d[b];
    }
    block_reduce<9>(w, red);
    if (threadIdx.x == 0) {
        const double f = -coef * dVds[0];
        for (int q = 0; q < 9; ++q) virial[q] += f * w[q];
    }
}

// d phi/d eps = sum_k (d phi/d b_k) b_k^T,  d phi/d b1 = -g_i, d phi/d b2 = -(g_i + g_j), d phi/d b3 = g_l
template <typename T>
__global__ void k_torsions_virial(int D, TorsTable tt, const T *__restrict__ pos, BoxD bd, const double *__restrict__ grad,
                                  double force_scale, const double *__restrict__ dVds, double *__restrict__ virial, const DevGeom *__restrict__ dg) {
    if (dg) bd = dg->bd;                          // device-resident box (NPT): metad_*_dev
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    for (int d = 0; d < D; ++d) {
        if (tt.kind[d] != METAD_CV_TORSION) continue;
        double b[3][3];
        for (int k = 0; k < 3; ++k) {
            for (int a = 0; a < 3; ++a)
                b[k][a] = (double)pos[3 * (size_t)tt.idx[d][k + 1] + a] - (double)pos[3 * (size_t)tt.idx[d][k] + a];
            min_image_d(bd, b[k][0], b[k][1], b[k][2]);
        }
        const double *g = grad + 12 * d;
        const double f = -force_scale * dVds[d];
        for (int a = 0; a < 3; ++a)
            for (int c = 0; c < 3; ++c)
                virial[3 * a + c] += f * (-g[a] * b[0][c] - (g[a] + g[3 + a]) * b[1][c] + g[9 + a] * b[2][c]);
    }
}

template <typename T>
static int chain_virial_t(metad_ctx *c, const double *d_dVds) {
    const T *pos = (const T *)ctx_last_pos(c);
    for (int dim = 0; dim < c->D; ++dim) {
        CvDev &d = c->cv[dim];
        if (d.kind == METAD_CV_RGYR) {
            k_rgyr_virial<<<1, 256, 0, c->stream>>>(d.nchain, d.d_mass, d.d_unwrapped, c->p.force_scale, d_dVds + dim, c->d_virial);
            c->launches++;
        } else if (d.kind == METAD_CV_CONTACTS) {
            k_contacts_virial<T><<<1, 256, 0, c->stream>>>(d.npairs, d.d_pairs, d.d_pair_r0, d.n, d.m, c->p.force_scale * d.scale,
                                                           pos, c->boxd, d_dVds + dim, c->d_virial, c->dg);
            c->launches++;
        }
    }
    if (c->has_torsion) {
        k_torsions_virial<T><<<1, 32, 0, c->stream>>>(c->D, tors_table(c), pos, c->boxd, c->d_tors_grad, c->p.force_scale, d_dVds,
                                                      c->d_virial, c->dg);
        c->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int chain_virial(metad_ctx *c, const double *d_dVds) {
    if (!c->p.want_virial) return METAD_OK;
    return c->prec == 32 ? chain_virial_t<float>(c, d_dVds) : chain_virial_t<double>(c, d_dVds);
}
