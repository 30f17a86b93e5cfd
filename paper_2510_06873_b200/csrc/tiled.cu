// tiled.cu — fp32 fast path of a1 (neighbour list), a3 (Q6 pass 1) and a6 (Q6 forces) on
// shared-memory tiles of the cell grid (tile.cuh).  One block per tile; one thread per own atom.
//   k_tile_build     candidates read from shared memory, no per-pair minimum image; pairs within a
//                    1e-5 band of rc^2 are re-decided with the canonical fp64 predicate (reading O)
//   k_tile_q6_pass1  neighbour positions gathered from shared memory (LDS)
//   k_tile_q6_force  neighbour positions AND 64-byte q6 records gathered from shared memory
#include "common.cuh"
#include "cv_q6.cuh"
#include "tile.cuh"

typedef unsigned short nl16_t;

// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TILE_THREADS)
k_tile_build(TileGeom g, const float4 *__restrict__ spos, const int *__restrict__ scell,
             const int *__restrict__ cell_start, BoxD bd, float rc2f, double rc2, int maxn,
             int *__restrict__ nl_count, nl16_t *__restrict__ nl, unsigned int *__restrict__ sticky) {
    extern __shared__ float4 dyn_smem[];
    __shared__ TileTables t;
    float4 *pos_s = dyn_smem;
    tile_setup(g, cell_start, t);
    tile_stage_pos(t, spos, pos_s);
    __syncthreads();
    if (t.total > 65535) { if (threadIdx.x == 0) atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW); return; }
    const float band = 1e-5f * rc2f;
    for (int a = threadIdx.x; a < t.nown; a += blockDim.x) {
        const int q = tile_own_row(t, a);
        const int o = a - t.own_off[q];
        const int li = t.own_l[q] + o, s = t.own_g[q] + o;
        const float4 pi = tile_pos(t, spos, pos_s, li);
        const int ix = scell[s] % g.nc0;
        const int ic = ix - t.x0 + 1;                       // halo-cell column of the own atom
        const int r0 = t.own_row[q];
        int cnt = 0;
#pragma unroll 1
        for (int dz = -1; dz <= 1; ++dz) {
#pragma unroll 1
            for (int dy = -1; dy <= 1; ++dy) {
                const int r = r0 + dz * (t.Tye + 2) + dy;
                const int lo = t.hcell[r][ic - 1], hi = t.hcell[r][ic + 2];
                for (int lj = lo; lj < hi; ++lj) {
                    const float4 pj = tile_pos(t, spos, pos_s, lj);
                    const float dx = pj.x - pi.x, dy2 = pj.y - pi.y, dz2 = pj.z - pi.z;
                    const float r2 = dx * dx + dy2 * dy2 + dz2 * dz2;
                    bool in = r2 < rc2f;
                    if (fabsf(r2 - rc2f) <= band) {         // borderline: canonical fp64 predicate on the inputs
                        const float4 gi = spos[s], gj = spos[__float_as_int(pj.w)];
                        in = r2_canonical(bd, (double)gj.x - (double)gi.x, (double)gj.y - (double)gi.y,
                                          (double)gj.z - (double)gi.z) < rc2;
                    }
                    if (in && lj != li) {
                        if (cnt < maxn) nl[nl_slot(s, cnt, maxn)] = (nl16_t)lj;
                        ++cnt;
                    }
                }
            }
        }
        if (cnt > maxn) { atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW); cnt = maxn; }
        nl_count[s] = cnt;
    }
}

// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TILE_THREADS)
k_tile_q6_pass1(TileGeom g, const float4 *__restrict__ spos, const int *__restrict__ cell_start, int maxn,
                const int *__restrict__ nl_count, const nl16_t *__restrict__ nl, float q_thresh, float inv_width,
                float *__restrict__ rec, double scale_mean, double scale_solid, int dim_mean, int dim_solid,
                double *__restrict__ partials, unsigned int *__restrict__ ticket, double *__restrict__ cv_out,
                unsigned int *__restrict__ sticky) {
    extern __shared__ float4 dyn_smem[];
    __shared__ TileTables t;
    __shared__ double red[64];
    float4 *pos_s = dyn_smem;
    tile_setup(g, cell_start, t);
    tile_stage_pos(t, spos, pos_s);
    __syncthreads();
    double v[2] = { 0.0, 0.0 };
    for (int a = threadIdx.x; a < t.nown; a += blockDim.x) {
        const int q = tile_own_row(t, a);
        const int o = a - t.own_off[q];
        const int li = t.own_l[q] + o, s = t.own_g[q] + o;
        const float4 pi = tile_pos(t, spos, pos_s, li);
        float A[13];
#pragma unroll
        for (int k = 0; k < 13; ++k) A[k] = 0.f;
        const int cnt = nl_count[s];
        for (int k = 0; k < cnt; ++k) {
            const int lj = nl[nl_slot(s, k, maxn)];
            const float4 pj = tile_pos(t, spos, pos_s, lj);
            const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
            const float rinv = rsqrtf(dx * dx + dy * dy + dz * dz);
            Y6<float> y;
            y6_eval<float>(dx * rinv, dy * rinv, dz * rinv, y);
            A[0] += y.E[0];
#pragma unroll
            for (int m = 1; m <= 6; ++m) { A[2 * m - 1] += y.E[m] * y.c[m]; A[2 * m] += y.E[m] * y.s[m]; }
        }
        float S = 0.f;
#pragma unroll
        for (int k = 0; k < 13; ++k) S += A[k] * A[k];
        float q6 = 0.f, norm = 0.f;
        if (cnt > 0 && S > 0.f) { float rs = sqrtf(S); q6 = rs / (float)cnt; norm = 1.f / ((float)cnt * rs); }
        const float f = 1.f / (1.f + expf(-(q6 - q_thresh) * inv_width));
        float4 *r4 = reinterpret_cast<float4 *>(rec + (size_t)s * METAD_NREC);
        r4[0] = make_float4(A[0] * norm, A[1] * norm, -A[2] * norm, A[3] * norm);
        r4[1] = make_float4(-A[4] * norm, A[5] * norm, -A[6] * norm, A[7] * norm);
        r4[2] = make_float4(-A[8] * norm, A[9] * norm, -A[10] * norm, A[11] * norm);
        r4[3] = make_float4(-A[12] * norm, f * (1.f - f) * inv_width, q6, 0.f);
        v[0] += (double)q6; v[1] += (double)f;
    }
    block_reduce<2>(v, red);
    if (threadIdx.x == 0) { partials[2 * blockIdx.x] = v[0]; partials[2 * blockIdx.x + 1] = v[1]; }
    if (last_block_ticket(ticket)) {
        double u[2] = { 0.0, 0.0 };
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) { u[0] += partials[2 * b]; u[1] += partials[2 * b + 1]; }
        block_reduce<2>(u, red);
        if (threadIdx.x == 0) {
            double a = scale_mean * u[0], b = scale_solid * u[1];
            if (dim_mean >= 0) cv_out[dim_mean] = a;
            if (dim_solid >= 0) cv_out[dim_solid] = b;
            if (!isfinite(a) || !isfinite(b)) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// record chunk c (16 B) of halo atom li lives at rec_s[4*li + (c ^ swz(li))]: spreads the 64-byte
// records of different atoms over all bank groups for the per-lane LDS.128 gathers
__device__ __forceinline__ int rec_slot(int li, int c) { return 4 * li + (c ^ ((li >> 1) & 3)); }

__global__ void __launch_bounds__(TILE_THREADS)
k_tile_q6_force(TileGeom g, const float4 *__restrict__ spos, const int *__restrict__ cell_start, int maxn,
                const int *__restrict__ nl_count, const nl16_t *__restrict__ nl, const int *__restrict__ perm,
                const float *__restrict__ rec, double scale_mean, double scale_solid, int dim_mean, int dim_solid,
                double force_scale, const double *__restrict__ dVds, float *__restrict__ F) {
    extern __shared__ float4 dyn_smem[];
    __shared__ TileTables t;
    tile_setup(g, cell_start, t);
    float4 *pos_s = dyn_smem;
    float4 *rec_s = dyn_smem + g.cap;
    tile_stage_pos(t, spos, pos_s);
    const float4 *rec4 = reinterpret_cast<const float4 *>(rec);
    if (t.staged) {
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
        for (int sg = wid; sg < 3 * t.nrows; sg += nw) {
            const int n4 = 4 * t.seg_len[sg], g0 = t.seg_g[sg], l0 = t.seg_off[sg];
            for (int i = lane; i < n4; i += 32) rec_s[rec_slot(l0 + (i >> 2), i & 3)] = rec4[(size_t)4 * g0 + i];
        }
    }
    __syncthreads();
    const float alpha = dim_mean >= 0 ? (float)(dVds[dim_mean] * scale_mean) : 0.f;
    const float beta = dim_solid >= 0 ? (float)(dVds[dim_solid] * scale_solid) : 0.f;
    for (int a = threadIdx.x; a < t.nown; a += blockDim.x) {
        const int q = tile_own_row(t, a);
        const int o = a - t.own_off[q];
        const int li = t.own_l[q] + o, s = t.own_g[q] + o;
        const float4 pi = tile_pos(t, spos, pos_s, li);
        float Bk[13];
        {
            const float4 a4 = rec4[(size_t)4 * s], b4 = rec4[(size_t)4 * s + 1], c4 = rec4[(size_t)4 * s + 2],
                         d4 = rec4[(size_t)4 * s + 3];
            const float gk = alpha + beta * d4.y;
            Bk[0] = gk * a4.x; Bk[1] = gk * a4.y; Bk[2] = gk * a4.z; Bk[3] = gk * a4.w;
            Bk[4] = gk * b4.x; Bk[5] = gk * b4.y; Bk[6] = gk * b4.z; Bk[7] = gk * b4.w;
            Bk[8] = gk * c4.x; Bk[9] = gk * c4.y; Bk[10] = gk * c4.z; Bk[11] = gk * c4.w;
            Bk[12] = gk * d4.x;
        }
        float fx = 0.f, fy = 0.f, fz = 0.f;
        const int cnt = nl_count[s];
        for (int k = 0; k < cnt; ++k) {
            const int lj = nl[nl_slot(s, k, maxn)];
            float4 pj, a4, b4, c4, d4;
            if (t.staged) {
                pj = pos_s[lj];
                a4 = rec_s[rec_slot(lj, 0)]; b4 = rec_s[rec_slot(lj, 1)]; c4 = rec_s[rec_slot(lj, 2)]; d4 = rec_s[rec_slot(lj, 3)];
            } else {
                pj = tile_pos(t, spos, pos_s, lj);
                const size_t gj = (size_t)__float_as_int(pj.w);
                a4 = rec4[4 * gj]; b4 = rec4[4 * gj + 1]; c4 = rec4[4 * gj + 2]; d4 = rec4[4 * gj + 3];
            }
            const float gj_w = alpha + beta * d4.y;
            float bb[13];
            bb[0] = Bk[0] + gj_w * a4.x; bb[1] = Bk[1] + gj_w * a4.y; bb[2] = Bk[2] + gj_w * a4.z; bb[3] = Bk[3] + gj_w * a4.w;
            bb[4] = Bk[4] + gj_w * b4.x; bb[5] = Bk[5] + gj_w * b4.y; bb[6] = Bk[6] + gj_w * b4.z; bb[7] = Bk[7] + gj_w * b4.w;
            bb[8] = Bk[8] + gj_w * c4.x; bb[9] = Bk[9] + gj_w * c4.y; bb[10] = Bk[10] + gj_w * c4.z; bb[11] = Bk[11] + gj_w * c4.w;
            bb[12] = Bk[12] + gj_w * d4.x;
            const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
            const float rinv = rsqrtf(dx * dx + dy * dy + dz * dz);
            const float ux = dx * rinv, uy = dy * rinv, uz = dz * rinv;
            Y6<float> y;
            y6_eval<float>(ux, uy, uz, y);
            float gx, gy, gz;
            y6_grad<float>(y, bb, gx, gy, gz);
            const float gu = gx * ux + gy * uy + gz * uz;
            fx += (gx - gu * ux) * rinv; fy += (gy - gu * uy) * rinv; fz += (gz - gu * uz) * rinv;
        }
        const int i = perm[s];
        F[3 * i] += (float)(force_scale * (double)fx);
        F[3 * i + 1] += (float)(force_scale * (double)fy);
        F[3 * i + 2] += (float)(force_scale * (double)fz);
    }
}

// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(TILE_THREADS)
k_tile_export(TileGeom g, const int *__restrict__ cell_start, int maxn, const int *__restrict__ perm,
              const int *__restrict__ nl_count, const nl16_t *__restrict__ nl, int *__restrict__ out_count,
              int *__restrict__ out_list) {
    __shared__ TileTables t;
    tile_setup(g, cell_start, t);
    for (int a = threadIdx.x; a < t.nown; a += blockDim.x) {
        const int q = tile_own_row(t, a);
        const int o = a - t.own_off[q];
        const int s = t.own_g[q] + o, i = perm[s], cnt = nl_count[s];
        out_count[i] = cnt;
        for (int k = 0; k < maxn; ++k)
            out_list[(size_t)i * maxn + k] = k < cnt ? perm[tile_global_of(t, nl[nl_slot(s, k, maxn)])] : -1;
    }
}

// ------------------------------------------------------------------------------------------------
// host side
TileGeom tile_geom(const metad_ctx *c);        // api.cu

static size_t smem_pos(const TileGeom &g) { return sizeof(float4) * (size_t)g.cap; }
static size_t smem_force(const TileGeom &g) { return sizeof(float4) * (size_t)g.cap * 5; }

int tiled_init() {
    static bool done = false;
    if (done) return METAD_OK;
    CUDA_TRY(cudaFuncSetAttribute(k_tile_q6_force, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    CUDA_TRY(cudaFuncSetAttribute(k_tile_q6_pass1, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    done = true;
    return METAD_OK;
}

int tiled_build(metad_ctx *c) {
    TileGeom g = tile_geom(c);
    int nt = g.ntx * g.nty * g.ntz;
    k_tile_build<<<nt, TILE_THREADS, smem_pos(g), c->stream>>>(g, (const float4 *)c->d_spos, c->d_scell, c->d_cell_start,
                                                            c->boxd, (float)c->rc2, c->rc2, c->maxn, c->d_nl_count,
                                                            (nl16_t *)c->d_nl, c->d_sticky);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int tiled_q6_pass1(metad_ctx *c, double *d_cv) {
    TileGeom g = tile_geom(c);
    int nt = g.ntx * g.nty * g.ntz;
    double sm = c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0;
    double ss = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0;
    double qt = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_thresh : 0.0;
    double qw = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_width : 1.0;
    k_tile_q6_pass1<<<nt, TILE_THREADS, smem_pos(g), c->stream>>>(g, (const float4 *)c->d_spos, c->d_cell_start, c->maxn,
                                                               c->d_nl_count, (const nl16_t *)c->d_nl, (float)qt,
                                                               (float)(1.0 / qw), (float *)c->d_rec, sm, ss, c->q6_mean_dim,
                                                               c->q6_solid_dim, c->d_partials + c->nblocks_atoms,
                                                               c->d_tickets + 1, d_cv, c->d_sticky);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int tiled_q6_force(metad_ctx *c, const double *d_dVds, void *d_F) {
    TileGeom g = tile_geom(c);
    int nt = g.ntx * g.nty * g.ntz;
    double sm = c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0;
    double ss = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0;
    k_tile_q6_force<<<nt, TILE_THREADS, smem_force(g), c->stream>>>(g, (const float4 *)c->d_spos, c->d_cell_start, c->maxn,
                                                                 c->d_nl_count, (const nl16_t *)c->d_nl, c->d_perm,
                                                                 (const float *)c->d_rec, sm, ss, c->q6_mean_dim,
                                                                 c->q6_solid_dim, c->p.force_scale, d_dVds, (float *)d_F);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int tiled_export(metad_ctx *c, int *d_count, int *d_list) {
    TileGeom g = tile_geom(c);
    int nt = g.ntx * g.nty * g.ntz;
    k_tile_export<<<nt, TILE_THREADS, 0, c->stream>>>(g, c->d_cell_start, c->maxn, c->d_perm, c->d_nl_count,
                                                     (const nl16_t *)c->d_nl, d_count, d_list);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
