// tiled64.cu — the fp64 counterpart of tiled.cu: a1 (neighbour list) fused with a3 (Q6 pass 1) on shared-memory tiles of the
// cell grid (tile.cuh) for contexts with fp64 pair math (reading R: the parity precision of configs 0-3).  One block per
// tile, one thread per own atom, the same two passes as the fp32 kernel:
//   scan    every halo atom of the 3 x 3 row-runs around the atom's cell with r^2 < rc^2 (1 + 1e-9) goes to a per-thread
//           candidate list in shared memory (uint16 local indices);
//   finish  the exact decision on that short list — pairs within the 1e-9 band of rc^2 are re-decided with the canonical
//           predicate of reading O on the original coordinates, so the sets are bit-exact —, the neighbour-list write and
//           the atom's 13 q6m components by the Y6m recurrence, all in fp64.
// What differs from the fp32 kernel: the halo is staged (as a structure of arrays) in RAW coordinates (plus the lattice shift of a periodic image,
// added once): in fp64 there is no exactness to gain from tile-local coordinates, and for a pair inside the primary cell
// pj - pi is then the very difference the canonical predicate forms.  The OUTPUT keeps the formats of the generic fp64
// kernels — list nl[k N + s] of plain sorted indices, records [N][16] = 13 components + position, q6 | f'(q6) arrays — so that every
// downstream kernel (k_q6_force<double>, the virial instance, the exports, metad_cv_owned_sum) runs unchanged: this
// kernel replaces k_build_list<double> + k_q6_pass1<double> (0.35 + 0.26 ms at 1,024,000 atoms) and nothing else.
#include <algorithm>
#include "common.cuh"
#include "cv_q6.cuh"
#include "tile.cuh"

typedef unsigned short nl16_t;   // local halo index (shared-memory candidate list only)
#define LIST_CAP64 40            // per-thread candidate slots (maxn <= 32 on this path + band + self)
#define TILE64_MINB 3            // resident blocks per SM: 34 KB of staged positions + 20 KB of candidate lists + tables

// Shared-memory staging area, structure of arrays: (x, y) pairs, z and the global sorted index of every halo atom.  An array of
// double4 would put the 16 bytes a lane reads at a 32-byte stride: two-way bank conflicts on the 128-bit load and four-way on
// the 64-bit one (profiles/r2l_fp64.md: the scan sat at 77 % of the shared-memory wavefronts); with 16- and 8-byte strides both
// loads are conflict-free.
struct Stage64 { double2 *xy; double *z; int *idx; };
#define STAGE64_BYTES 28         // per staged atom
struct P64 { double x, y, z; int j; };

// staged position of a halo atom: (x, y, z) of the image this tile sees, .w = its global sorted index
__device__ __forceinline__ double4 tile_transform64(const TileGeom &g, const TileTables &t, int seg, double4 p, int gidx,
                                                    const DevGeom *dg) {
    if (t.seg_wrapped[seg]) {                  // periodic image: the lattice shift is added once, here
        const int code = t.seg_code[seg];
        const int wx = code % 3 - 1, wy = (code / 3) % 3 - 1, wz = code / 9 - 1;
        const TileBox b = tile_box(g, dg);
        p.x += wx * b.ax + wy * b.bx + wz * b.cx;
        p.y += wy * b.by + wz * b.cy;
        p.z += wz * b.cz;
    }
    p.w = (double)gidx;
    return p;
}

__device__ __forceinline__ void tile_stage_pos64(const TileGeom &g, const TileTables &t, const double4 *__restrict__ spos,
                                                 const Stage64 &pos_s, const DevGeom *dg) {
    if (!t.staged) return;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int s = wid; s < 3 * t.nrows; s += nw) {
        const int len = t.seg_len[s], g0 = t.seg_g[s], l0 = t.seg_off[s];
        for (int i = lane; i < len; i += 32) {
            const double4 p = tile_transform64(g, t, s, ldg4<double>(spos + g0 + i), g0 + i, dg);
            pos_s.xy[l0 + i] = make_double2(p.x, p.y);
            pos_s.z[l0 + i] = p.z;
            pos_s.idx[l0 + i] = g0 + i;
        }
    }
}

template <bool STAGED>
__device__ __forceinline__ P64 hpos64(const TileGeom &g, const TileTables &t, const double4 *__restrict__ spos,
                                      const Stage64 &pos_s, int li, const DevGeom *dg) {
    P64 o;
    if (STAGED) {
        const double2 xy = pos_s.xy[li];
        o.x = xy.x; o.y = xy.y; o.z = pos_s.z[li]; o.j = pos_s.idx[li];
        return o;
    }
    const int s = tile_seg_of(t, li);          // halo larger than the staging area: global memory, segment by binary search
    const int gi = t.seg_g[s] + (li - t.seg_off[s]);
    const double4 p = tile_transform64(g, t, s, spos[gi], gi, dg);
    o.x = p.x; o.y = p.y; o.z = p.z; o.j = gi;
    return o;
}

// candidate scan of own atom a into list column `col`; returns the number of candidates kept
template <bool STAGED>
__device__ __forceinline__ int scan_atom64(const TileGeom &g, const TileTables &t, const double4 *__restrict__ spos,
                                           const Stage64 &pos_s, nl16_t *list_s, const int *__restrict__ scell, int a, int col,
                                           double rc2_hi, bool &ovf, const DevGeom *dg) {
    const int q = tile_own_row(t, a);
    const int o = a - t.own_off[q];
    const int li = t.own_l[q] + o, s = t.own_g[q] + o;
    const P64 pi = hpos64<STAGED>(g, t, spos, pos_s, li, dg);
    const int ic = scell[s] % g.nc0 - t.x0 + g.hx;       // halo-cell column of the own atom
    const int r0 = t.own_row[q], rstride = t.Tye + 2;
    const unsigned STRIDE = TILE_THREADS * (unsigned)sizeof(nl16_t);
    const unsigned w0 = (unsigned)__cvta_generic_to_shared(list_s + col);
    unsigned wp = w0;
    const unsigned wend = w0 + (LIST_CAP64 - 1) * STRIDE;
#pragma unroll 1
    for (int dz = -1; dz <= 1; ++dz) {
#pragma unroll 1
        for (int dy = -1; dy <= 1; ++dy) {
            const int r = r0 + dz * rstride + dy;
            int lo = t.hcell[r][ic - g.hx];
            const int hi = t.hcell[r][ic + g.hx + 1];
            while (lo < hi) {
                // every candidate is stored and the slot kept only if it passes; capacity is checked once per stretch
                const int room = (int)((wend - wp) / STRIDE);
                if (room <= 0) { ovf = true; break; }
                const int h2 = min(hi, lo + room);
#pragma unroll 2
                for (int lj = lo; lj < h2; ++lj) {
                    // staged: one 128-bit and one 64-bit conflict-free shared-memory load; the index is read by the exact pass only
                    double ex, ey, ez;
                    if (STAGED) {
                        const double2 xy = pos_s.xy[lj];
                        ex = xy.x - pi.x; ey = xy.y - pi.y; ez = pos_s.z[lj] - pi.z;
                    } else {
                        const P64 pj = hpos64<STAGED>(g, t, spos, pos_s, lj, dg);
                        ex = pj.x - pi.x; ey = pj.y - pi.y; ez = pj.z - pi.z;
                    }
                    const double r2 = fma(ez, ez, fma(ey, ey, ex * ex));
                    asm volatile("st.shared.u16 [%0], %1;" ::"r"(wp), "h"((unsigned short)lj));
                    asm volatile("{ .reg .pred p; setp.lt.f64 p, %1, %2; @p add.u32 %0, %0, %3; }"
                                 : "+r"(wp) : "d"(r2), "d"(rc2_hi), "r"(STRIDE));
                }
                lo = h2;
            }
        }
    }
    return (int)((wp - w0) / STRIDE);
}

// exact decision on the short list, neighbour-list write (generic layout), q6m accumulation, record; returns q6 and f(q6)
template <bool STAGED>
__device__ __forceinline__ void finish_atom64(const TileGeom &g, const TileTables &t, const double4 *__restrict__ spos,
                                              const Stage64 &pos_s, const nl16_t *list_s, int a, int col, int cnt, bool ovf,
                                              const BoxD &bd, double rc2, double rc2_lo, int maxn, int *__restrict__ nl_count,
                                              int *__restrict__ nl, unsigned int *__restrict__ sticky, double q_thresh,
                                              double inv_width, double *__restrict__ rec, double *__restrict__ q6arr,
                                              const DevGeom *__restrict__ dg,
                                              double &q6_out, double &f_out) {
    const int q = tile_own_row(t, a);
    const int o = a - t.own_off[q];
    const int li = t.own_l[q] + o, s = t.own_g[q] + o;
    const size_t N = (size_t)g.natoms;
    const P64 pi = hpos64<STAGED>(g, t, spos, pos_s, li, dg);
    const nl16_t *myl = list_s + col;
    if (ovf) atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW);
    double A[13];
#pragma unroll
    for (int k = 0; k < 13; ++k) A[k] = 0.0;
    int n = 0;
    for (int k = 0; k < cnt; ++k) {
        const int lj = myl[k * TILE_THREADS];
        if (lj == li) continue;
        const P64 pj = hpos64<STAGED>(g, t, spos, pos_s, lj, dg);
        const double dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        const double r2 = dx * dx + dy * dy + dz * dz;
        const int j = pj.j;
        bool in = r2 < rc2;
        if (r2 >= rc2_lo) {                                // borderline: canonical predicate on the original coordinates
            const double4 gi = spos[s], gj = spos[j];
            in = r2_canonical(dg ? dg->bd : bd, gj.x - gi.x, gj.y - gi.y, gj.z - gi.z) < rc2;
        }
        if (!in) continue;
        if (n < maxn) {
            nl[(size_t)n * N + s] = j;
            const double rinv = 1.0 / sqrt(r2);
            Y6<double> y;
            y6_eval<double>(dx * rinv, dy * rinv, dz * rinv, y);
            A[0] += y.E[0];
#pragma unroll
            for (int m = 1; m <= 6; ++m) {
                A[2 * m - 1] += y.E[m] * y.c[m];
                A[2 * m] += y.E[m] * y.s[m];
            }
        }
        ++n;
    }
    if (n > maxn) { atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW); n = maxn; }
    nl_count[s] = n;
    double S = 0.0;
#pragma unroll
    for (int k = 0; k < 13; ++k) S += A[k] * A[k];
    double q6 = 0.0, norm = 0.0;
    if (n > 0 && S > 0.0) { const double rs = sqrt(S); q6 = rs / (double)n; norm = 1.0 / ((double)n * rs); }
    const double f = 1.0 / (1.0 + exp(-(q6 - q_thresh) * inv_width));
    // record of the generic fp64 kernels (cv.cu: k_q6_pass1): B_m = conj(A_m) / (n sqrt(S)); [13..15] = the atom's position;
    // q6 and f'(q6) go to the dense per-atom arrays
    double4 *r4 = reinterpret_cast<double4 *>(rec + (size_t)s * METAD_NREC);
    stg4(r4, make_double4(A[0] * norm, A[1] * norm, -A[2] * norm, A[3] * norm));
    stg4(r4 + 1, make_double4(-A[4] * norm, A[5] * norm, -A[6] * norm, A[7] * norm));
    stg4(r4 + 2, make_double4(-A[8] * norm, A[9] * norm, -A[10] * norm, A[11] * norm));
    stg4(r4 + 3, make_double4(-A[12] * norm, pi.x, pi.y, pi.z));       // own atoms are never periodic images: pi is the raw position
    q6arr[s] = q6; q6arr[N + s] = f * (1.0 - f) * inv_width;
    q6_out = q6; f_out = f;
}

template <bool STAGED>
__device__ __forceinline__ void build_body64(const TileGeom &g, const TileTables &t, const double4 *__restrict__ spos,
                                             const Stage64 &pos_s, nl16_t *list_s, const int *__restrict__ scell,
                                             const BoxD &bd, double rc2, int maxn, int *__restrict__ nl_count,
                                             int *__restrict__ nl, unsigned int *__restrict__ sticky, double q_thresh,
                                             double inv_width, double *__restrict__ rec, double *__restrict__ q6arr, double (&v)[2],
                                             const DevGeom *__restrict__ dg) {
    const double rc2_hi = rc2 * (1.0 + 1e-9), rc2_lo = rc2 * (1.0 - 1e-9);
    const int tid = threadIdx.x;
    // list column of this thread: the two 16-bit halves of a 32-bit shared-memory word belong to the SAME lane of two
    // neighbouring warps, so the lanes of a warp store to 32 different banks whatever slot each of them is at (with column =
    // thread index, lanes 2i and 2i + 1 shared a bank and conflicted whenever their candidate counts differed)
    const int col = ((((tid >> 6) << 5) + (tid & 31)) << 1) + ((tid >> 5) & 1);
    for (int a = tid; a < t.nown; a += blockDim.x) {
        bool ovf = false;
        const int cnt = scan_atom64<STAGED>(g, t, spos, pos_s, list_s, scell, a, col, rc2_hi, ovf, dg);
        double q6, f;
        finish_atom64<STAGED>(g, t, spos, pos_s, list_s, a, col, cnt, ovf, bd, rc2, rc2_lo, maxn, nl_count, nl, sticky,
                              q_thresh, inv_width, rec, q6arr, dg, q6, f);
        v[0] += q6; v[1] += f;
    }
}

__global__ void __launch_bounds__(TILE_THREADS, TILE64_MINB)
k_tile_build64(TileGeom g, const double4 *__restrict__ spos, const int *__restrict__ scell,
               const int *__restrict__ cell_start, BoxD bd, double rc2, int maxn,
               int *__restrict__ nl_count, int *__restrict__ nl, unsigned int *__restrict__ sticky,
               double q_thresh, double inv_width, double *__restrict__ rec, double *__restrict__ q6arr /* [N] q6 | [N] f'(q6) */,
               double *__restrict__ partials, unsigned int *__restrict__ ticket, double scale_mean, double scale_solid,
               double *__restrict__ cv_q6 /* [2]: Q6 mean, solid count */,
               double *__restrict__ cv_out /* the context's CV vector on the run paths, else NULL (k_q6_publish) */,
               int dim0, int dim1, const DevGeom *__restrict__ dg) {
    pdl_enter();
    extern __shared__ double4 dyn_smem64[];
    __shared__ TileTables t;
    __shared__ double red[64];
    Stage64 pos_s;
    pos_s.xy = reinterpret_cast<double2 *>(dyn_smem64);
    pos_s.z = reinterpret_cast<double *>(pos_s.xy + g.cap);
    pos_s.idx = reinterpret_cast<int *>(pos_s.z + g.cap);
    nl16_t *list_s = reinterpret_cast<nl16_t *>(pos_s.idx + g.cap);
    double v[2] = { 0.0, 0.0 };
    if (g.sparse && tile_is_empty(g, cell_start)) {
        // nothing to build here (block-uniform): the block only takes part in the reduction below
    } else {
        tile_setup(g, cell_start, t, *reinterpret_cast<TileScratch *>(dyn_smem64), dg);   // scratch = the (still unused) staging area
        tile_stage_pos64(g, t, spos, pos_s, dg);
        __syncthreads();
        if (t.total > 65535) {
            if (threadIdx.x == 0) atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW);
        } else if (t.staged) {
            build_body64<true>(g, t, spos, pos_s, list_s, scell, bd, rc2, maxn, nl_count, nl, sticky, q_thresh, inv_width, rec, q6arr, v, dg);
        } else {
            build_body64<false>(g, t, spos, pos_s, list_s, scell, bd, rc2, maxn, nl_count, nl, sticky, q_thresh, inv_width, rec, q6arr, v, dg);
        }
    }
    block_reduce<2>(v, red);
    const int bid = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x, nblk = gridDim.x * gridDim.y * gridDim.z;
    if (threadIdx.x == 0) { partials[2 * bid] = v[0]; partials[2 * bid + 1] = v[1]; }
    if (last_block_ticket(ticket)) {                      // fixed-order sum of the per-tile partials
        double u[2] = { 0.0, 0.0 };
        for (int b = threadIdx.x; b < nblk; b += blockDim.x) { u[0] += partials[2 * b]; u[1] += partials[2 * b + 1]; }
        block_reduce<2>(u, red);
        if (threadIdx.x == 0) {
            cv_q6[0] = scale_mean * u[0]; cv_q6[1] = scale_solid * u[1];
            if (cv_out) {
                if (dim0 >= 0) cv_out[dim0] = cv_q6[0];
                if (dim1 >= 0) cv_out[dim1] = cv_q6[1];
            }
            if (!isfinite(cv_q6[0]) || !isfinite(cv_q6[1])) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host side
TileGeom tile_geom(const metad_ctx *c);        // api.cu

static size_t smem_build64(const TileGeom &g) {
    return std::max((size_t)STAGE64_BYTES * (size_t)g.cap, (size_t)TILE_SCRATCH_BYTES) + sizeof(nl16_t) * LIST_CAP64 * TILE_THREADS;
}

int tiled64_init() {
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build64, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    return METAD_OK;
}

int tiled64_build(metad_ctx *c) {
    TileGeom g = tile_geom(c);
    const dim3 grid3(g.ntx, g.nty, g.ntz_launch);
    const double qt = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_thresh : 0.0;
    const double qw = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_width : 1.0;
    klaunch_pdl(true, k_tile_build64, grid3, TILE_THREADS, smem_build64(g), c->stream,
                g, (const double4 *)c->d_spos, (const int *)c->d_scell, (const int *)c->d_cell_start, c->boxd, c->rcl2, c->maxn,
                c->d_nl_count, c->d_nl, c->d_sticky, qt, 1.0 / qw, (double *)c->d_rec, (double *)c->d_q6,
                c->d_partials + c->nblocks_atoms, c->d_tickets + 1,
                c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0, c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0,
                c->d_cvq6, c->cv_direct, c->q6_mean_dim, c->q6_solid_dim, (const DevGeom *)c->dg);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
