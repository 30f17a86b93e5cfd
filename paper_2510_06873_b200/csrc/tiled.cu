// tiled.cu — fp32 fast path of a1 (neighbour list) fused with a3 (Q6 pass 1) or a2 (ungrouped coordination sum)
// on shared-memory tiles of the cell grid (tile.cuh).  One block per tile; one thread per own atom.
//   k_tile_build<MODE> candidate scan from shared memory with no per-pair minimum image: every
//                     candidate with r^2 < rc^2(1+1e-5) goes to a per-thread list in shared memory;
//                     a second loop over that short list takes the exact decision (pairs within the
//                     1e-5 band are re-decided with the canonical fp64 predicate, reading O), writes
//                     the neighbour list and — fused — accumulates the atom's 13 q6m components (MODE 1) or its
//                     sum of switching functions (MODE 2); MODE 0 builds the list only.
//   k_q6_publish      hands the sums finished by the last block of k_tile_build to the caller (Q6 / solid-like / C.N.)
// (the force kernels of this path, k_q6_force_g and k_coord_force_g, live in cv.cu)
#include <algorithm>
#include "common.cuh"
#include "cv_q6.cuh"
#include "cv_switch.cuh"
#include "tile.cuh"


typedef unsigned short nl16_t;   // local halo index (shared-memory candidate list only)
#define LIST_CAP 40            // per-thread candidate slots in shared memory (maxn <= 32 on this path + band + self)

// Packed fp32 pairs (sm_100 FADD2 / FMUL2 / FFMA2: one issue slot for two lanes of arithmetic; this kernel is bound by
// instruction issue, not by the FMA pipe).  A scalar second operand is broadcast by the instruction itself.
typedef unsigned long long f32x2_t;
__device__ __forceinline__ f32x2_t pk2(float a, float b) { f32x2_t r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(f32x2_t r, float &a, float &b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(r)); }
__device__ __forceinline__ f32x2_t add2(f32x2_t a, f32x2_t b) { f32x2_t r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2_t mul2(f32x2_t a, f32x2_t b) { f32x2_t r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2_t fma2(f32x2_t a, f32x2_t b, f32x2_t c) { f32x2_t r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

template <bool STAGED>
__device__ __forceinline__ float4 hpos(const TileGeom &g, const TileTables &t, const float4 *__restrict__ spos, const float4 *pos_s, int li,
                                       const DevGeom *dg) {
    if (STAGED) return pos_s[li];
    int s = tile_seg_of(t, li);
    int gi = t.seg_g[s] + (li - t.seg_off[s]);
    return tile_transform(g, t, s, spos[gi], gi, dg);
}

// ------------------------------------------------------------------------------------------------
// Candidate scan of own atom a into list column `col`: every halo atom of the 3 x 3 row-runs around the atom's cell with
// r^2 < rc^2 (1 + 1e-5) (tile-local coordinates, no per-pair minimum image).  Returns the number of candidates kept.
template <bool STAGED>
__device__ __forceinline__ int scan_atom(const TileGeom &g, const TileTables &t, const float4 *__restrict__ spos,
                                         const float4 *pos_s, nl16_t *list_s, const int *__restrict__ scell, int a, int col,
                                         float rc2_hi, bool &ovf, const DevGeom *dg) {
    const int q = tile_own_row(t, a);
    const int o = a - t.own_off[q];
    const int li = t.own_l[q] + o, s = t.own_g[q] + o;
    const float4 pi = hpos<STAGED>(g, t, spos, pos_s, li, dg);
    const int ic = scell[s] % g.nc0 - t.x0 + g.hx;       // halo-cell column of the own atom
    const int r0 = t.own_row[q], rstride = t.Tye + 2;
    // candidate list written through 32-bit shared-memory addresses (generic 64-bit pointer bumps cost 4 extra
    // instructions per candidate): slot k of this column lives at w0 + k * STRIDE
    const unsigned STRIDE = TILE_THREADS * (unsigned)sizeof(nl16_t);
    const unsigned w0 = (unsigned)__cvta_generic_to_shared(list_s + col);
    unsigned wp = w0;
    const unsigned wend = w0 + (LIST_CAP - 1) * STRIDE;
    const f32x2_t npi_xy = pk2(-pi.x, -pi.y);
#pragma unroll 1
    for (int dz = -1; dz <= 1; ++dz) {
#pragma unroll 1
        for (int dy = -1; dy <= 1; ++dy) {
            const int r = r0 + dz * rstride + dy;
            int lo = t.hcell[r][ic - g.hx];
            const int hi = t.hcell[r][ic + g.hx + 1];
            while (lo < hi) {
                // every candidate is stored unconditionally and the slot kept only if it passes (load, 6 flop, store,
                // compare, bump): one free slot is needed, capacity is checked once per stretch
                const int room = (int)((wend - wp) / STRIDE);
                if (room <= 0) { ovf = true; break; }
                const int h2 = min(hi, lo + room);
#pragma unroll 2
                for (int lj = lo; lj < h2; ++lj) {
                    const float4 pj = hpos<STAGED>(g, t, spos, pos_s, lj, dg);
                    // (dx, dy) and their squares as one packed pair each: 5 issue slots instead of 6 per candidate (the
                    // rounding differs from the exact pass by an ulp: far inside the 1e-5 band of this prefilter)
                    const f32x2_t dxy = add2(pk2(pj.x, pj.y), npi_xy);
                    float sx, sy;
                    upk2(mul2(dxy, dxy), sx, sy);
                    const float dz2 = pj.z - pi.z;
                    const float r2 = fmaf(dz2, dz2, sx + sy);
                    asm volatile("st.shared.u16 [%0], %1;" ::"r"(wp), "h"((unsigned short)lj));
                    // keep the slot iff the candidate passes: one predicated add (the compiler's select form costs 3)
                    asm volatile("{ .reg .pred p; setp.lt.f32 p, %1, %2; @p add.u32 %0, %0, %3; }"
                                 : "+r"(wp) : "f"(r2), "f"(rc2_hi), "r"(STRIDE));
                }
                lo = h2;
            }
        }
    }
    return (int)((wp - w0) / STRIDE);
}

// Exact decision on the short list of own atom a (list column `col`, cnt candidates), neighbour-list write, fused q6m
// accumulation and the atom's q6 record.  Returns q6.
template <bool STAGED, int MODE>
__device__ __forceinline__ float finish_atom(const TileGeom &g, const TileTables &t, const float4 *__restrict__ spos,
                                             const float4 *pos_s, const nl16_t *list_s, int a, int col, int cnt, bool ovf,
                                             const BoxD &bd, float rc2f, float rc2_lo, double rc2, int maxn,
                                             int *__restrict__ nl_count, int *__restrict__ nl, unsigned int *__restrict__ sticky,
                                             float q_thresh, float inv_width, float *__restrict__ rec,
                                             float *__restrict__ q6_out, bool solid, int sw_n, int sw_m,
                                             const int *__restrict__ perm, const DevGeom *__restrict__ dg) {
    const bool WITH_Q6 = MODE == 1;
    float csum = 0.f;                                      // MODE 2: sum of sw(r / r0) over the neighbours (q_thresh = 1 / r0)
    float cgx = 0.f, cgy = 0.f, cgz = 0.f;                 // MODE 2: sum of 2 sw' d / (r0 r)
    const int q = tile_own_row(t, a);
    const int o = a - t.own_off[q];
    const int li = t.own_l[q] + o, s = t.own_g[q] + o;
    const float4 pi = hpos<STAGED>(g, t, spos, pos_s, li, dg);
    const nl16_t *myl = list_s + col;
    if (ovf) atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW);
    int *out = nl + ((size_t)(s >> 5) * maxn) * 32 + (s & 31);
    float A[13];
#pragma unroll
    for (int k = 0; k < 13; ++k) A[k] = 0.f;
    f32x2_t AP[6];                                        // (A[2m-1], A[2m]), m = 1..6: one FFMA2 per m and neighbour
#pragma unroll
    for (int k = 0; k < 6; ++k) AP[k] = 0ull;
    int n = 0;
    for (int k = 0; k < cnt; ++k) {
        const int lj = myl[k * TILE_THREADS];
        if (lj == li) continue;
        const float4 pj = hpos<STAGED>(g, t, spos, pos_s, lj, dg);
        const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        const float r2 = dx * dx + dy * dy + dz * dz;
        bool in = r2 < rc2f;
        if (r2 >= rc2_lo) {                                // borderline: canonical fp64 predicate on the inputs
            const float4 gi = spos[s], gj = spos[__float_as_int(pj.w) & NL_IDX_MASK];
            in = r2_canonical(dg ? dg->bd : bd, (double)gj.x - (double)gi.x, (double)gj.y - (double)gi.y,
                              (double)gj.z - (double)gi.z) < rc2;
        }
        if (!in) continue;
        if (n < maxn) {
            // streaming store: the list is read once, by the force pass (MODE 2 with nl == NULL: list-free pass, the sum
            // and the gradient below are all the step needs — params.lazy_neighbors)
            if (MODE != 2 || nl) __stcs(out + n * 32, __float_as_int(pj.w));
            if (MODE == 2) {
                // the per-atom gradient sum_j 2 sw'(r_ij) d_ij / (r0 r_ij) does not depend on dV/ds: accumulated here, the
                // force stage only scales it (k_force_add, cv.cu) instead of walking the list again
                float gpair;
                if (sw_m == 2 * sw_n && !(sw_n & 1)) {
                    // sw = 1 / (1 + x^n) with n even needs only x^2 = r^2 / r0^2 (no square roots):
                    // 2 sw' / (r0 r) = -2 n (x^2)^(n/2 - 1) sw^2 / r0^2        (block-uniform branch; all five configs)
                    const float x2 = r2 * q_thresh * q_thresh;
                    const float xh = sw_n == 6 ? x2 * x2 : ipow(x2, sw_n / 2 - 1);
                    const float sw = __fdividef(1.f, 1.f + xh * x2);
                    csum += sw;
                    gpair = (float)(-2 * sw_n) * xh * sw * sw * (q_thresh * q_thresh);
                } else {
                    float dsw;
                    csum += switch_fn<float>(sqrtf(r2) * q_thresh, sw_n, sw_m, dsw);
                    gpair = 2.f * dsw * q_thresh * rsqrtf(r2);
                }
                cgx += gpair * dx; cgy += gpair * dy; cgz += gpair * dz;
            }
            if (WITH_Q6) {
                const float rinv = rsqrtf(r2);
                Y6<float> y;
                y6_eval<float>(dx * rinv, dy * rinv, dz * rinv, y);
                A[0] += y.E[0];
#pragma unroll
                for (int m = 1; m <= 6; ++m) AP[m - 1] = fma2(pk2(y.c[m], y.s[m]), pk2(y.E[m], y.E[m]), AP[m - 1]);
            }
        }
        ++n;
    }
#pragma unroll
    for (int m = 1; m <= 6; ++m) upk2(AP[m - 1], A[2 * m - 1], A[2 * m]);
    if (n > maxn) { atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW); n = maxn; }
    if (MODE != 2 || nl) nl_count[s] = n;
    float q6 = 0.f;
    if (WITH_Q6) {
        float S = 0.f;
#pragma unroll
        for (int k = 0; k < 13; ++k) S += A[k] * A[k];
        float norm = 0.f;
        if (n > 0 && S > 0.f) { float rs = sqrtf(S); q6 = rs / (float)n; norm = 1.f / ((float)n * rs); }
        // the two 32-byte halves of a record live in two arrays (a 128-byte line then holds four atoms per half: the
        // lanes of the force pass, whose neighbours are near one another in the sorted order, touch fewer lines per load)
        float4 *r4 = reinterpret_cast<float4 *>(rec + (size_t)s * 8);
        float4 *r4b = reinterpret_cast<float4 *>(rec + (size_t)g.natoms * 8 + (size_t)s * 8) - 2;
        r4[0] = make_float4(A[0] * norm, A[1] * norm, -A[2] * norm, A[3] * norm);
        r4[1] = make_float4(-A[4] * norm, A[5] * norm, -A[6] * norm, A[7] * norm);
        r4b[2] = make_float4(-A[8] * norm, A[9] * norm, -A[10] * norm, A[11] * norm);
        {                                                 // the record carries the atom's own (global, exact fp32)
            const float4 gp = spos[s];                    // position, so the force pass needs no second 16-byte gather
            r4b[3] = make_float4(-A[12] * norm, gp.x, gp.y, gp.z);
        }
        if (solid) {                                      // f'(q6) of the solid-like count: a dense 4-byte array of its own
            const float f = 1.f / (1.f + expf(-(q6 - q_thresh) * inv_width));
            q6_out[(size_t)g.natoms + s] = f * (1.f - f) * inv_width;
        }
        q6_out[s] = q6;
    }
    // ORIGINAL atom order (one scattered 16-byte store here, where the memory pipes idle): the force stage is then a
    // coalesced pass over F (k_force_add)
    if (MODE == 2 && rec) reinterpret_cast<float4 *>(rec)[perm[s]] = make_float4(cgx, cgy, cgz, 0.f);
    return MODE == 2 ? csum : q6;
}

// One thread per own atom: scan, then the exact pass.  (Re-dealing the atoms to the threads by candidate count between the
// two passes, so that the lanes of a warp run equal trip counts, was measured and dropped: profiles/r1h_rejected.md.)
template <bool STAGED, int MODE>
__device__ __forceinline__ void build_body(const TileGeom &g, const TileTables &t, const float4 *__restrict__ spos,
                                           const float4 *pos_s, nl16_t *list_s, const int *__restrict__ scell,
                                           const BoxD &bd, float rc2f, double rc2, int maxn, int *__restrict__ nl_count,
                                           int *__restrict__ nl, unsigned int *__restrict__ sticky, float q_thresh,
                                           float inv_width, float *__restrict__ rec, float *__restrict__ q6_out, bool solid,
                                           int sw_n, int sw_m, const int *__restrict__ perm, double (&v)[2],
                                           const DevGeom *__restrict__ dg) {
    const float rc2_hi = rc2f * (1.f + 1e-5f), rc2_lo = rc2f * (1.f - 1e-5f);
    const int tid = threadIdx.x;
    // list column of this thread: the two 16-bit halves of a 32-bit shared-memory word belong to the SAME lane of two
    // neighbouring warps, so the lanes of a warp store to 32 different banks whatever slot each of them is at (with column =
    // thread index, lanes 2i and 2i + 1 shared a bank and conflicted whenever their candidate counts differed)
    const int col = ((((tid >> 6) << 5) + (tid & 31)) << 1) + ((tid >> 5) & 1);
    for (int a = tid; a < t.nown; a += blockDim.x) {
        bool ovf = false;
        const int cnt = scan_atom<STAGED>(g, t, spos, pos_s, list_s, scell, a, col, rc2_hi, ovf, dg);
        const float q6 = finish_atom<STAGED, MODE>(g, t, spos, pos_s, list_s, a, col, cnt, ovf, bd, rc2f, rc2_lo, rc2, maxn,
                                                   nl_count, nl, sticky, q_thresh, inv_width, rec, q6_out, solid, sw_n, sw_m, perm, dg);
        if (MODE != 0) v[0] += (double)q6;
        if (MODE == 1) v[1] += (double)(1.f / (1.f + expf(-(q6 - q_thresh) * inv_width)));
    }
}

// DEVBOX: the step's box lives in device memory (metad_*_dev, NPT); the host-box instances never touch the pointer, so they
// keep the registers and the schedule they had without it
template <int MODE, bool DEVBOX>   // 0: list only, 1: + Q6 pass 1, 2: + coordination sum (ungrouped COORD, q_thresh = 1 / r0)
__global__ void __launch_bounds__(TILE_THREADS, 5)
k_tile_build(TileGeom g, const float4 *__restrict__ spos, const int *__restrict__ scell,
             const int *__restrict__ cell_start, BoxD bd, float rc2f, double rc2, int maxn,
             int *__restrict__ nl_count, int *__restrict__ nl, unsigned int *__restrict__ sticky,
             float q_thresh, float inv_width, float *__restrict__ rec, float *__restrict__ q6_out, int solid,
             int sw_n, int sw_m, const int *__restrict__ perm, double *__restrict__ partials, unsigned int *__restrict__ ticket, double scale_mean, double scale_solid,
             double *__restrict__ cv_q6 /* [2]: Q6 mean, solid count */,
             double *__restrict__ cv_out /* the context's CV vector on the run paths (NULL: k_q6_publish hands the sums over) */,
             int dim0, int dim1, const DevGeom *__restrict__ dg_arg,
             const int *__restrict__ skin_flag, const int *__restrict__ step) {
    pdl_enter();
    if (MODE == 0 && SKIN_SKIP(skin_flag, step)) return;        // Verlet skin: the kept list is still valid (neighbor.cu)
    const DevGeom *dg = DEVBOX ? dg_arg : nullptr;
    extern __shared__ float4 dyn_smem[];
    __shared__ TileTables t;
    __shared__ double red[64];
    float4 *pos_s = dyn_smem;
    nl16_t *list_s = reinterpret_cast<nl16_t *>(dyn_smem + g.cap);
    __shared__ unsigned long long stage_bar;
    double v[2] = { 0.0, 0.0 };
    if (g.sparse && tile_is_empty(g, cell_start)) {
        // nothing to build here (block-uniform): the block only takes part in the reduction below
    } else {
    // a device-resident box (NPT, dg != NULL) replaces the lattice rows of the arguments at their few points of use (tile
    // origin, periodic images, fp64 recheck): the common case costs no registers
    tile_setup(g, cell_start, t, *reinterpret_cast<TileScratch *>(dyn_smem), dg);   // scratch = the (still unused) staging area
    if (t.staged && !t.any_wrapped && t.total > 0) tile_stage_pos_tma(t, spos, pos_s, &stage_bar);   // block-uniform choice
    else
    tile_stage_pos(g, t, spos, pos_s, dg);
    __syncthreads();
    if (t.total > 65535) {
        if (threadIdx.x == 0) atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW);
    } else if (t.staged) {
        build_body<true, MODE>(g, t, spos, pos_s, list_s, scell, bd, rc2f, rc2, maxn, nl_count, nl, sticky, q_thresh,
                                  inv_width, rec, q6_out, solid != 0, sw_n, sw_m, perm, v, dg);
    } else {
        build_body<false, MODE>(g, t, spos, pos_s, list_s, scell, bd, rc2f, rc2, maxn, nl_count, nl, sticky, q_thresh,
                                   inv_width, rec, q6_out, solid != 0, sw_n, sw_m, perm, v, dg);
    }
    }
    if (MODE != 0) {
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
}

// a3 on the tiled path: the sums were finished by the last block of k_tile_build; hand them to the caller
__global__ void k_q6_publish(const double *__restrict__ cv_q6, int dim_mean, int dim_solid, double *__restrict__ cv_out) {
    if (threadIdx.x == 0) {
        if (dim_mean >= 0) cv_out[dim_mean] = cv_q6[0];
        if (dim_solid >= 0) cv_out[dim_solid] = cv_q6[1];
    }
}

// ------------------------------------------------------------------------------------------------
// host side
TileGeom tile_geom(const metad_ctx *c);        // api.cu

static size_t smem_build(const TileGeom &g) {
    return std::max(sizeof(float4) * (size_t)g.cap, (size_t)TILE_SCRATCH_BYTES) + sizeof(nl16_t) * LIST_CAP * TILE_THREADS;
}

int tiled_init() {
    // per (device, function) attribute: set on every metad_create — no process-wide "done" flag, so contexts created from
    // several threads or on several devices need no synchronisation
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    CUDA_TRY(cudaFuncSetAttribute(k_tile_build<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
    return METAD_OK;
}

int tiled_build(metad_ctx *c) {
    TileGeom g = tile_geom(c);
    const dim3 grid3(g.ntx, g.nty, g.ntz_launch);  // tile (tx, ty, tz) = blockIdx (+ the window offset tz0): no division in the kernel
    double qt = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_thresh : 0.0;
    double qw = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_width : 1.0;
#define TILE_LAUNCH(MODE, ...)                                                                                        \
    do {                                                                                                              \
        if (c->dg) klaunch_pdl(!c->skin_on, k_tile_build<MODE, true>, grid3, TILE_THREADS, smem_build(g), c->stream, __VA_ARGS__);   \
        else klaunch_pdl(!c->skin_on, k_tile_build<MODE, false>, grid3, TILE_THREADS, smem_build(g), c->stream, __VA_ARGS__);        \
    } while (0)
    const int *sf = c->skin_on ? c->d_skin_flag : nullptr;
    if (c->has_q6 && !c->skin_on)
        TILE_LAUNCH(1,
            g, (const float4 *)c->d_spos, c->d_scell, c->d_cell_start, c->boxd, (float)c->rcl2, c->rcl2, c->maxn,
            c->d_nl_count, c->d_nl, c->d_sticky, (float)qt, (float)(1.0 / qw), (float *)c->d_rec, c->d_q6,
            c->q6_solid_dim >= 0 ? 1 : 0, 0, 0, c->d_perm, c->d_partials + c->nblocks_atoms, c->d_tickets + 1,
            c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0, c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0,
            c->d_cvq6, c->cv_direct, c->q6_mean_dim, c->q6_solid_dim, c->dg, nullptr, c->d_step);
    else if (c->has_coord && !c->skin_on) {                   // ungrouped coordination number: the sum of sw rides on the exact pass
        const CvDev &d = c->cv[c->coord_dim];
        // lazy_neighbors: nothing downstream reads the list (the force stage scales the per-atom gradient; the virial would
        // walk the list) — the pass runs list-free and metad_get_neighbors reports that there is no list
        c->list_skipped = c->p.lazy_neighbors && !c->p.want_virial && c->d_cgrad;
        TILE_LAUNCH(2,
            g, (const float4 *)c->d_spos, c->d_scell, c->d_cell_start, c->boxd, (float)c->rcl2, c->rcl2, c->maxn,
            c->d_nl_count, c->list_skipped ? nullptr : c->d_nl, c->d_sticky, (float)(1.0 / d.r0), 1.f, c->d_cgrad, nullptr, 0, d.n, d.m, c->d_perm,
            c->d_partials + c->nblocks_atoms, c->d_tickets + 1, d.scale, 0.0, c->d_cvq6, c->cv_direct, c->coord_dim, -1, c->dg, nullptr, c->d_step);
    } else
        TILE_LAUNCH(0,
            g, (const float4 *)c->d_spos, c->d_scell, c->d_cell_start, c->boxd, (float)c->rcl2, c->rcl2, c->maxn,
            c->d_nl_count, c->d_nl, c->d_sticky, 0.f, 1.f, nullptr, nullptr, 0, 0, 0, c->d_perm, nullptr, nullptr, 0.0, 0.0, nullptr, nullptr, -1, -1, c->dg, sf, c->d_step);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

// the q6m accumulation and its reduction already ran inside k_tile_build
int tiled_q6_pass1(metad_ctx *c, double *d_cv) {
    if (c->cv_direct && c->cv_direct == d_cv) return METAD_OK;      // the build kernel wrote these dimensions itself
    if (c->has_q6) k_q6_publish<<<1, 32, 0, c->stream>>>(c->d_cvq6, c->q6_mean_dim, c->q6_solid_dim, d_cv);
    else k_q6_publish<<<1, 32, 0, c->stream>>>(c->d_cvq6, c->coord_dim, -1, d_cv);          // tiled coordination number
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
