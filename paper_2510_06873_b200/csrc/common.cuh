// common.cuh — shared device helpers and the context of the B200 metadynamics library.
// (CUDA path only; shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/metad.h"

// generic (non-tiled) kernels switch from one thread to one warp per atom below this size: a system this small cannot
// fill 148 SMs with one thread per atom (BASELINE.json configs[0]-[2] are latency-bound otherwise)
#define METAD_WARP_PER_ATOM_MAX 32768
// below this size the neighbour stage is one brute-force kernel without cells (k_build_list_small)
#define METAD_SMALL_N 1024

#define METAD_NREC 16  // per-atom Q6 record: 13 normalised q6m components + the atom's position (the force pass gathers ONE array);
                       // q6 and f'(q6) live in the dense per-atom arrays d_q6 [N] | [N]

// ------------------------------------------------------------------------------------------------
// Periodic box for the pair arithmetic in precision T.  Lattice rows a=(ax,0,0), b=(bx,by,0),
// c=(cx,cy,cz).  For T=float every component is split hi+lo so that a lattice shift applied to an
// (exact) fp32 coordinate difference stays accurate to ~1 ulp of the result.
template <typename T>
struct PBox {
    T ax, bx, by, cx, cy, cz;        // hi parts (the whole value for T=double)
    T lax, lbx, lby, lcx, lcy, lcz;  // lo parts (0 for T=double)
    T hx, hy, hz;                    // half box: 0.5*ax, 0.5*by, 0.5*cz
    T band;                          // T=float: |r^2 - rc^2| <= band is re-decided in fp64 (neighbor.cu: pair_in_range); 0 for double
};

struct BoxD {                        // fp64 box, used by the canonical neighbour predicate
    double ax, bx, by, cx, cy, cz, hx, hy, hz;
};

struct CellGrid {
    int nc[3];                       // cells along a, b, c
    int ncell;
    double inv[6];                   // fractional transform: s_c = z*i0; s_b = (y - s_c*cy)*i1; ...
    double cx, cy, bx;               // tilt terms for cartesian -> fractional
    double wlo, wlen;                // window of fractional c-coordinates that holds every atom (params.fill_fraction < 1); wlen >= 1: none
};

// Device-resident geometry of the current step (metad_build_neighbors_dev / metad_run_dev: the box lives in device memory and
// may change every step without the host seeing it — NPT).  k_geom_update derives it from the 9 box doubles;
// every kernel takes a `const DevGeom *dg` that is NULL on the host-box paths (geometry in the kernel arguments, constant bank)
// and overrides the by-value arguments otherwise.  The cell COUNTS stay those of the capture; the kernel checks that the cells
// are still at least rc wide and sets METAD_DEV_BOX otherwise.
struct DevGeom {
    BoxD bd;
    PBox<float> pbf;
    PBox<double> pbd;
    double inv[6], cx, cy, bx;       // CellGrid: cartesian -> fractional
    double box[9];
};
template <typename T> __device__ __forceinline__ const PBox<T> &dg_pb(const DevGeom *dg);
template <> __device__ __forceinline__ const PBox<float> &dg_pb<float>(const DevGeom *dg) { return dg->pbf; }
template <> __device__ __forceinline__ const PBox<double> &dg_pb<double>(const DevGeom *dg) { return dg->pbd; }

template <typename T> struct Vec4;
template <> struct Vec4<float> { typedef float4 type; };
template <> struct Vec4<double> { typedef double4 type; };

template <typename T>
__device__ __forceinline__ typename Vec4<T>::type ld4(const typename Vec4<T>::type *p) { return *p; }

// Read-only gather of one Vec4: a double4 is 32 bytes but only 16-byte aligned for the compiler, which splits it into two
// 128-bit loads; the arrays gathered here (cell-sorted positions, q6 records) have 32-byte element strides on 256-byte
// aligned allocations, so the fp64 kernels fetch an element with ONE 256-bit load (sm_100 LDG.E.256: half the L1 requests
// of a gather-bound kernel).  Only for arrays the kernel does not write.
template <typename T>
__device__ __forceinline__ typename Vec4<T>::type ldg4(const typename Vec4<T>::type *p);
template <> __device__ __forceinline__ float4 ldg4<float>(const float4 *p) { return *p; }
// one 256-bit store of a double4 (st.global.v4.f64; 32-byte aligned address)
__device__ __forceinline__ void stg4(double4 *p, const double4 &v) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(v.x), "d"(v.y), "d"(v.z), "d"(v.w) : "memory");
}
template <typename T> __device__ __forceinline__ void st4(typename Vec4<T>::type *p, const typename Vec4<T>::type &v);
template <> __device__ __forceinline__ void st4<float>(float4 *p, const float4 &v) { *p = v; }
template <> __device__ __forceinline__ void st4<double>(double4 *p, const double4 &v) { stg4(p, v); }
template <> __device__ __forceinline__ double4 ldg4<double>(const double4 *p) {
    double4 v;
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}

// Minimum-image displacement (reading O order: z against c, y against b, x against a).
template <typename T>
__device__ __forceinline__ void min_image(const PBox<T> &b, T &dx, T &dy, T &dz) {
    T sz = dz > b.hz ? T(-1) : (dz < -b.hz ? T(1) : T(0));
    dx += sz * b.cx; dy += sz * b.cy; dz += sz * b.cz;
    dx += sz * b.lcx; dy += sz * b.lcy; dz += sz * b.lcz;
    T sy = dy > b.hy ? T(-1) : (dy < -b.hy ? T(1) : T(0));
    dx += sy * b.bx; dy += sy * b.by;
    dx += sy * b.lbx; dy += sy * b.lby;
    T sx = dx > b.hx ? T(-1) : (dx < -b.hx ? T(1) : T(0));
    dx += sx * b.ax;
    dx += sx * b.lax;
}

// The canonical fp64 predicate arithmetic (reading O): identical operation order and rounding to
// the definition — no FMA contraction in r^2.
__device__ __forceinline__ double r2_canonical(const BoxD &b, double dx, double dy, double dz) {
    if (dz > b.hz) { dx -= b.cx; dy -= b.cy; dz -= b.cz; }
    else if (dz < -b.hz) { dx += b.cx; dy += b.cy; dz += b.cz; }
    if (dy > b.hy) { dx -= b.bx; dy -= b.by; }
    else if (dy < -b.hy) { dx += b.bx; dy += b.by; }
    if (dx > b.hx) { dx -= b.ax; }
    else if (dx < -b.hx) { dx += b.ax; }
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

// The same arithmetic with the branch decisions taken once per run of cells instead of once per pair: inside a cell list
// with >= 3 cells per direction the neighbouring cell (jc, jb, ja) of (ic, ib, ia) names ONE image of its atoms, the wrap
// flags (wz, wy, wx) in {-1, 0, +1} of that cell are the branch outcomes of r2_canonical for every pair within rc (the
// margins hz - rc, hy - rc, hx - rc are positive by the box check), and adding +-c, +-b, +-a or 0.0 in the same order
// rounds identically.  Pairs farther than rc may land on another image than the canonical one; both are >= rc.
// sz = wz (cx, cy, cz), sy = wy (bx, by), sx = wx ax.
struct RunShift { double zx, zy, zz, yx, yy, xx; };
__device__ __forceinline__ double r2_shifted(const RunShift &w, double dx, double dy, double dz) {
    dx = __dadd_rn(dx, w.zx); dy = __dadd_rn(dy, w.zy); dz = __dadd_rn(dz, w.zz);
    dx = __dadd_rn(dx, w.yx); dy = __dadd_rn(dy, w.yy);
    dx = __dadd_rn(dx, w.xx);
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

// Neighbour decision of a pair of cell-sorted atoms in precision T (reading O).  fp64: the canonical predicate.  fp32: fast
// test; any pair within the recheck band of rc^2 is re-decided with the canonical fp64 arithmetic on the (exactly
// representable) fp32 coordinates, so the sets are identical to the fp64 definition.
template <typename T>
__device__ __forceinline__ bool pair_in_range(const PBox<T> &pb, const BoxD &bd, T rc2T, double rc2,
                                              const typename Vec4<T>::type &pi, const typename Vec4<T>::type &pj);
template <>
__device__ __forceinline__ bool pair_in_range<double>(const PBox<double> &, const BoxD &bd, double, double rc2,
                                                      const double4 &pi, const double4 &pj) {
    return r2_canonical(bd, pj.x - pi.x, pj.y - pi.y, pj.z - pi.z) < rc2;
}
template <>
__device__ __forceinline__ bool pair_in_range<float>(const PBox<float> &pb, const BoxD &bd, float rc2T, double rc2,
                                                     const float4 &pi, const float4 &pj) {
    float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
    min_image(pb, dx, dy, dz);
    float r2 = dx * dx + dy * dy + dz * dz;
    bool in = r2 < rc2T;
    if (fabsf(r2 - rc2T) <= pb.band)
        in = r2_canonical(bd, (double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y,
                          (double)pj.z - (double)pi.z) < rc2;
    return in;
}

// Verlet-skin reuse (params.skin): the build kernels of a step do nothing unless the step's rebuild flag is set
// (k_skin_check, neighbor.cu); flag == NULL: no skin, always build
#define SKIN_SKIP(flag, step) ((flag) != nullptr && (flag)[*(step) & 1] == 0)

// Programmatic dependent launch (sort phase and tile build): a kernel launched with klaunch_pdl(true, ...) may be scheduled while its
// predecessor in the stream still drains; pdl_enter() at its top (1) lets ITS successor be scheduled likewise and (2) waits until the
// predecessor grid has completed and its writes are visible.  Nothing is read or written before it, so the chain is as ordered as
// plain stream order; what is gained is the launch latency at every kernel boundary: 10 us per build on the stream paths (stage
// calls, metad_step_host), nothing inside the captured graph, whose node-to-node latency is already small.  The hill sum and the
// force kernel are NOT launched this way: their early-resident blocks cost the tail of k_tile_build 0.11 ms (measured,
// profiles/r2_experiments.md).  A kernel launched without the attribute passes through both instructions at once.
__device__ __forceinline__ void pdl_enter() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}
template <typename... P, typename... A>
static inline void klaunch_pdl(bool pdl, void (*kernel)(P...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, A &&...args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    (void)cudaLaunchKernelEx(&cfg, kernel, static_cast<P>(args)...);          // errors surface through cudaGetLastError at the call sites
}

// fp64 minimum image in the order of reading O (chain / torsion CVs, fused small-molecule step)
__device__ __forceinline__ void min_image_d(const BoxD &b, double &dx, double &dy, double &dz) {
    if (dz > b.hz) { dx -= b.cx; dy -= b.cy; dz -= b.cz; }
    else if (dz < -b.hz) { dx += b.cx; dy += b.cy; dz += b.cz; }
    if (dy > b.hy) { dx -= b.bx; dy -= b.by; }
    else if (dy < -b.hy) { dx += b.bx; dy += b.by; }
    if (dx > b.hx) { dx -= b.ax; }
    else if (dx < -b.hx) { dx += b.ax; }
}

// ------------------------------------------------------------------------------------------------
// Deterministic block reduction of K doubles per thread (fixed tree: shuffle inside the warp, then
// warp 0 sums the per-warp partials in warp order).
template <int K>
__device__ __forceinline__ void block_reduce(double (&v)[K], double *smem /* >= K*32 doubles */) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int k = 0; k < K; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
    }
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) smem[k * 32 + wid] = v[k];
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            double x = lane < nw ? smem[k * 32 + lane] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            v[k] = x;  // valid in thread 0
        }
    }
}

// "Last block finishes" pattern: every block writes its partials, the last one to arrive (atomic
// ticket) sums them in block order -> deterministic, one launch.  Returns true in the last block.
__device__ __forceinline__ bool last_block_ticket(unsigned int *ticket) {
    __shared__ bool is_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int t = atomicAdd(ticket, 1u);
        is_last = (t == gridDim.x * gridDim.y * gridDim.z - 1);
        if (is_last) *ticket = 0u;  // re-arm for the next launch
    }
    __syncthreads();
    if (is_last) __threadfence();
    return is_last;
}

// Bias virial (NEXT-3b, reading AD): every thread of the block hands in its 9 partial sums of G_a d_b over the pairs
// it visited; fixed-order block reduction, per-block partials, the last block adds coef * dv * sum to out9.
struct VirArgs { double *partials; unsigned int *ticket; double *out9; };
__device__ __forceinline__ void virial_finish(double (&w)[9], double *smem /* >= 9*32 doubles */, const VirArgs &va,
                                              double coef, const double *dv /* device scalar or NULL */) {
    block_reduce<9>(w, smem);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < 9; ++k) va.partials[(size_t)blockIdx.x * 9 + k] = w[k];
    }
    if (last_block_ticket(va.ticket)) {
        double t[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) t[k] = 0.0;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) {
#pragma unroll
            for (int k = 0; k < 9; ++k) t[k] += va.partials[(size_t)b * 9 + k];
        }
        block_reduce<9>(t, smem);
        if (threadIdx.x == 0) {
            const double f = coef * (dv ? dv[0] : 1.0);
#pragma unroll
            for (int k = 0; k < 9; ++k) va.out9[k] += f * t[k];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Host-side context
struct CvDev {                      // device copies of one CV descriptor
    int kind, n, m;
    double r0, scale, q_thresh, q_width;
    int npairs, nchain;
    int *d_pairs; double *d_pair_r0;      // CONTACTS
    int *d_csr_off, *d_csr_pair;          // CONTACTS: per touched atom incident pairs (gather form)
    int *d_catoms; int ncatoms;           //           the touched atoms
    int *d_chain; double *d_mass;         // RGYR
    double *d_unwrapped;                  // RGYR scratch: [nchain*3] + com[3] + rg
    bool use_groups;
    int fshift;                           // COORD, MINDIST: bit offset of this CV's (in A, in B) pair in the per-atom group flags
    int tors[4];                          // TORSION
    int *d_ga, *d_gb; int n_ga, n_gb;     // MINDIST: device copies of the group index lists (list-free variant)
};

struct metad_ctx {
    metad_params p;
    cudaStream_t stream;
    int N, prec, maxn, D;
    // neighbour / cell state
    CellGrid grid;
    BoxD boxd;
    double rc, rc2;                       // CV cutoff
    double rcl, rcl2;                     // list cutoff rc + skin (== rc without a skin): cells, list build
    int skin_on;                          // params.skin > 0 and a CV of the context reads the list
    int geom_ncell;                       // cells of the last setup_geometry before any x-subdivision (skin: detects a new grid)
    int *d_skin_flag;                     // [2] rebuild flags, indexed by the parity of the device step counter (neighbor.cu)
    void *d_ref;                          // Vec4<T>[N]: cell-sorted positions at the last build (displacement check)
    int *d_own_count; int own_count_valid; // slab-decomposition rank (fill_fraction < 1), tiled Q6 path: neighbour counts with the atoms the
                                          // rank does not own set to 0 (metad_cv_owned_sum), read by the force pass of the same step
    int *d_rc_count, *d_rc_list;          // skin, tiled Q6 path: the entries of the kept list that lie within rc THIS step (pass 1 -> force pass)
    int *d_nbuilds;                       // number of neighbour-list builds so far (metad_get_rebuilds)
    bool have_neighbors, list_built;
    int cell_cap;
    int *d_cell_count, *d_cell_start, *d_block_sums;
    int *d_cell_of, *d_slot, *d_perm, *d_perm_raw, *d_scell;   // perm_raw: counting-sort output before the in-cell ordering
    unsigned char *d_flags;               // per original atom: bit0 in A, bit1 in B (COORD)
    void *d_spos;                         // Vec4<T>[N], cell-sorted
    int *d_nl_count, *d_nl;               // sorted space; nl[k*N + s]
    // CV state
    CvDev cv[METAD_MAX_CV];
    bool has_q6, has_coord, has_torsion, has_mindist, has_lattice;
    double *d_traj;                       // traj_capacity > 0: [capacity][D] CV frames, frame k = step k + 1 since the last reset
    double *d_virial, *d_vir_partials;    // want_virial: [9] bias virial of the last apply_forces; per-block partials
    double *d_box_force;                  // LATTICE: [9] bias force on the box rows, written by apply_forces
    int mindist_dim;                      // first MINDIST dimension (-1: none); n_mindist of them, n_coord COORD dimensions
    int n_coord, n_mindist;
    double *d_mind;                       // MINDIST: per CV dimension d, at + 8 d: [r, dx, dy, dz] of the nearest pair + its two original indices
    double *d_tors_grad;                  // TORSION: [D][12] d phi / d r of the four atoms, written by the CV kernel
    int *d_tors_atoms; int ntors_atoms;   //          unique touched atoms (gather-form force kernel: thread per atom)
    int q6_mean_dim, q6_solid_dim, coord_dim;
    void *d_rec;                          // T[N][METAD_NREC]
    double *d_partials;                   // block partial sums
    double *d_partials_warp;              // block partial sums of the warp-per-atom coordination kernel (N/4 blocks)
    unsigned int *d_tickets;
    int nblocks_atoms;
    // bias state (all device)
    double *d_centers;                    // SoA [D][max_hills]
    double *d_heights;
    int *d_nhills, *d_step;
    unsigned int *d_sticky;
    double *d_cv, *d_V, *d_dVds;          // internal state of the last step
    double *d_bias_partials;
    double *d_table;                      // grid [4][n0][n1]
    int grid_on;
    // host-path staging
    void *d_pos_stage, *d_F_stage;
    void *h_pin; size_t h_pin_bytes;
    // graph
    DevGeom *d_geom;                      // device-resident geometry (box in device memory), written by k_geom_update
    const DevGeom *dg;                    // d_geom while the current step runs on a device box, else NULL
    const double *d_box_last;             // device box of the last *_dev call
    int dev_geom_ready;                   // the cell grid / tiling was derived for the device box (frozen until metad_reset_box)
    int graph_devbox;                     // the captured graph reads the box from device memory
    const double *graph_dbox;             //   ... from this pointer
    cudaGraphExec_t graph_exec;
    cudaGraphExec_t graph_exec_h;         // metad_step_host: the step on the staging buffers (waits for the F upload before the forces)
    double graph_h_rc, graph_h_box[9]; int launches_per_step_h, wait_copy;
    int graph_counts[9];                  // node counts of the captured step (metad_graph_info)
    int graph_captures, graph_updates;    // how often metad_run captured a step / updated the instantiated graph in place
    int owns_stream;                      // metad_create made the stream (cuda_stream == NULL): destroyed with the context
    double *d_hill_stage;                 // [(D + 1) * max_hills] staging of metad_set_hills / metad_get_hills with host pointers
    const void *graph_pos; void *graph_F; double graph_rc; double graph_box[9];
    long long launches; int launches_per_step;
    const void *d_pos_last;               // positions snapshot pointer of the last build (chain CVs read it)
    int *d_aux;                           // device scalars: grid-miss flag, index of the hill deposited this step
    // shared-memory tiled fast path (fp32, Q6): tile.cuh / tiled.cu
    int tiled; int tile_T[3]; int tile_cap; int tile_hx;
    int tiled64;                          // the same tiling with fp64 pair math (tiled64.cu: Q6 contexts; output in the generic formats)
    int *d_tile_cuts; int tile_cuts_key[6];    // tile boundaries per direction (device) and the (nc, nt) they were computed for
    int timing; int capturing; int timing_recorded; cudaEvent_t ev[3];
    cudaStream_t copy_stream; cudaEvent_t ev_copy;   // metad_step_host: the force upload overlaps the first three stages
    float *d_q6;                          // per-atom q6 (sorted order) [N], then f'(q6) [N], in the pair precision (double on fp64 contexts)
    float *d_cgrad;                       // tiled coordination path: per-atom sum_j 2 sw' d / (r0 r) as float4, ORIGINAL atom
                                          // order (k_tile_build<2>), scaled and added to F by k_force_add
    double *d_cvq6;                       // tiled path: [Q6 mean, solid count] finished by k_tile_build
    int list_skipped;                     // the last tiled coordination build ran list-free (lazy_neighbors)
    double *cv_direct;                    // run paths (metad_run, metad_step_host): the context's CV vector, which the last block
                                          // of k_tile_build fills itself (no k_q6_publish launch); NULL on the stage calls
};

static inline const void *ctx_last_pos(const metad_ctx *c) { return c->d_pos_last; }
static inline int *ctx_aux(const metad_ctx *c) { return c->d_aux; }

void metad_set_error(const char *msg);
#define CUDA_TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { metad_set_error(cudaGetErrorString(e_)); (void)cudaGetLastError(); return METAD_ERR_CUDA; } } while (0)

static inline int div_up(long long a, int b) { return (int)((a + b - 1) / b); }

// stage entry points implemented in the .cu files (host functions that enqueue kernels)
int nb_build(metad_ctx *c, const void *d_pos);
int geom_update(metad_ctx *c, const double *d_box);
int tiled_q6_pass1_skin(metad_ctx *c, double *d_cv);
int nb_export(metad_ctx *c, int *d_count, int *d_list);
int cv_eval_all(metad_ctx *c, double *d_cv);
int cv_forces_all(metad_ctx *c, const double *d_dVds, void *d_F);
int q6_export(metad_ctx *c, void *d_q6);
int chain_virial(metad_ctx *c, const double *d_dVds);
int lattice_eval(metad_ctx *c, double *d_cv);
int lattice_forces(metad_ctx *c, const double *d_dVds);
int mindist_eval(metad_ctx *c, double *d_cv);
int mindist_forces(metad_ctx *c, const double *d_dVds, void *d_F);
int torsion_eval_all(metad_ctx *c, double *d_cv);
int torsion_forces(metad_ctx *c, const double *d_dVds, void *d_F);
int bias_eval(metad_ctx *c, const double *d_cv, double *d_V, double *d_dVds, bool with_deposit = false);
int bias_deposit(metad_ctx *c, const double *d_cv, const double *d_V);
int bias_grid_rebuild(metad_ctx *c);
int bias_fused_torsion_step(metad_ctx *c, const void *d_pos, void *d_F);
int bias_set_hills_dev(metad_ctx *c, const double *d_centers_rowmajor, const double *d_heights, int count);
int bias_get_hills_dev(metad_ctx *c, double *d_centers_rowmajor, double *d_heights, int capacity);
int bias_batch(metad_ctx *c, const double *d_points, int T, double *d_V);
int reweight_run(metad_ctx *c, const double *d_traj, int T, const int *nbins, const double *lo, const double *hi,
                 double *d_P, double *d_F);
int tiled_init();
int tiled_build(metad_ctx *c);
int tiled_q6_pass1(metad_ctx *c, double *d_cv);
int tiled_q6_force(metad_ctx *c, const double *d_dVds, void *d_F);
int tiled_coord_force(metad_ctx *c, const double *d_dVds, void *d_F);
int tiled64_init();
int tiled64_build(metad_ctx *c);
