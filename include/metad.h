/* metad.h — C ABI of the B200-native per-step metadynamics hot path (GPU-MetaD, arxiv 2510.06873).
 *
 * One context = one simulated system on one GPU.  Per MD step the caller issues, in this order
 * (DESIGN.md §3 reading U; "end-to-end ... entirely implemented on GPUs"):
 *
 *     metad_build_neighbors -> metad_eval_cv -> metad_bias -> metad_apply_forces -> metad_deposit
 *
 * or metad_run(), which captures those five in a CUDA graph and replays it n times with zero host
 * round trips.  Every hot-path call only ENQUEUES kernels on the context's stream and returns;
 * nothing synchronises or copies to the host except the calls marked [sync].
 *
 * Pointers: "d_" = device pointer owned by the caller (never freed / reallocated by the library),
 * "h_" = host pointer.  Plain pointers without a prefix in metad_params are HOST pointers read
 * (copied) during metad_create only.  All scratch memory is allocated in metad_create.
 *
 * Precision: params.precision = 64 -> positions / forces are double[N][3]; 32 -> float[N][3]
 * ("fp32 pair math with fp64 reductions", BASELINE.json configs[4]).  CV values, V, dV/ds, hills,
 * grid and all reductions are double in both modes.
 *
 * Box: 9 doubles on the HOST, rows a=(ax,0,0), b=(bx,by,0), c=(cx,cy,cz) (lower-triangular;
 * orthorhombic = diagonal).  Positions must lie in the primary cell (fractional coords in [0,1),
 * up to rounding).  Requires rc < half of every perpendicular box width (else METAD_ERR_BOX).
 *
 * Return value: 0 (METAD_OK) or a metad_error.  Device-side conditions (neighbour-list overflow,
 * hill-array overflow, grid out of range, non-finite CV) never abort: they set sticky bits read by
 * metad_status(), and the kernels continue with defined behaviour (excess neighbours / hills are
 * dropped, out-of-grid points fall back to the exact hill sum).
 */
#ifndef METAD_B200_H
#define METAD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct metad_ctx metad_ctx;

enum metad_error { METAD_OK = 0, METAD_ERR_ARG = 1, METAD_ERR_BOX = 2, METAD_ERR_STATE = 3,
                   METAD_ERR_CUDA = 4, METAD_ERR_NOMEM = 5 };

enum metad_dev_bits { METAD_DEV_NEIGH_OVERFLOW = 1, METAD_DEV_HILL_OVERFLOW = 2,
                      METAD_DEV_GRID_RANGE = 4, METAD_DEV_NONFINITE = 8,
                      METAD_DEV_POS_RANGE = 16 /* a position lies outside the primary cell */,
                      METAD_DEV_TRAJ_FULL = 32 /* the recorded CV trajectory is full, later frames are dropped */,
                      METAD_DEV_BOX = 64 /* device-resident box (metad_*_dev calls): not lower-triangular / not positive, rc not
                                            below half of every perpendicular width, or the box shrank so far that a cell of the
                                            frozen cell grid is narrower than rc — neighbour sets of that step are not valid;
                                            call metad_reset_box and repeat the step */ };

enum metad_cv_kind {
    METAD_CV_COORD = 0,    /* s = scale * sum_{i in A} sum_{j in B, j!=i, r<rc} sw(r_ij/r0),
                              sw(x) = (1-x^n)/(1-x^m)           (BASELINE.json configs[0],[2]) */
    METAD_CV_Q6_MEAN = 1,  /* s = scale * sum_i q6(i), Steinhardt q6 over hard-cutoff neighbours
                              (BASELINE.json configs[3]; reading E); scale = 1/N for the mean   */
    METAD_CV_Q6_SOLID = 2, /* s = scale * sum_i 1/(1+exp(-(q6(i)-q_thresh)/q_width))
                              (BASELINE.json configs[4]; reading F)                                        */
    METAD_CV_RGYR = 3,     /* radius of gyration of an ordered chain, unwrapped by sequential minimum
                              image (BASELINE.json configs[1]; reading G)                                  */
    METAD_CV_CONTACTS = 4, /* s = scale * sum_p sw(r_p / r0_p), n, m as given (configs[1]; reading H)      */
    METAD_CV_MINDIST = 6,  /* s = min over i in A, j in B, j != i, r_ij < rc of the minimum-image distance; forces act on the
                              nearest pair only (the derivative of a minimum is that of its arg-min, which is what automatic
                              differentiation returns); nobody within rc: s = rc, no force
                              ("distance between a surface oxygen atom and its nearest hydrogen atom"; reading AA).
                              Groups as for COORD.  A context may hold several COORD / MINDIST CVs, each with its own groups    */
    METAD_CV_LATTICE = 7,  /* s = |h_k|, the length of box row k = cv.n in {0, 1, 2} ("the triaxial lattice parameters as
                              CVs"; reading AB).  No atomic forces: the bias acts on the cell, see metad_get_box_force          */
    METAD_CV_TORSION = 5   /* dihedral angle of atoms torsion[0..3] in (-pi, pi], IUPAC sign, minimum-image bonds
                              ("Phi(C-N-Ca-C) and Psi(N-Ca-C-N) serve as the CVs"; reading V).
                              Normally used with params.period = 2 pi for that dimension                  */
};

typedef struct {
    int kind;                       /* metad_cv_kind */
    int n, m;                       /* switching exponents (COORD, CONTACTS) */
    double r0;                      /* switching length (COORD) */
    double scale;                   /* normalisation, see metad_cv_kind */
    const int *group_a; int n_a;    /* COORD, MINDIST: host index lists; NULL = all atoms */
    const int *group_b; int n_b;
    const int *pairs;               /* CONTACTS: host int[2*npairs] */
    const double *pair_r0;          /* CONTACTS: host double[npairs] */
    int npairs;
    const int *chain; int nchain;   /* RGYR: host ordered atom indices */
    const double *mass;             /* RGYR: host double[nchain] or NULL (equal masses) */
    double q_thresh, q_width;       /* Q6_SOLID */
    int torsion[4];                 /* TORSION: atom indices i, j, k, l */
} metad_cv_desc;

#define METAD_MAX_CV 4

typedef struct {
    int natoms;
    int precision;                  /* 32 or 64: dtype of pos / F and of the pair arithmetic */
    int max_neigh;                  /* neighbour-list capacity per atom */
    int ncv;                        /* 1..METAD_MAX_CV */
    metad_cv_desc cv[METAD_MAX_CV];
    double sigma[METAD_MAX_CV];     /* Gaussian width per CV dimension */
    double w0;                      /* initial hill height (PAPER.md:37 W_k) */
    double kT;                      /* k_B T in the hill energy unit */
    double bias_factor;             /* gamma; <= 1 -> plain metadynamics (reading I) */
    int max_hills;                  /* hill-array capacity */
    int stride;                     /* deposit every `stride` steps; 0 = never ("periodically") */
    int grid_n[2];                  /* grid_n[0] == 0 -> exact hill sum; else ncv must be 2 (reading M) */
    double grid_lo[2], grid_hi[2];
    double force_scale;             /* F += -force_scale * dV/dr (unit conversion; reading N) */
    double period[METAD_MAX_CV];    /* > 0: the CV dimension is periodic with this period (PAPER.md:37 torsions: 2 pi);
                                       (s - s_tau) in PAPER.md:81 is then the nearest-image difference (reading W).
                                       With a grid, a periodic dimension needs grid_hi - grid_lo == period and has
                                       grid_n nodes at lo + i * period / grid_n, no "outside" (reading X).  0: not periodic */
    int traj_capacity;              /* > 0: every metad_deposit also appends the step's CV values to a device-resident trajectory
                                       of this many frames ("GSTA" keeps the CV outputs aligned with the MD run;
                                       PAPER.md:85-87 reweights them) — see metad_reweight_recorded.  Full: METAD_DEV_TRAJ_FULL */
    int lazy_neighbors;             /* != 0: metad_build_neighbors only snapshots the positions when no CV of the context reads the
                                       neighbour list (torsion / Rg / contacts / lattice CVs): a 22-atom torsion step is pure
                                       launch latency and the list build is half of its launches.  An ungrouped coordination
                                       number in fp32 (tiled path, no virial) then runs list-free as well: the candidate scan
                                       accumulates the sum and the per-atom gradient and stores no list.  metad_get_neighbors
                                       returns METAD_ERR_STATE in both cases.  0 (default): always built */
    int want_virial;                /* != 0: metad_apply_forces also computes the bias virial (metad_get_virial) for NPT runs
                                       (reading AD), for every CV kind */
    double skin;                    /* > 0: Verlet-skin reuse of the neighbour list.  The list is built with
                                       the cutoff rc + skin and kept while no atom has moved more than skin / 2 from where it was
                                       at the build (checked on the device every step: no host read, the rebuild decision is taken
                                       inside the captured graph); every CV / force kernel filters the pairs with the canonical
                                       predicate r < rc on the current positions, so CVs, forces and metad_get_neighbors are those
                                       of the exact rc list at every step.  max_neigh must hold the rc + skin list; the box needs
                                       rc + skin < half of every perpendicular width.  Supported by the list CVs (COORD, Q6_*,
                                       MINDIST).  The two rebuild flags alternate with the step counter that metad_deposit
                                       advances: a caller of the stage calls who never calls metad_deposit gets a rebuild in every
                                       step after the first one that needed it.  0 (default): the list is rebuilt every step */
    double box_slack;               /* metad_*_dev calls: the cell grid is derived ONCE (first call / after metad_reset_box) with
                                       cells at least rc (1 + box_slack) wide, so the device-resident box may shrink by that
                                       fraction before METAD_DEV_BOX is raised; 0 = cells as small as rc allows */
    double fill_fraction;           /* fraction of the box volume the atoms occupy, in (0, 1]; 0 (default) = 1.  A rank of a slab
                                       decomposition holds its slab + halo in the GLOBAL box: the shared-memory
                                       tiles are sized for natoms / (fill_fraction * cells) atoms per cell instead of the box average */
    double c_window_lo;             /* read when fill_fraction < 1: every atom has its fractional c-coordinate in the window
                                       [c_window_lo, c_window_lo + fill_fraction) modulo 1 (the slab + halo of the rank); only the
                                       tiles of that window are launched.  An atom outside it raises METAD_DEV_POS_RANGE */
} metad_params;

/* Creates a context on the current CUDA device; `cuda_stream` is the cudaStream_t on which every later call is enqueued.
 * NULL: the library creates a private NON-BLOCKING stream for the context (owned by it, destroyed by metad_destroy) — the
 * legacy default stream cannot be captured into a CUDA graph, which metad_run needs.  Work of the caller on other streams
 * (the legacy default stream included) is then NOT ordered with the library's kernels: order it with metad_synchronize()
 * or any [sync] call before reading results, and finish writing d_pos / d_F before calling in.
 * On failure nothing stays allocated.  [sync] */
int metad_create(metad_ctx **out, const metad_params *params, void *cuda_stream);
int metad_destroy(metad_ctx *ctx);

/* a1 (BASELINE.json north_star "build the neighbour list"; reading O, P): bins atoms into cells,
 * counting-sorts them, and builds the full neighbour list (all j != i with minimum-image
 * r_ij < rc, strict).  d_pos: [N][3] in params.precision; the pointer is kept, not the data: the chain, torsion and
 * nearest-distance CVs (and their forces / virial) read d_pos again in metad_eval_cv / metad_apply_forces, so the caller must
 * leave d_pos unmodified until the metad_apply_forces of this step has completed (the neighbour-list CVs work on the
 * cell-sorted copy made here).  box: host.  Errors: METAD_ERR_BOX, METAD_ERR_ARG. */
int metad_build_neighbors(metad_ctx *ctx, const void *d_pos, const double *h_box, double rc);

/* a2-a4: evaluates all CVs; d_cv: double[ncv] (device, caller-owned). */
int metad_eval_cv(metad_ctx *ctx, double *d_cv);

/* a5: V(s) = sum_k w_k prod_d exp(-(s_d-c_kd)^2/(2 sigma_d^2)) and dV/ds_d at
 * the point d_cv[ncv] over the hills deposited so far (through the grid if enabled).
 * d_V: double[1], d_dVds: double[ncv]. */
int metad_bias(metad_ctx *ctx, const double *d_cv, double *d_V, double *d_dVds);

/* a6: F_i += -force_scale * sum_d d_dVds[d] * d s_d / d r_i for the CVs evaluated
 * by the last metad_eval_cv.  Gather form, deterministic, no float atomics.
 * d_F: [N][3] in params.precision, read-modify-write. */
int metad_apply_forces(metad_ctx *ctx, const double *d_dVds, void *d_F);

/* a7 ("periodically depositing"; PAPER.md:43 well-tempered; readings I, J, U):
 * advances the device step counter; if (step % stride == 0) appends the hill
 * (d_cv, w0 * exp(-V/((gamma-1) kT))) and, in grid mode, adds it to the table. */
int metad_deposit(metad_ctx *ctx, const double *d_cv, const double *d_V);

/* The five calls above for nsteps steps as one CUDA graph replayed nsteps times (fixed d_pos:
 * positions are an input of this library, the MD integrator is out of scope).  Results of the last
 * step are in the context (metad_get_state). */
int metad_run(metad_ctx *ctx, const void *d_pos, const double *h_box, double rc, void *d_F, int nsteps);

/* NEXT-3 ("ran NPT simulation at 300K and 50 GPa" with lattice parameters as CVs; PAPER.md:61 on the cost of
 * GPU-CPU transfers) — the box lives in DEVICE memory (d_box: double[9], same convention as h_box) and may change every step
 * without the host ever seeing it: a kernel derives the step's geometry from it, every other kernel reads that.  The cell
 * grid and tiling are derived from the box ONCE ([sync]: one 72-byte read on the first call, or the first call after
 * metad_reset_box) and then frozen, so metad_run_dev captures its CUDA graph once and replays it for every later box; a box
 * that has become invalid for the frozen grid raises the sticky bit METAD_DEV_BOX instead of an error code.  The two calls
 * otherwise behave like metad_build_neighbors / metad_run; stage calls that follow metad_build_neighbors_dev use its box. */
int metad_build_neighbors_dev(metad_ctx *ctx, const void *d_pos, const double *d_box, double rc);
int metad_run_dev(metad_ctx *ctx, const void *d_pos, const double *d_box, double rc, void *d_F, int nsteps);
/* Forget the frozen cell grid (and the captured graph): the next *_dev call derives it again from the then current box. */
int metad_reset_box(metad_ctx *ctx);

/* One step with HOST buffers (end-to-end path): copies h_pos -> device, h_F -> device (on a second stream, while the
 * neighbour build, the CVs and the bias run), runs the five stages as one captured graph on the library's staging buffers
 * (re-captured only when h_box or rc changes), copies F, cv[ncv] and V back.  [sync] */
int metad_step_host(metad_ctx *ctx, const void *h_pos, const double *h_box, double rc, void *h_F,
                    double *h_cv, double *h_V);

/* Page-locked host memory for the buffers of metad_step_host (cudaHostAlloc, default flags; *ptr is owned by the caller
 * until metad_host_free).  Any host pointer works with metad_step_host, but pageable memory is staged by the driver, and
 * memory pinned after the fact has been measured at 12-19 GB/s host -> device on the test machine against 54 GB/s for
 * these buffers.  bytes == 0 or ptr == NULL: METAD_ERR_ARG; allocation failure: METAD_ERR_CUDA. */
int metad_host_alloc(void **ptr, size_t bytes);
int metad_host_free(void *ptr);

/* [sync] ORs the sticky device bits into *bits (and clears nothing). */
int metad_status(metad_ctx *ctx, unsigned *bits);

/* [sync] last step's cv[ncv], V, dVds[ncv], step counter, hill count (any pointer may be NULL). */
int metad_get_state(metad_ctx *ctx, double *h_cv, double *h_V, double *h_dVds, int *h_step, int *h_nhills);

/* Neighbour list in ORIGINAL atom indices: d_count int[N], d_list int[N][max_neigh] row-major
 * (unused slots = -1, order within a row unspecified).  Enqueued, not synchronised. */
int metad_get_neighbors(metad_ctx *ctx, int *d_count, int *d_list);

/* Per-atom q6 of the last metad_eval_cv in original atom order (d_q6: [N] in params.precision). */
int metad_get_q6(metad_ctx *ctx, void *d_q6);

/* Hills: centers [count][ncv] row-major, heights [count].  on_device: pointers are device (1) or
 * host (0).  set_hills replaces all hills (and rebuilds the grid table).  [sync] */
int metad_set_hills(metad_ctx *ctx, const double *centers, const double *heights, int count, int on_device);
int metad_get_hills(metad_ctx *ctx, double *centers, double *heights, int capacity, int *count, int on_device);

/* Grid table [4][n0][n1] = V, dV/ds0, dV/ds1, d2V/ds0ds1 at the nodes; copied to d_table. */
int metad_get_grid(metad_ctx *ctx, double *d_table);

/* NEXT-2 — batched bias: V_b at npoints CV points (d_points: double[npoints][ncv], d_V: double[npoints]) by the exact
 * hill sum over the hills deposited so far (periodic dimensions by nearest image).  Enqueued. */
int metad_bias_batch(metad_ctx *ctx, const double *d_points, int npoints, double *d_V);

/* NEXT-2 — free-energy reconstruction by reweighting:
 *     P(s) = < delta[s - s(R)] e^{V_b(s)/kT} > / < e^{V_b(s)/kT} >,   F(s) = -kT log P(s),
 * averages over the nframes CV frames d_traj (double[nframes][ncv], ncv = 1 or 2) of a biased run, V_b = the current
 * hills.  The delta is a histogram (reading Z): h_nbins[d] uniform bins on [h_lo[d], h_hi[d]) (periodic
 * dimensions are wrapped first and need hi - lo == period); frames outside a non-periodic range count in the
 * denominator only.  d_P, d_F: double[nbins0 * nbins1] row-major (nbins1 = 1 if ncv = 1); empty bins: P = 0, F = +inf.
 * Weights are accumulated per bin, relative to the largest weight of that bin, as 2^-64 fixed point in 128-bit integer
 * sums (integer atomics: bit-identical from run to run; up to 2^63 frames per bin), and the bins are combined in log space:
 * a bin any number of kT below the most probable one keeps full precision, and F is finite for every bin that holds a frame
 * (P may underflow to 0 there).  Not a per-step call: allocates and frees its scratch (V and bin per frame, bins).  [sync] */
int metad_reweight(metad_ctx *ctx, const double *d_traj, int nframes, const int *h_nbins, const double *h_lo,
                   const double *h_hi, double *d_P, double *d_F);

/* Bias force on the cell for NPT integrators (reading AB): F_h[3][3] = -force_scale * sum_d dVds[d] * d s_d/d h
 * of the last metad_apply_forces, h = the box rows; non-zero only for METAD_CV_LATTICE dimensions.  Copied to d_out9
 * (device double[9]); enqueued, not synchronised. */
int metad_get_box_force(metad_ctx *ctx, double *d_out9);

/* Bias virial of the last metad_apply_forces (needs params.want_virial): W[3][3] = -force_scale * sum_d dVds[d] * d s_d/d eps,
 * eps = homogeneous strain of positions and box (PAPER.md:51 NPT; reading AD); energy units, its contribution to the pressure
 * tensor is W / volume.  Copied to d_out9 (device double[9], row-major); enqueued, not synchronised. */
int metad_get_virial(metad_ctx *ctx, double *d_out9);

/* metad_reweight over the CV frames recorded on the device since the last metad_reset_steps (params.traj_capacity > 0):
 * the frames never leave the GPU.  h_nframes (may be NULL) receives the number of frames used.  [sync] */
int metad_reweight_recorded(metad_ctx *ctx, const int *h_nbins, const double *h_lo, const double *h_hi, double *d_P,
                            double *d_F, int *h_nframes);

/* Resets the step counter and the recorded trajectory (hills stay). */
int metad_reset_steps(metad_ctx *ctx);

/* Kernel-level timing for bench.py: when enabled, metad_build_neighbors records CUDA events around its
 * sort phase (binning, scan, scatter, in-cell sort + gather) and its list phase (candidate scan; on the tiled
 * paths, fp32 and fp64, fused with Q6 pass 1).  metad_get_timing [sync] returns the last two durations in ms.
 * Not usable inside metad_run (events are not recorded during graph capture). */
int metad_set_timing(metad_ctx *ctx, int enabled);
int metad_get_timing(metad_ctx *ctx, float *h_ms_sort, float *h_ms_list);

/* Number of kernels the library has launched on this context so far (graph replays included). */
long long metad_launch_count(metad_ctx *ctx);

/* [sync] Number of neighbour-list builds (cell sort + list) the context has executed so far: with params.skin > 0 fewer than
 * the number of steps.  The count lives on the device; the rebuild decision itself is never read by the host. */
int metad_get_rebuilds(metad_ctx *ctx, int *h_count);

/* [sync] Waits for everything enqueued on the context's stream (the way to order a context created with cuda_stream ==
 * NULL against the caller's own work). */
int metad_synchronize(metad_ctx *ctx);

/* Proof of the zero-host-copy step (BASELINE.json north_star: "a multi-step loop makes zero host round-trips"; PAPER.md:61 on
 * GPU-CPU transfer overhead): node counts of the CUDA graph metad_run captured last.
 * h_counts: int[9] = { nodes, kernel nodes, memcpy nodes, memset nodes, host nodes, other nodes,
 *                      captures so far, in-place graph updates so far, conditional nodes }.
 * With params.skin > 0 the graph holds ONE conditional IF node whose body (the list-build kernels) runs only in the steps
 * whose displacement check asks for a rebuild; the condition is set on the device (cudaGraphSetConditional).
 * Errors: METAD_ERR_STATE before the first metad_run. */
int metad_graph_info(metad_ctx *ctx, int *h_counts);

/* Scalar-pipe roofline denominators: dependent-free FMA chains on every SM of the current device,
 * timed with CUDA events, best of four launches after two warm-up launches.  kind 0: fp32 FFMA, 1: fp32 FFMA2 (packed pairs,
 * sm_100), 2: fp64 DFMA.  *h_tflops: achieved TFLOP/s (an FMA = 2 flop); *h_ms (may be NULL): duration of that launch.
 * Needs no context.  [sync] */
int metad_fma_peak(int kind, double *h_tflops, double *h_ms);

/* The hill sum V(s), dV/ds (reading W for periodic dimensions) WITHOUT a context and WITHOUT any allocation: for
 * callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).  The call
 * makes no cudaMalloc / cudaFree and uses no allocating library routine; its scratch (one row of partial sums per 2,048 hills +
 * the ticket of the fixed-order reduction) is a file-scope __device__ array of METAD_NOALLOC_SCRATCH_BYTES that every GPU
 * loading this library holds until the process exits.
 *   d_centers  device, [ncv][ld_centers] doubles: centre of hill k in dimension d at d_centers[d * ld_centers + k]
 *   d_heights  device, [nhills] doubles;   nhills  0..METAD_NOALLOC_MAX_HILLS (more: METAD_ERR_ARG, the message names the limit)
 *   h_sigma    host, [ncv] Gaussian widths (> 0);   h_period  host, [ncv] periods (0: not periodic) or NULL
 *   d_cv       device, [ncv] the point s;   d_V  device, 1 double (out);   d_dVds  device, [ncv] doubles (out)
 *   cuda_stream  the cudaStream_t to enqueue on (NULL: the default stream).  [async]: a memset of the ticket and one kernel;
 *                all device arrays stay owned by the caller and must stay valid until the work has completed.
 * Every call shares the one scratch array, which keeps the last call's contents (the call clears what must start at zero):
 * calls that OVERLAP on the GPU — different streams with no ordering between them, or several host threads — race on it.
 * The result equals metad_bias's up to the order of the fp64 sum (another fixed order: run-to-run identical).
 * Errors: METAD_ERR_ARG (null pointer, ncv outside 1..METAD_MAX_CV, nhills beyond the limit, ld_centers < nhills,
 * sigma <= 0), METAD_ERR_CUDA. */
#define METAD_NOALLOC_MAX_HILLS 1048576
#define METAD_NOALLOC_SCRATCH_BYTES 20736
int metad_bias_noalloc(const double *d_centers, int ld_centers, const double *d_heights, int nhills, int ncv,
                       const double *h_sigma, const double *h_period, const double *d_cv, double *d_V, double *d_dVds,
                       void *cuda_stream);

/* Slab decomposition over several GPUs: after metad_eval_cv, replaces the Q6 CVs in
 * d_cv (device, [ncv]) by their sums over the atoms this rank OWNS — d_owned: device, natoms bytes, != 0 for an owned atom,
 * indexed like d_pos.  The ranks then add their d_cv (one all-reduce of ncv doubles) and go on with metad_bias /
 * metad_apply_forces / metad_deposit on the same global s.  Fixed-order sum (run-to-run identical).  On the tiled fp32 path
 * (fill_fraction < 1) the metad_apply_forces of the SAME step then skips the atoms that are not owned: their rows of d_F
 * belong to other ranks and get nothing added.  [async]
 * Errors: METAD_ERR_STATE unless every CV dimension of the context is a Q6 CV and the CVs have been evaluated. */
int metad_cv_owned_sum(metad_ctx *ctx, const unsigned char *d_owned, double *d_cv);

const char *metad_version(void);
const char *metad_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
