// api.cu — the C ABI of include/metad.h: context, argument checks, CUDA-graph step loop.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <vector>
#include "common.cuh"
#include "tile.cuh"

static thread_local char g_err[512] = "";
void metad_set_error(const char *msg) { snprintf(g_err, sizeof(g_err), "%s", msg ? msg : ""); }
extern "C" const char *metad_last_error(void) { return g_err; }
extern "C" const char *metad_version(void) { return "metad-b200 0.1 (sm_100a)"; }


#define FAIL(code, msg) do { metad_set_error(msg); return code; } while (0)

template <typename X>
static cudaError_t dev_alloc(X **p, size_t n) { return cudaMalloc((void **)p, sizeof(X) * (n ? n : 1)); }

static int upload_ints(int **dst, const int *src, size_t n) {
    CUDA_TRY(dev_alloc(dst, n));
    CUDA_TRY(cudaMemcpy(*dst, src, sizeof(int) * n, cudaMemcpyHostToDevice));
    return METAD_OK;
}
static int upload_doubles(double **dst, const double *src, size_t n) {
    CUDA_TRY(dev_alloc(dst, n));
    CUDA_TRY(cudaMemcpy(*dst, src, sizeof(double) * n, cudaMemcpyHostToDevice));
    return METAD_OK;
}

static int create_impl(metad_ctx *c, const metad_params *p, void *cuda_stream);

extern "C" int metad_create(metad_ctx **out, const metad_params *p, void *cuda_stream) {
    if (!out || !p) FAIL(METAD_ERR_ARG, "null argument");
    if (p->natoms <= 0) FAIL(METAD_ERR_ARG, "natoms must be positive");
    if (p->precision != 32 && p->precision != 64) FAIL(METAD_ERR_ARG, "precision must be 32 or 64");
    if (p->ncv < 1 || p->ncv > METAD_MAX_CV) FAIL(METAD_ERR_ARG, "ncv out of range");
    if (p->max_neigh < 1 || p->max_hills < 1) FAIL(METAD_ERR_ARG, "max_neigh / max_hills must be positive");
    for (int d = 0; d < p->ncv; ++d) {
        if (!(p->sigma[d] > 0.0)) FAIL(METAD_ERR_ARG, "sigma must be positive");
        if (!(p->period[d] >= 0.0)) FAIL(METAD_ERR_ARG, "period must be >= 0");
        if (p->grid_n[0] != 0 && d < 2 && p->period[d] > 0.0 &&
            fabs((p->grid_hi[d] - p->grid_lo[d]) - p->period[d]) > 1e-12 * p->period[d])
            FAIL(METAD_ERR_ARG, "a periodic grid dimension needs grid_hi - grid_lo == period");
    }
    if (p->grid_n[0] != 0 && (p->ncv != 2 || p->grid_n[0] < 2 || p->grid_n[1] < 2 ||
                              !(p->grid_hi[0] > p->grid_lo[0]) || !(p->grid_hi[1] > p->grid_lo[1])))
        FAIL(METAD_ERR_ARG, "grid needs ncv == 2, n >= 2 and hi > lo");
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0)
        FAIL(METAD_ERR_CUDA, "no CUDA device: this library has no CPU fallback");

    if (tiled_init() || tiled64_init()) return METAD_ERR_CUDA;
    metad_ctx *c = new metad_ctx();
    memset(c, 0, sizeof(*c));
    // every failure below leaves through ONE path that frees whatever was allocated so far (metad_destroy works on a
    // partially built context: all members start as zero)
    const int r = create_impl(c, p, cuda_stream);
    if (r != METAD_OK) {
        char keep[sizeof(g_err)];
        snprintf(keep, sizeof(keep), "%s", g_err);
        metad_destroy(c);
        metad_set_error(keep);
        return r;
    }
    *out = c;
    return METAD_OK;
}

static int create_impl(metad_ctx *c, const metad_params *p, void *cuda_stream) {
    c->p = *p;
    c->N = p->natoms; c->prec = p->precision; c->maxn = p->max_neigh; c->D = p->ncv;
    if (c->p.force_scale == 0.0) c->p.force_scale = 1.0;
    c->stream = (cudaStream_t)cuda_stream;
    if (!c->stream) {                             // include/metad.h: NULL = a private non-blocking stream owned by the context
        CUDA_TRY(cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking));
        c->owns_stream = 1;
    }
    c->q6_mean_dim = c->q6_solid_dim = c->coord_dim = c->mindist_dim = -1;
    const int N = c->N;
    const size_t tsz = c->prec == 32 ? sizeof(float) : sizeof(double);

    // ---- CV descriptors
    std::vector<unsigned char> flags;
    for (int d = 0; d < c->D; ++d) {
        const metad_cv_desc &s = p->cv[d];
        CvDev &v = c->cv[d];
        v.kind = s.kind; v.n = s.n; v.m = s.m; v.r0 = s.r0; v.scale = s.scale;
        v.q_thresh = s.q_thresh; v.q_width = s.q_width;
        switch (s.kind) {
        case METAD_CV_COORD:
        case METAD_CV_MINDIST: {
            // any number of them (up to METAD_MAX_CV): every list CV owns two bits (in A, in B) of the per-atom flag byte
            v.fshift = 2 * (c->n_coord + c->n_mindist);
            if (s.kind == METAD_CV_COORD) {
                if (!(s.r0 > 0.0) || s.n < 1 || s.m <= s.n) FAIL(METAD_ERR_ARG, "COORD needs r0 > 0, 0 < n < m");
                if (c->coord_dim < 0) c->coord_dim = d;
                c->has_coord = true; c->n_coord++;
            } else {
                if (c->mindist_dim < 0) c->mindist_dim = d;
                c->has_mindist = true; c->n_mindist++;
                if (s.group_a && s.group_b && s.n_a > 0 && s.n_b > 0) {      // list-free variant needs explicit groups
                    v.n_ga = s.n_a; v.n_gb = s.n_b;
                    if (upload_ints(&v.d_ga, s.group_a, s.n_a) || upload_ints(&v.d_gb, s.group_b, s.n_b)) return METAD_ERR_CUDA;
                }
            }
            v.use_groups = s.group_a || s.group_b;
            if (s.group_a) for (int k = 0; k < s.n_a; ++k) if (s.group_a[k] < 0 || s.group_a[k] >= N) FAIL(METAD_ERR_ARG, "group index");
            if (s.group_b) for (int k = 0; k < s.n_b; ++k) if (s.group_b[k] < 0 || s.group_b[k] >= N) FAIL(METAD_ERR_ARG, "group index");
            break;
        }
        case METAD_CV_Q6_MEAN:
            if (c->q6_mean_dim >= 0) FAIL(METAD_ERR_ARG, "only one Q6_MEAN CV per context");
            c->q6_mean_dim = d; c->has_q6 = true; break;
        case METAD_CV_Q6_SOLID:
            if (c->q6_solid_dim >= 0) FAIL(METAD_ERR_ARG, "only one Q6_SOLID CV per context");
            if (!(s.q_width > 0.0)) FAIL(METAD_ERR_ARG, "q_width must be positive");
            c->q6_solid_dim = d; c->has_q6 = true; break;
        case METAD_CV_RGYR: {
            if (!s.chain || s.nchain < 1) FAIL(METAD_ERR_ARG, "RGYR needs a chain");
            for (int k = 0; k < s.nchain; ++k) if (s.chain[k] < 0 || s.chain[k] >= N) FAIL(METAD_ERR_ARG, "chain index");
            v.nchain = s.nchain;
            if (upload_ints(&v.d_chain, s.chain, s.nchain)) return METAD_ERR_CUDA;
            if (s.mass && upload_doubles(&v.d_mass, s.mass, s.nchain)) return METAD_ERR_CUDA;
            CUDA_TRY(dev_alloc(&v.d_unwrapped, 3 * (size_t)s.nchain + 8));
            break;
        }
        case METAD_CV_CONTACTS: {
            if (!s.pairs || !s.pair_r0 || s.npairs < 1 || s.n < 1 || s.m <= s.n) FAIL(METAD_ERR_ARG, "CONTACTS needs pairs, r0, 0 < n < m");
            v.npairs = s.npairs;
            std::vector<std::pair<int, int>> inc;   // (atom, pair)
            for (int q = 0; q < s.npairs; ++q) {
                int a = s.pairs[2 * q], b = s.pairs[2 * q + 1];
                if (a < 0 || a >= N || b < 0 || b >= N || a == b) FAIL(METAD_ERR_ARG, "pair index");
                inc.push_back({ a, q }); inc.push_back({ b, q });
            }
            std::sort(inc.begin(), inc.end());
            std::vector<int> atoms, off, prs;
            for (size_t t = 0; t < inc.size(); ++t) {
                if (t == 0 || inc[t].first != inc[t - 1].first) { atoms.push_back(inc[t].first); off.push_back((int)t); }
                prs.push_back(inc[t].second);
            }
            off.push_back((int)inc.size());
            v.ncatoms = (int)atoms.size();
            if (upload_ints(&v.d_pairs, s.pairs, 2 * (size_t)s.npairs) || upload_doubles(&v.d_pair_r0, s.pair_r0, s.npairs) ||
                upload_ints(&v.d_catoms, atoms.data(), atoms.size()) || upload_ints(&v.d_csr_off, off.data(), off.size()) ||
                upload_ints(&v.d_csr_pair, prs.data(), prs.size()))
                return METAD_ERR_CUDA;
            break;
        }
        case METAD_CV_LATTICE:
            if (s.n < 0 || s.n > 2) FAIL(METAD_ERR_ARG, "LATTICE needs an axis n in {0, 1, 2}");
            c->has_lattice = true;
            break;
        case METAD_CV_TORSION: {
            for (int k = 0; k < 4; ++k) {
                if (s.torsion[k] < 0 || s.torsion[k] >= N) FAIL(METAD_ERR_ARG, "torsion index");
                for (int q = 0; q < k; ++q) if (s.torsion[q] == s.torsion[k]) FAIL(METAD_ERR_ARG, "torsion atoms must be distinct");
                v.tors[k] = s.torsion[k];
            }
            c->has_torsion = true;
            break;
        }
        default: FAIL(METAD_ERR_ARG, "unknown CV kind");
        }
    }

    // group flags: needed as soon as a list CV has groups or there is more than one list CV (a context with ONE ungrouped
    // list CV keeps w = 3 in the sorted positions and no flag array)
    {
        bool need = c->n_coord + c->n_mindist > 1;
        for (int d = 0; d < c->D; ++d) need = need || c->cv[d].use_groups;
        if (need) {
            flags.assign(N, 0);
            for (int d = 0; d < c->D; ++d) {
                const metad_cv_desc &s = p->cv[d];
                if (s.kind != METAD_CV_COORD && s.kind != METAD_CV_MINDIST) continue;
                const unsigned char ba = (unsigned char)(1u << c->cv[d].fshift), bb = (unsigned char)(2u << c->cv[d].fshift);
                if (s.group_a) for (int k = 0; k < s.n_a; ++k) flags[s.group_a[k]] |= ba;
                else for (int i = 0; i < N; ++i) flags[i] |= ba;
                if (s.group_b) for (int k = 0; k < s.n_b; ++k) flags[s.group_b[k]] |= bb;
                else for (int i = 0; i < N; ++i) flags[i] |= bb;
            }
        }
    }
    if (c->has_mindist) CUDA_TRY(dev_alloc(&c->d_mind, 8 * METAD_MAX_CV));
    if (p->traj_capacity < 0) FAIL(METAD_ERR_ARG, "traj_capacity must be >= 0");
    if (p->traj_capacity > 0) CUDA_TRY(dev_alloc(&c->d_traj, (size_t)p->traj_capacity * c->D));
    if (p->want_virial) {
        CUDA_TRY(dev_alloc(&c->d_virial, 9));
        CUDA_TRY(cudaMemset(c->d_virial, 0, sizeof(double) * 9));
        CUDA_TRY(dev_alloc(&c->d_vir_partials, 9 * ((size_t)div_up(N, 128) + 1)));
    }
    CUDA_TRY(dev_alloc(&c->d_cvq6, 2));
    CUDA_TRY(dev_alloc(&c->d_box_force, 9));
    CUDA_TRY(cudaMemset(c->d_box_force, 0, sizeof(double) * 9));
    if (c->has_torsion) {
        std::vector<int> ta;
        for (int d = 0; d < c->D; ++d)
            if (c->cv[d].kind == METAD_CV_TORSION) for (int k = 0; k < 4; ++k) ta.push_back(c->cv[d].tors[k]);
        std::sort(ta.begin(), ta.end());
        ta.erase(std::unique(ta.begin(), ta.end()), ta.end());
        c->ntors_atoms = (int)ta.size();
        if (upload_ints(&c->d_tors_atoms, ta.data(), ta.size())) return METAD_ERR_CUDA;
        CUDA_TRY(dev_alloc(&c->d_tors_grad, 12 * METAD_MAX_CV));
    }
    // ---- buffers (everything the hot path needs; nothing is allocated later)
    // fill_fraction < 1 (a rank of a slab decomposition: N atoms in that fraction of the GLOBAL box): cells and tiles cover the
    // whole box, so their tables are sized for the N / fill_fraction atoms a full box of this density would hold
    const double fill = p->fill_fraction > 0.0 ? p->fill_fraction : 1.0;
    const long long n_full = (long long)ceil((double)N / fill);
    if (n_full > (1ll << 29)) FAIL(METAD_ERR_ARG, "natoms / fill_fraction too large");
    c->cell_cap = (int)std::max(4 * n_full, 4096ll);
    c->nblocks_atoms = div_up((int)n_full, 128) + 1;
    int max_pair_blocks = 1;
    for (int d = 0; d < c->D; ++d) max_pair_blocks = std::max(max_pair_blocks, div_up(c->cv[d].npairs, 256) + 1);
    CUDA_TRY(dev_alloc(&c->d_cell_count, (size_t)c->cell_cap + 1));
    CUDA_TRY(cudaMemset(c->d_cell_count, 0, sizeof(int) * ((size_t)c->cell_cap + 1)));
    CUDA_TRY(dev_alloc(&c->d_cell_start, (size_t)c->cell_cap + 1));
    CUDA_TRY(dev_alloc(&c->d_block_sums, (size_t)c->cell_cap / 1024 + 8));
    CUDA_TRY(dev_alloc(&c->d_cell_of, N));
    CUDA_TRY(dev_alloc(&c->d_slot, N));
    CUDA_TRY(dev_alloc(&c->d_perm, N));
    CUDA_TRY(dev_alloc(&c->d_perm_raw, 2 * (size_t)N));      // (atom, cell) pairs in raw counting-sort order
    CUDA_TRY(dev_alloc(&c->d_scell, N));
    CUDA_TRY(cudaMalloc(&c->d_spos, 4 * tsz * (size_t)N));
    CUDA_TRY(dev_alloc(&c->d_nl_count, N));
    // the tiled path stores the list in slabs of 32 atoms x maxn entries (tile.cuh: nl_slot): the last slab is a whole one
    CUDA_TRY(dev_alloc(&c->d_nl, (size_t)c->maxn * (((size_t)N + 31) / 32 * 32)));
    if (!flags.empty()) {
        CUDA_TRY(dev_alloc(&c->d_flags, N));
        CUDA_TRY(cudaMemcpy(c->d_flags, flags.data(), N, cudaMemcpyHostToDevice));
    }
    if (c->n_coord == 1 && !c->has_mindist && !c->has_q6 && c->prec == 32 && !c->cv[c->coord_dim].use_groups)   // candidates for the tiled path
        CUDA_TRY(dev_alloc(&c->d_cgrad, 4 * (size_t)N));
    if (c->has_q6) {
        CUDA_TRY(cudaMalloc(&c->d_rec, METAD_NREC * tsz * (size_t)N));
        CUDA_TRY(cudaMalloc((void **)&c->d_q6, 2 * tsz * (size_t)N));   // q6 per atom, then f'(q6) per atom, in the pair precision
    }
    // (+ 2 x 4096: per-tile partials of the fp64 tiled build on systems too small for one tile per 128 atoms; partials never
    // outlive the kernel that writes them, so the regions of different kernels may overlap)
    CUDA_TRY(dev_alloc(&c->d_partials, 3 * (size_t)c->nblocks_atoms + max_pair_blocks + 2 * 4096));
    if (c->has_coord && N <= METAD_WARP_PER_ATOM_MAX) CUDA_TRY(dev_alloc(&c->d_partials_warp, (size_t)N / 4 + 2));
    CUDA_TRY(dev_alloc(&c->d_tickets, 16));
    CUDA_TRY(cudaMemset(c->d_tickets, 0, sizeof(unsigned) * 16));
    CUDA_TRY(dev_alloc(&c->d_centers, (size_t)c->D * p->max_hills));
    CUDA_TRY(dev_alloc(&c->d_heights, p->max_hills));
    CUDA_TRY(dev_alloc(&c->d_nhills, 1));
    CUDA_TRY(dev_alloc(&c->d_step, 1));
    CUDA_TRY(dev_alloc(&c->d_sticky, 1));
    CUDA_TRY(cudaMemset(c->d_nhills, 0, sizeof(int)));
    CUDA_TRY(cudaMemset(c->d_step, 0, sizeof(int)));
    CUDA_TRY(cudaMemset(c->d_sticky, 0, sizeof(unsigned)));
    CUDA_TRY(dev_alloc(&c->d_cv, METAD_MAX_CV));
    CUDA_TRY(dev_alloc(&c->d_V, 1));
    CUDA_TRY(dev_alloc(&c->d_dVds, METAD_MAX_CV));
    CUDA_TRY(cudaMemset(c->d_cv, 0, sizeof(double) * METAD_MAX_CV));
    CUDA_TRY(cudaMemset(c->d_V, 0, sizeof(double)));
    CUDA_TRY(cudaMemset(c->d_dVds, 0, sizeof(double) * METAD_MAX_CV));
    CUDA_TRY(dev_alloc(&c->d_bias_partials, 592 * (1 + METAD_MAX_CV)));
    c->grid_on = p->grid_n[0] != 0;
    if (c->grid_on) {
        size_t nn = 4 * (size_t)p->grid_n[0] * p->grid_n[1];
        CUDA_TRY(dev_alloc(&c->d_table, nn));
        CUDA_TRY(cudaMemset(c->d_table, 0, sizeof(double) * nn));
    }
    CUDA_TRY(cudaMalloc(&c->d_pos_stage, 3 * tsz * (size_t)N));
    CUDA_TRY(cudaMalloc(&c->d_F_stage, 3 * tsz * (size_t)N));
    CUDA_TRY(dev_alloc(&c->d_aux, 4));
    int aux0[4] = { 0, -1, 0, 0 };
    CUDA_TRY(cudaMemcpy(c->d_aux, aux0, sizeof(aux0), cudaMemcpyHostToDevice));
    for (int k = 0; k < 3; ++k) CUDA_TRY(cudaEventCreate(&c->ev[k]));
    CUDA_TRY(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    CUDA_TRY(cudaEventCreateWithFlags(&c->ev_copy, cudaEventDisableTiming));
    CUDA_TRY(dev_alloc(&c->d_hill_stage, (size_t)(c->D + 1) * p->max_hills));
    CUDA_TRY(dev_alloc(&c->d_geom, 1));
    CUDA_TRY(dev_alloc(&c->d_tile_cuts, (size_t)c->cell_cap / 4 + 64));
    CUDA_TRY(dev_alloc(&c->d_nbuilds, 1));
    CUDA_TRY(cudaMemset(c->d_nbuilds, 0, sizeof(int)));
    if (!(p->box_slack >= 0.0) || p->box_slack > 1.0) FAIL(METAD_ERR_ARG, "box_slack must be in [0, 1]");
    if (!(p->fill_fraction >= 0.0) || p->fill_fraction > 1.0) FAIL(METAD_ERR_ARG, "fill_fraction must be in [0, 1] (0 = 1)");
    if (!(p->c_window_lo >= 0.0) || !(p->c_window_lo < 1.0)) FAIL(METAD_ERR_ARG, "c_window_lo must be in [0, 1)");
    if (!(p->skin >= 0.0)) FAIL(METAD_ERR_ARG, "skin must be >= 0");
    c->skin_on = p->skin > 0.0 && (c->has_q6 || c->has_coord || c->has_mindist);
    if (c->skin_on) {
        CUDA_TRY(dev_alloc(&c->d_skin_flag, 2));
        const int ones[2] = { 1, 1 };                       // the first step builds
        CUDA_TRY(cudaMemcpy(c->d_skin_flag, ones, sizeof(ones), cudaMemcpyHostToDevice));
        CUDA_TRY(cudaMalloc(&c->d_ref, 4 * tsz * (size_t)N));
    }
    if (p->fill_fraction > 0.0 && p->fill_fraction < 1.0 && c->has_q6 && c->prec == 32 && c->maxn <= 32)
        CUDA_TRY(dev_alloc(&c->d_own_count, N));             // slab-decomposition rank on the tiled Q6 path (domain.cu)
    if (c->skin_on) {
        if (c->has_q6 && c->prec == 32 && c->maxn <= 32) {            // the tiled Q6 path may run: its per-step rc list
            CUDA_TRY(dev_alloc(&c->d_rc_count, N));
            CUDA_TRY(dev_alloc(&c->d_rc_list, (size_t)c->maxn * (((size_t)N + 31) / 32 * 32)));
        }
    }
    CUDA_TRY(cudaDeviceSynchronize());
    return METAD_OK;
}

extern "C" int metad_destroy(metad_ctx *c) {
    if (!c) return METAD_OK;
    if (c->stream) cudaStreamSynchronize(c->stream);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->graph_exec_h) cudaGraphExecDestroy(c->graph_exec_h);
    for (int k = 0; k < 3; ++k) if (c->ev[k]) cudaEventDestroy(c->ev[k]);
    if (c->ev_copy) cudaEventDestroy(c->ev_copy);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    void *ptrs[] = { c->d_cell_count, c->d_cell_start, c->d_block_sums, c->d_cell_of, c->d_slot, c->d_perm, c->d_scell,
                     c->d_spos, c->d_nl_count, c->d_nl, c->d_flags, c->d_rec, c->d_partials, c->d_tickets, c->d_centers,
                     c->d_heights, c->d_nhills, c->d_step, c->d_sticky, c->d_cv, c->d_V, c->d_dVds, c->d_bias_partials,
                     c->d_table, c->d_pos_stage, c->d_F_stage, c->d_aux, c->d_q6, c->d_cgrad, c->d_cvq6, c->d_perm_raw, c->d_tors_grad, c->d_tors_atoms, c->d_partials_warp, c->d_mind, c->d_box_force, c->d_virial, c->d_vir_partials, c->d_traj, c->d_hill_stage, c->d_geom, c->d_skin_flag, c->d_ref, c->d_nbuilds, c->d_rc_count, c->d_rc_list, c->d_tile_cuts, c->d_own_count };
    for (void *q : ptrs) if (q) cudaFree(q);
    for (int d = 0; d < c->D; ++d) {
        CvDev &v = c->cv[d];
        void *q2[] = { v.d_pairs, v.d_pair_r0, v.d_csr_off, v.d_csr_pair, v.d_catoms, v.d_chain, v.d_mass, v.d_unwrapped, v.d_ga, v.d_gb };
        for (void *q : q2) if (q) cudaFree(q);
    }
    if (c->owns_stream && c->stream) cudaStreamDestroy(c->stream);
    (void)cudaGetLastError();
    delete c;
    return METAD_OK;
}

// host-side geometry: box checks (reading O) and the cell grid
static int setup_geometry(metad_ctx *c, const double *box, double rc, double slack = 0.0) {
    if (!box) FAIL(METAD_ERR_ARG, "null box");
    if (box[1] != 0.0 || box[2] != 0.0 || box[5] != 0.0) FAIL(METAD_ERR_BOX, "box must be lower-triangular (rows a,b,c)");
    if (!(box[0] > 0.0) || !(box[4] > 0.0) || !(box[8] > 0.0)) FAIL(METAD_ERR_BOX, "box diagonal must be positive");
    if (!(rc > 0.0)) FAIL(METAD_ERR_ARG, "rc must be positive");
    const double rcl = rc + (c->skin_on ? c->p.skin : 0.0);      // the list (and the cells) reach rc + skin
    const double ax = box[0], bx = box[3], by = box[4], cx = box[6], cy = box[7], cz = box[8];
    const double vol = ax * by * cz;
    // perpendicular widths: V / |b x c|, V / |c x a|, V / |a x b|
    const double bxc[3] = { by * cz, -bx * cz, bx * cy - by * cx };
    const double cxa[3] = { 0.0, cz * ax, -cy * ax };
    double w[3];
    w[0] = vol / sqrt(bxc[0] * bxc[0] + bxc[1] * bxc[1] + bxc[2] * bxc[2]);
    w[1] = vol / sqrt(cxa[1] * cxa[1] + cxa[2] * cxa[2]);
    w[2] = cz;
    for (int d = 0; d < 3; ++d)
        if (!(rcl < 0.5 * w[d])) FAIL(METAD_ERR_BOX, "rc (+ skin) must be smaller than half of every perpendicular box width");
    CellGrid g;
    double shrink = 1.0;
    for (;;) {
        long long tot = 1;
        for (int d = 0; d < 3; ++d) {
            int n = (int)floor(w[d] / (rcl * 1.000001 * (1.0 + slack) * shrink));
            g.nc[d] = n < 1 ? 1 : n;
            tot *= g.nc[d];
        }
        if (tot <= c->cell_cap) { g.ncell = (int)tot; break; }
        shrink *= 1.26;   // cells larger than rc are still valid; keeps ncell within the fixed allocation
    }
    g.inv[0] = 1.0 / ax; g.inv[1] = 1.0 / by; g.inv[2] = 1.0 / cz;
    g.inv[3] = g.inv[4] = g.inv[5] = 0.0;
    g.cx = cx; g.cy = cy; g.bx = bx;
    g.wlo = c->p.c_window_lo; g.wlen = (c->p.fill_fraction > 0.0 && c->p.fill_fraction < 1.0) ? c->p.fill_fraction : 2.0;
    BoxD b = { ax, bx, by, cx, cy, cz, 0.5 * ax, 0.5 * by, 0.5 * cz };
    // a changed cell grid or cutoff invalidates a kept list: the next step rebuilds (set outside any capture: run_impl calls
    // this function before it starts one)
    if (c->skin_on && !c->capturing && (c->rc != rc || c->geom_ncell != g.ncell || memcmp(&c->boxd, &b, sizeof(b)) != 0)) {
        const int ones[2] = { 1, 1 };
        cudaMemcpyAsync(c->d_skin_flag, ones, sizeof(ones), cudaMemcpyHostToDevice, c->stream);
    }
    c->grid = g; c->geom_ncell = g.ncell;
    c->boxd = b;
    c->rc = rc; c->rc2 = rc * rc; c->rcl = rcl; c->rcl2 = rcl * rcl;
    // shared-memory tiled fast path: fp32, neighbour-list CVs = Q6 only or an ungrouped coordination number only,
    // >= 3 cells per direction
    c->tiled = 0; c->tiled64 = 0;
    const bool q6_only = c->has_q6 && !c->has_coord;
    const bool coord_only = c->n_coord == 1 && !c->has_q6 && !c->cv[c->coord_dim].use_groups && !c->skin_on;
    // fp64 pair math: the same tiles for Q6 contexts without a skin (tiled64.cu; 32 bytes per staged atom)
    const bool tile32 = c->prec == 32 && (q6_only || coord_only), tile64 = c->prec == 64 && q6_only && !c->skin_on;
    if ((tile32 || tile64) && !c->has_mindist && c->N < (1 << NL_IDX_BITS) && g.nc[0] >= 3 && g.nc[1] >= 3 && g.nc[2] >= 3 && c->maxn <= 32) {
        // the rc-wide cells are subdivided along x (the direction of the contiguous row runs): an atom then scans
        // 2 xsub + 1 sub-cells per row (2.5 / 2.25 cell widths for xsub = 2 / 4) instead of 3 cells
        int xsub = 2;
        while (xsub > 1 && (long long)g.ncell * xsub > c->cell_cap) --xsub;
        CellGrid gs = g;
        gs.nc[0] *= xsub; gs.ncell *= xsub;
        // atoms per cell where there are atoms (a slab-decomposition rank fills only part of the global box)
        const double rho = (double)c->N / (gs.ncell * (c->p.fill_fraction > 0.0 ? c->p.fill_fraction : 1.0)), margin = 1.3;
        int cap = 1216;
        double best = 1e30; int bt[3] = { 0, 0, 0 };
        // two passes: the smallest halo ratio, then among the shapes within 2 % of it the longest along x (rows are the
        // contiguous runs of the staging copies and of the scan: 11 x 3 x 3 beats 8 x 4 x 3 by 1.8 % at c3)
        for (int pass = 0; pass < 2; ++pass)
        for (int ty = 1; ty <= 4; ++ty) for (int tz = 1; tz <= 4; ++tz) for (int tx = 1; tx <= TILE_TXMAX; ++tx) {
            if (tx > gs.nc[0] - 2 * xsub || ty > gs.nc[1] - 2 || tz > gs.nc[2] - 2) continue;
            double own = rho * tx * ty * tz, halo = rho * (tx + 2 * xsub) * (ty + 2) * (tz + 2);
            if (halo * margin > cap || own > TILE_THREADS) continue;
            long long ntl = (long long)((gs.nc[0] + tx - 1) / tx) * ((gs.nc[1] + ty - 1) / ty) * ((gs.nc[2] + tz - 1) / tz);
            if (ntl > c->nblocks_atoms + (tile64 ? 4096 : 0)) continue;     // per-tile partials live in the per-block scratch
            double score = halo / own + (own < 128 ? 2.0 : 0.0);   // halo ratio; keep the block busy
            if (pass == 0) { if (score < best) best = score; }
            else if (score <= 1.02 * best && tx > bt[0]) { bt[0] = tx; bt[1] = ty; bt[2] = tz; }
        }
        if (bt[0] > 0) {
            c->tiled = tile32; c->tiled64 = tile64; c->tile_T[0] = bt[0]; c->tile_T[1] = bt[1]; c->tile_T[2] = bt[2]; c->tile_cap = cap; c->tile_hx = xsub;
            c->grid = gs;
            // tile boundaries (tile k of a direction covers cells [k nc / nt, (k + 1) nc / nt)): a small device table,
            // uploaded only when the tiling changes (never inside a capture: run_impl derives the geometry before it starts one)
            const int ncs[3] = { gs.nc[0], gs.nc[1], gs.nc[2] };
            int nts[3], key[6];
            for (int d = 0; d < 3; ++d) { nts[d] = (ncs[d] + bt[d] - 1) / bt[d]; key[d] = ncs[d]; key[3 + d] = nts[d]; }
            if (memcmp(key, c->tile_cuts_key, sizeof(key)) != 0) {
                std::vector<int> cuts;
                for (int d = 0; d < 3; ++d)
                    for (int k = 0; k <= nts[d]; ++k) cuts.push_back((int)(((long long)k * ncs[d]) / nts[d]));
                if ((int)cuts.size() > c->cell_cap / 4 + 64) FAIL(METAD_ERR_ARG, "tile table overflow");
                CUDA_TRY(cudaMemcpyAsync(c->d_tile_cuts, cuts.data(), sizeof(int) * cuts.size(), cudaMemcpyHostToDevice, c->stream));
                memcpy(c->tile_cuts_key, key, sizeof(key));
            }
        }
    }
    return METAD_OK;
}

TileGeom tile_geom(const metad_ctx *c) {
    TileGeom t;
    t.Tx = c->tile_T[0]; t.Ty = c->tile_T[1]; t.Tz = c->tile_T[2];
    t.nc0 = c->grid.nc[0]; t.nc1 = c->grid.nc[1]; t.nc2 = c->grid.nc[2];
    t.ntx = (t.nc0 + t.Tx - 1) / t.Tx; t.nty = (t.nc1 + t.Ty - 1) / t.Ty; t.ntz = (t.nc2 + t.Tz - 1) / t.Tz;
    t.cap = c->tile_cap; t.hx = c->tile_hx; t.natoms = c->N;
    t.sparse = (c->p.fill_fraction > 0.0 && c->p.fill_fraction < 1.0) ? 1 : 0;
    t.tz0 = 0; t.ntz_launch = t.ntz;
    if (t.sparse) {
        // the z-tiles that overlap the window of occupied cells [c0, c1] along c (periodic); tile k covers cells
        // [k nc / nt, (k + 1) nc / nt), so the tile of cell j is the largest k with k nc / nt <= j
        const int c0 = std::min((int)floor(c->p.c_window_lo * t.nc2), t.nc2 - 1);
        const int ncw = std::min((int)ceil((c->p.c_window_lo + c->p.fill_fraction) * t.nc2) - c0, t.nc2);   // cells in the window
        auto tile_of = [&](int j) { int k = (int)(((long long)(j + 1) * t.ntz - 1) / t.nc2); while ((long long)k * t.nc2 / t.ntz > j) --k;
                                    while ((long long)(k + 1) * t.nc2 / t.ntz <= j) ++k; return k; };
        if (ncw < t.nc2) {
            const int k0 = tile_of(c0), k1 = tile_of((c0 + ncw - 1) % t.nc2);
            const int n = ((k1 - k0) % t.ntz + t.ntz) % t.ntz + 1;
            // a window that wraps onto its own first tile would launch that tile twice: then launch everything
            if (!(c0 + ncw - 1 >= t.nc2 && k1 == k0)) { t.tz0 = k0; t.ntz_launch = n; }
        }
    }
    t.cshift = 0;
    while ((1 << t.cshift) < t.Tx + 2 * t.hx + 2) ++t.cshift;      // Txe <= Tx + 1 columns + the end-of-row entry
    t.cuts = c->d_tile_cuts;
    t.ax = c->boxd.ax; t.bx = c->boxd.bx; t.by = c->boxd.by; t.cx = c->boxd.cx; t.cy = c->boxd.cy; t.cz = c->boxd.cz;
    t.wa = t.wb = t.wc = 0.0;
    return t;
}

static int build_neighbors_impl(metad_ctx *c, const void *d_pos, const double *h_box, double rc);

extern "C" int metad_build_neighbors(metad_ctx *c, const void *d_pos, const double *h_box, double rc) {
    if (!c || !d_pos) FAIL(METAD_ERR_ARG, "null argument");
    c->dg = nullptr;                               // host box: geometry travels in the kernel arguments
    return build_neighbors_impl(c, d_pos, h_box, rc);
}

// device box: derive the cell grid once from the box as it is now (the only host read), then freeze it
static int dev_geometry(metad_ctx *c, const double *d_box, double rc) {
    if (!c->dev_geom_ready || c->rc != rc) {
        double hb[9];
        CUDA_TRY(cudaMemcpyAsync(hb, d_box, sizeof(hb), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        int r = setup_geometry(c, hb, rc, c->p.box_slack);
        if (r) return r;
        c->dev_geom_ready = 1;
    }
    return METAD_OK;
}

extern "C" int metad_build_neighbors_dev(metad_ctx *c, const void *d_pos, const double *d_box, double rc) {
    if (!c || !d_pos || !d_box) FAIL(METAD_ERR_ARG, "null argument");
    int r = dev_geometry(c, d_box, rc);
    if (r) return r;
    c->dg = c->d_geom; c->d_box_last = d_box;
    if ((r = geom_update(c, d_box))) return r;
    return build_neighbors_impl(c, d_pos, nullptr, rc);
}

extern "C" int metad_reset_box(metad_ctx *c) {
    if (!c) FAIL(METAD_ERR_ARG, "null argument");
    c->dev_geom_ready = 0;
    if (c->graph_exec && c->graph_devbox) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    return METAD_OK;
}

static int build_neighbors_impl(metad_ctx *c, const void *d_pos, const double *h_box, double rc) {
    int r = c->dg ? METAD_OK : setup_geometry(c, h_box, rc);     // device box: geometry frozen by metad_build_neighbors_dev
    if (r) return r;
    c->d_pos_last = d_pos;
    c->own_count_valid = 0;                         // masked counts of the last step (metad_cv_owned_sum) are stale now
    // no CV reads the list; a nearest-distance CV with a few explicit centres is scanned without one (k_mindist_brute)
    bool mind_brute = c->has_mindist;
    for (int d = 0; d < c->D; ++d)
        if (c->cv[d].kind == METAD_CV_MINDIST)
            mind_brute = mind_brute && c->cv[d].d_ga && c->cv[d].n_ga <= 64 && div_up(c->cv[d].n_gb, 128) <= c->nblocks_atoms;
    if (c->p.lazy_neighbors && !c->has_q6 && !c->has_coord && (!c->has_mindist || mind_brute)) {
        c->have_neighbors = true; c->list_built = false;
        return METAD_OK;
    }
    c->list_skipped = 0;
    r = nb_build(c, d_pos);
    if (r == METAD_OK) { c->have_neighbors = true; c->list_built = !c->list_skipped; }
    return r;
}

extern "C" int metad_eval_cv(metad_ctx *c, double *d_cv) {
    if (!c || !d_cv) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->have_neighbors) FAIL(METAD_ERR_STATE, "metad_build_neighbors has not been called");
    return cv_eval_all(c, d_cv);
}

extern "C" int metad_bias(metad_ctx *c, const double *d_cv, double *d_V, double *d_dVds) {
    if (!c || !d_cv || !d_V || !d_dVds) FAIL(METAD_ERR_ARG, "null argument");
    return bias_eval(c, d_cv, d_V, d_dVds);
}

extern "C" int metad_apply_forces(metad_ctx *c, const double *d_dVds, void *d_F) {
    if (!c || !d_dVds || !d_F) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->have_neighbors) FAIL(METAD_ERR_STATE, "metad_build_neighbors has not been called");
    return cv_forces_all(c, d_dVds, d_F);
}

extern "C" int metad_host_alloc(void **ptr, size_t bytes) {
    if (!ptr || bytes == 0) FAIL(METAD_ERR_ARG, "null pointer or zero size");
    *ptr = nullptr;
    CUDA_TRY(cudaHostAlloc(ptr, bytes, cudaHostAllocDefault));
    return METAD_OK;
}

extern "C" int metad_host_free(void *ptr) {
    if (!ptr) return METAD_OK;
    CUDA_TRY(cudaFreeHost(ptr));
    return METAD_OK;
}

extern "C" int metad_deposit(metad_ctx *c, const double *d_cv, const double *d_V) {
    if (!c || !d_cv || !d_V) FAIL(METAD_ERR_ARG, "null argument");
    return bias_deposit(c, d_cv, d_V);
}

static bool fused_torsion_ok(const metad_ctx *c) {
    if (!c->p.lazy_neighbors || c->p.want_virial || c->ntors_atoms > 256) return false;
    for (int d = 0; d < c->D; ++d) if (c->cv[d].kind != METAD_CV_TORSION) return false;
    return c->D <= 2 || !c->grid_on;
}

// d_box != NULL: the step reads its box from device memory (geometry frozen by dev_geometry before the capture)
static int enqueue_step(metad_ctx *c, const void *d_pos, const double *box, double rc, void *d_F, const double *d_box = nullptr) {
    int r;
    if (fused_torsion_ok(c)) {                    // torsion-only context: the whole step is one kernel (bias.cu)
        if (d_box) { c->dg = c->d_geom; c->d_box_last = d_box; if ((r = geom_update(c, d_box))) return r; }
        else { c->dg = nullptr; if ((r = setup_geometry(c, box, rc))) return r; }
        c->d_pos_last = d_pos; c->have_neighbors = true; c->list_built = false;
        if (c->wait_copy) CUDA_TRY(cudaStreamWaitEvent(c->stream, c->ev_copy, cudaEventWaitExternal));
        return bias_fused_torsion_step(c, d_pos, d_F);
    }
    // without a grid the deposition rides on the hill sum (one launch less; same V, same order of effects: the forces of
    // this step use the dV/ds of the hills deposited before it, reading U)
    const bool fuse = !c->grid_on;
    c->cv_direct = c->d_cv;
    if (d_box) {
        c->dg = c->d_geom; c->d_box_last = d_box;
        r = geom_update(c, d_box);
        if (!r) r = build_neighbors_impl(c, d_pos, nullptr, rc);
    } else {
        r = metad_build_neighbors(c, d_pos, box, rc);
    }
    if (!r) r = metad_eval_cv(c, c->d_cv);
    c->cv_direct = nullptr;
    if (r) return r;
    if ((r = bias_eval(c, c->d_cv, c->d_V, c->d_dVds, fuse))) return r;
    // metad_step_host: the caller's forces travel on the copy stream while the build, the CVs and the bias run; the force
    // kernel waits for them (an external event-wait node of the captured step)
    if (c->wait_copy) CUDA_TRY(cudaStreamWaitEvent(c->stream, c->ev_copy, cudaEventWaitExternal));
    if ((r = metad_apply_forces(c, c->d_dVds, d_F))) return r;
    return fuse ? METAD_OK : metad_deposit(c, c->d_cv, c->d_V);
}

// One step captured into a graph (the caller instantiates it or updates its instantiated graph).  Argument errors must have
// surfaced before: the geometry is derived outside the capture.
static int capture_step(metad_ctx *c, const void *d_pos, const double *h_box, const double *d_box, double rc, void *d_F,
                        bool wait_copy, cudaGraph_t *graph, int *launches_per_step) {
    const long long before = c->launches;
    CUDA_TRY(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    c->capturing = 1; c->wait_copy = wait_copy ? 1 : 0;
    int r = enqueue_step(c, d_pos, h_box, rc, d_F, d_box);
    c->capturing = 0; c->wait_copy = 0;
    cudaError_t e = cudaStreamEndCapture(c->stream, graph);
    *launches_per_step = (int)(c->launches - before);
    c->launches = before;                          // capture enqueued nothing
    if (r) { if (e == cudaSuccess) cudaGraphDestroy(*graph); return r; }
    CUDA_TRY(e);
    return METAD_OK;
}

// a changed box (NPT) or pointer changes kernel arguments and grid sizes, not the topology: update the
// instantiated graph in place when the driver allows it, re-instantiate otherwise
static int instantiate_or_update(cudaGraphExec_t *exec, cudaGraph_t graph, bool *updated) {
    *updated = false;
    if (*exec) {
        cudaGraphExecUpdateResultInfo info;
        if (cudaGraphExecUpdate(*exec, graph, &info) == cudaSuccess) *updated = true;
        else { cudaGetLastError(); cudaGraphExecDestroy(*exec); *exec = nullptr; }
    }
    if (!*updated) CUDA_TRY(cudaGraphInstantiate(exec, graph, 0));
    return METAD_OK;
}

static int run_impl(metad_ctx *c, const void *d_pos, const double *h_box, const double *d_box, double rc, void *d_F, int nsteps);
static int count_graph_nodes(cudaGraph_t graph, int *k);

extern "C" int metad_run(metad_ctx *c, const void *d_pos, const double *h_box, double rc, void *d_F, int nsteps) {
    if (!c || !d_pos || !d_F || !h_box || nsteps < 0) FAIL(METAD_ERR_ARG, "bad argument");
    return run_impl(c, d_pos, h_box, nullptr, rc, d_F, nsteps);
}

extern "C" int metad_run_dev(metad_ctx *c, const void *d_pos, const double *d_box, double rc, void *d_F, int nsteps) {
    if (!c || !d_pos || !d_F || !d_box || nsteps < 0) FAIL(METAD_ERR_ARG, "bad argument");
    return run_impl(c, d_pos, nullptr, d_box, rc, d_F, nsteps);
}

static int run_impl(metad_ctx *c, const void *d_pos, const double *h_box, const double *d_box, double rc, void *d_F, int nsteps) {
    bool same = c->graph_exec && c->graph_pos == d_pos && c->graph_F == d_F && c->graph_rc == rc &&
                (d_box ? (c->graph_devbox && c->graph_dbox == d_box && c->dev_geom_ready)
                       : (!c->graph_devbox && h_box && memcmp(c->graph_box, h_box, sizeof(double) * 9) == 0));
    if (!same) {
        // argument errors surface before the capture starts; a device box is read ONCE here to derive the frozen cell grid
        int r = d_box ? dev_geometry(c, d_box, rc) : setup_geometry(c, h_box, rc);
        if (r) return r;
        cudaGraph_t graph;
        int lps = 0;
        if ((r = capture_step(c, d_pos, h_box, d_box, rc, d_F, false, &graph, &lps))) return r;
        int cr = count_graph_nodes(graph, c->graph_counts);      // for metad_graph_info (the zero-host-copy proof)
        bool updated = false;
        r = instantiate_or_update(&c->graph_exec, graph, &updated);
        cudaGraphDestroy(graph);
        if (r) return r;
        if (cr) return cr;
        c->graph_captures++;
        c->graph_updates += updated ? 1 : 0;
        c->launches_per_step = lps;
        c->graph_pos = d_pos; c->graph_F = d_F; c->graph_rc = rc;
        c->graph_devbox = d_box != nullptr; c->graph_dbox = d_box;
        if (h_box) memcpy(c->graph_box, h_box, sizeof(double) * 9);
    }
    for (int s = 0; s < nsteps; ++s) CUDA_TRY(cudaGraphLaunch(c->graph_exec, c->stream));
    c->launches += (long long)c->launches_per_step * nsteps;
    return METAD_OK;
}

extern "C" int metad_step_host(metad_ctx *c, const void *h_pos, const double *h_box, double rc, void *h_F,
                               double *h_cv, double *h_V) {
    if (!c || !h_pos || !h_F || !h_box) FAIL(METAD_ERR_ARG, "null argument");
    const size_t bytes = 3 * (size_t)c->N * (c->prec == 32 ? sizeof(float) : sizeof(double));
    // the kernels of the step are a captured graph on the staging buffers (lower node-to-node latency than eight stream
    // launches), re-captured only when the box or the cutoff changes
    int r;
    const bool same = c->graph_exec_h && c->graph_h_rc == rc && memcmp(c->graph_h_box, h_box, sizeof(double) * 9) == 0;
    if (!same) {
        if ((r = setup_geometry(c, h_box, rc))) return r;
        cudaGraph_t graph;
        int lps = 0;
        if ((r = capture_step(c, c->d_pos_stage, h_box, nullptr, rc, c->d_F_stage, true, &graph, &lps))) return r;
        bool updated = false;
        r = instantiate_or_update(&c->graph_exec_h, graph, &updated);
        cudaGraphDestroy(graph);
        if (r) return r;
        c->launches_per_step_h = lps;
        c->graph_h_rc = rc; memcpy(c->graph_h_box, h_box, sizeof(double) * 9);
    }
    // positions first; the caller's forces travel on a second stream while the neighbour build, the CVs and the bias
    // run (they are not needed before apply_forces)
    CUDA_TRY(cudaMemcpyAsync(c->d_pos_stage, h_pos, bytes, cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(c->d_F_stage, h_F, bytes, cudaMemcpyHostToDevice, c->copy_stream));
    CUDA_TRY(cudaEventRecord(c->ev_copy, c->copy_stream));
    CUDA_TRY(cudaGraphLaunch(c->graph_exec_h, c->stream));
    c->launches += c->launches_per_step_h;
    CUDA_TRY(cudaMemcpyAsync(h_F, c->d_F_stage, bytes, cudaMemcpyDeviceToHost, c->stream));
    if (h_cv) CUDA_TRY(cudaMemcpyAsync(h_cv, c->d_cv, sizeof(double) * c->D, cudaMemcpyDeviceToHost, c->stream));
    if (h_V) CUDA_TRY(cudaMemcpyAsync(h_V, c->d_V, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return METAD_OK;
}

extern "C" int metad_status(metad_ctx *c, unsigned *bits) {
    if (!c || !bits) FAIL(METAD_ERR_ARG, "null argument");
    unsigned b = 0;
    CUDA_TRY(cudaMemcpyAsync(&b, c->d_sticky, sizeof(unsigned), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    *bits |= b;
    return METAD_OK;
}

extern "C" int metad_get_state(metad_ctx *c, double *h_cv, double *h_V, double *h_dVds, int *h_step, int *h_nhills) {
    if (!c) FAIL(METAD_ERR_ARG, "null argument");
    if (h_cv) CUDA_TRY(cudaMemcpyAsync(h_cv, c->d_cv, sizeof(double) * c->D, cudaMemcpyDeviceToHost, c->stream));
    if (h_V) CUDA_TRY(cudaMemcpyAsync(h_V, c->d_V, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    if (h_dVds) CUDA_TRY(cudaMemcpyAsync(h_dVds, c->d_dVds, sizeof(double) * c->D, cudaMemcpyDeviceToHost, c->stream));
    if (h_step) CUDA_TRY(cudaMemcpyAsync(h_step, c->d_step, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    if (h_nhills) CUDA_TRY(cudaMemcpyAsync(h_nhills, c->d_nhills, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return METAD_OK;
}

extern "C" int metad_get_neighbors(metad_ctx *c, int *d_count, int *d_list) {
    if (!c || !d_count || !d_list) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->have_neighbors) FAIL(METAD_ERR_STATE, "metad_build_neighbors has not been called");
    if (!c->list_built) FAIL(METAD_ERR_STATE, "lazy_neighbors: nothing in this context reads the list, it was not built");
    return nb_export(c, d_count, d_list);
}

extern "C" int metad_get_q6(metad_ctx *c, void *d_q6) {
    if (!c || !d_q6) FAIL(METAD_ERR_ARG, "null argument");
    return q6_export(c, d_q6);
}

extern "C" int metad_set_hills(metad_ctx *c, const double *centers, const double *heights, int count, int on_device) {
    if (!c || count < 0 || (count > 0 && (!centers || !heights))) FAIL(METAD_ERR_ARG, "bad argument");
    if (count > c->p.max_hills) FAIL(METAD_ERR_ARG, "count exceeds max_hills");
    int r;
    if (on_device || count == 0) {
        r = bias_set_hills_dev(c, centers, heights, count);
    } else {
        double *dc = c->d_hill_stage, *dh = c->d_hill_stage + (size_t)c->D * c->p.max_hills;   // staging from metad_create
        CUDA_TRY(cudaMemcpyAsync(dc, centers, sizeof(double) * (size_t)count * c->D, cudaMemcpyHostToDevice, c->stream));
        CUDA_TRY(cudaMemcpyAsync(dh, heights, sizeof(double) * count, cudaMemcpyHostToDevice, c->stream));
        r = bias_set_hills_dev(c, dc, dh, count);
    }
    if (r) return r;
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return METAD_OK;
}

extern "C" int metad_get_hills(metad_ctx *c, double *centers, double *heights, int capacity, int *count, int on_device) {
    if (!c) FAIL(METAD_ERR_ARG, "null argument");
    int H = 0;
    CUDA_TRY(cudaMemcpyAsync(&H, c->d_nhills, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    if (count) *count = H;
    if (!centers || !heights || capacity <= 0) return METAD_OK;
    int n = H < capacity ? H : capacity;
    if (on_device) {
        int r = bias_get_hills_dev(c, centers, heights, capacity);
        if (r) return r;
    } else {
        double *dc = c->d_hill_stage, *dh = c->d_hill_stage + (size_t)c->D * c->p.max_hills;
        int r = bias_get_hills_dev(c, dc, dh, std::min(capacity, c->p.max_hills));
        if (r) return r;
        CUDA_TRY(cudaMemcpyAsync(centers, dc, sizeof(double) * (size_t)n * c->D, cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaMemcpyAsync(heights, dh, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    }
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return METAD_OK;
}

extern "C" int metad_get_grid(metad_ctx *c, double *d_table) {
    if (!c || !d_table) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->grid_on) FAIL(METAD_ERR_STATE, "grid not enabled");
    size_t nn = 4 * (size_t)c->p.grid_n[0] * c->p.grid_n[1];
    CUDA_TRY(cudaMemcpyAsync(d_table, c->d_table, sizeof(double) * nn, cudaMemcpyDeviceToDevice, c->stream));
    return METAD_OK;
}

extern "C" int metad_bias_batch(metad_ctx *c, const double *d_points, int npoints, double *d_V) {
    if (!c || npoints < 0 || (npoints > 0 && (!d_points || !d_V))) FAIL(METAD_ERR_ARG, "bad argument");
    return bias_batch(c, d_points, npoints, d_V);
}

extern "C" int metad_reweight(metad_ctx *c, const double *d_traj, int nframes, const int *h_nbins, const double *h_lo,
                              const double *h_hi, double *d_P, double *d_F) {
    if (!c || nframes < 0 || (nframes > 0 && !d_traj) || !h_nbins || !h_lo || !h_hi || !d_P || !d_F)
        FAIL(METAD_ERR_ARG, "bad argument");
    if (c->D > 2) FAIL(METAD_ERR_ARG, "reweighting histograms 1 or 2 CV dimensions");
    if (!(c->p.kT > 0.0)) FAIL(METAD_ERR_ARG, "kT must be positive");
    for (int d = 0; d < c->D; ++d) {
        if (h_nbins[d] < 1 || !(h_hi[d] > h_lo[d])) FAIL(METAD_ERR_ARG, "bins need n >= 1 and hi > lo");
        if (c->p.period[d] > 0.0 && fabs((h_hi[d] - h_lo[d]) - c->p.period[d]) > 1e-12 * c->p.period[d])
            FAIL(METAD_ERR_ARG, "a periodic dimension needs hi - lo == period");
    }
    if ((long long)h_nbins[0] * (c->D > 1 ? h_nbins[1] : 1) > (1ll << 26)) FAIL(METAD_ERR_ARG, "too many bins");
    return reweight_run(c, d_traj, nframes, h_nbins, h_lo, h_hi, d_P, d_F);
}

extern "C" int metad_get_box_force(metad_ctx *c, double *d_out9) {
    if (!c || !d_out9) FAIL(METAD_ERR_ARG, "null argument");
    CUDA_TRY(cudaMemcpyAsync(d_out9, c->d_box_force, sizeof(double) * 9, cudaMemcpyDeviceToDevice, c->stream));
    return METAD_OK;
}

extern "C" int metad_get_virial(metad_ctx *c, double *d_out9) {
    if (!c || !d_out9) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->p.want_virial) FAIL(METAD_ERR_STATE, "params.want_virial was not set");
    CUDA_TRY(cudaMemcpyAsync(d_out9, c->d_virial, sizeof(double) * 9, cudaMemcpyDeviceToDevice, c->stream));
    return METAD_OK;
}

extern "C" int metad_reweight_recorded(metad_ctx *c, const int *h_nbins, const double *h_lo, const double *h_hi, double *d_P,
                                       double *d_F, int *h_nframes) {
    if (!c) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->d_traj) FAIL(METAD_ERR_STATE, "params.traj_capacity was 0: no trajectory is recorded");
    int steps = 0;
    CUDA_TRY(cudaMemcpyAsync(&steps, c->d_step, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    const int n = steps < c->p.traj_capacity ? steps : c->p.traj_capacity;
    if (h_nframes) *h_nframes = n;
    return metad_reweight(c, c->d_traj, n, h_nbins, h_lo, h_hi, d_P, d_F);
}

extern "C" int metad_reset_steps(metad_ctx *c) {
    if (!c) FAIL(METAD_ERR_ARG, "null argument");
    CUDA_TRY(cudaMemsetAsync(c->d_step, 0, sizeof(int), c->stream));
    return METAD_OK;
}

extern "C" int metad_set_timing(metad_ctx *c, int enabled) {
    if (!c) FAIL(METAD_ERR_ARG, "null argument");
    c->timing = enabled != 0;
    c->timing_recorded = 0;
    return METAD_OK;
}

extern "C" int metad_get_timing(metad_ctx *c, float *ms_sort, float *ms_list) {
    if (!c || !ms_sort || !ms_list) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->timing) FAIL(METAD_ERR_STATE, "timing is not enabled");
    if (!c->timing_recorded) FAIL(METAD_ERR_STATE, "no neighbour build has been timed yet");
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    CUDA_TRY(cudaEventElapsedTime(ms_sort, c->ev[0], c->ev[1]));
    CUDA_TRY(cudaEventElapsedTime(ms_list, c->ev[1], c->ev[2]));
    return METAD_OK;
}

extern "C" long long metad_launch_count(metad_ctx *c) { return c ? c->launches : 0; }

extern "C" int metad_get_rebuilds(metad_ctx *c, int *h_count) {
    if (!c || !h_count) FAIL(METAD_ERR_ARG, "null argument");
    CUDA_TRY(cudaMemcpyAsync(h_count, c->d_nbuilds, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return METAD_OK;
}

extern "C" int metad_synchronize(metad_ctx *c) {
    if (!c) FAIL(METAD_ERR_ARG, "null argument");
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return METAD_OK;
}

// node counts of a freshly captured step graph (taken before instantiation and cached in the context)
static int count_graph_nodes(cudaGraph_t graph, int *k /* [9] */) {
    size_t n = 0;
    CUDA_TRY(cudaGraphGetNodes(graph, nullptr, &n));
    std::vector<cudaGraphNode_t> nodes(n);
    if (n) CUDA_TRY(cudaGraphGetNodes(graph, nodes.data(), &n));
    for (int q = 0; q < 9; ++q) k[q] = 0;
    k[0] = (int)n;
    for (size_t i = 0; i < n; ++i) {
        cudaGraphNodeType t;
        if (cudaGraphNodeGetType(nodes[i], &t) != cudaSuccess) {
            // CUDA 12.9 / driver 580 answers cudaErrorUnknown for a conditional node (the only node kind this library adds by
            // hand: the skin's IF node); every node a stream capture records has a type the call knows
            (void)cudaGetLastError();
            k[8]++;
            continue;
        }
        if (t == cudaGraphNodeTypeKernel) k[1]++;
        else if (t == cudaGraphNodeTypeMemcpy) k[2]++;
        else if (t == cudaGraphNodeTypeMemset) k[3]++;
        else if (t == cudaGraphNodeTypeHost) k[4]++;
        else if (t == cudaGraphNodeTypeConditional) k[8]++;
        else k[5]++;
    }
    return METAD_OK;
}

extern "C" int metad_graph_info(metad_ctx *c, int *h_counts) {
    if (!c || !h_counts) FAIL(METAD_ERR_ARG, "null argument");
    if (!c->graph_exec) FAIL(METAD_ERR_STATE, "metad_run has not captured a step yet");
    memcpy(h_counts, c->graph_counts, sizeof(int) * 9);
    h_counts[6] = c->graph_captures;
    h_counts[7] = c->graph_updates;
    return METAD_OK;
}
