// domain.cu — the one device piece of the slab decomposition over several GPUs (DESIGN.md
// section 8): the Q6 CVs summed over the atoms a rank OWNS.
//
// A rank holds its slab of the box plus a halo of 2 (rc + skin) on either side, at the atoms' GLOBAL coordinates in the
// GLOBAL box (paper_2510_06873_b200/domain.py), so every pair it sees is computed exactly as in the whole system.  After
// metad_build_neighbors + metad_eval_cv the per-atom q6 of the owned atoms and of the halo atoms within rc + skin of the slab
// are those of the whole system; metad_cv_owned_sum replaces the context-wide sums in d_cv by the sums over the owned atoms,
// the ranks add these partial sums (ONE all-reduce of ncv doubles per step, NCCL), and every rank goes on with the same
// s: metad_bias, metad_apply_forces (the forces of the owned atoms are complete: they need the records of their neighbours,
// which need THEIR neighbours — hence the 2 (rc + skin) halo), metad_deposit (identical hills on every rank).
#include <algorithm>
#include "common.cuh"

#define OWN_THREADS 256
#define OWN_MAX_BLOCKS 592                                  // 4 x 148 SMs: a few atoms per thread, ONE block reduction per block

// q6 of sorted atom s: the dense per-atom array d_q6 of every Q6 path (q6_stride = 1).
// Fixed assignment of atoms to threads and blocks, fixed-order reductions: run-to-run identical.
template <typename T>
__global__ void __launch_bounds__(OWN_THREADS)
k_cv_owned_sum(int N, const int *__restrict__ perm, const unsigned char *__restrict__ owned, const T *__restrict__ q6,
               int q6_stride, T q_thresh, T inv_width, double scale_mean, double scale_solid, int dim_mean, int dim_solid,
               double *__restrict__ partials, unsigned int *__restrict__ ticket, double *__restrict__ cv_out,
               const int *__restrict__ count_in, int *__restrict__ count_out /* tiled path: neighbour counts, 0 for atoms not owned */) {
    __shared__ double red[64];
    double v[2] = { 0.0, 0.0 };
    for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < N; s += gridDim.x * blockDim.x) {
        const bool mine = owned[perm[s]] != 0;
        if (count_out) count_out[s] = mine ? count_in[s] : 0;
        if (!mine) continue;
        const T q = q6[(size_t)s * q6_stride];
        v[0] += (double)q;
        if (dim_solid >= 0) v[1] += (double)(T(1) / (T(1) + exp(-(q - q_thresh) * inv_width)));     // the expression of the pass-1 kernels
    }
    block_reduce<2>(v, red);
    if (threadIdx.x == 0) { partials[2 * blockIdx.x] = v[0]; partials[2 * blockIdx.x + 1] = v[1]; }
    if (last_block_ticket(ticket)) {                      // fixed-order sum of the per-block partials
        double u[2] = { 0.0, 0.0 };
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) { u[0] += partials[2 * b]; u[1] += partials[2 * b + 1]; }
        block_reduce<2>(u, red);
        if (threadIdx.x == 0) {
            if (dim_mean >= 0) cv_out[dim_mean] = scale_mean * u[0];
            if (dim_solid >= 0) cv_out[dim_solid] = scale_solid * u[1];
        }
    }
}

extern "C" int metad_cv_owned_sum(metad_ctx *c, const unsigned char *d_owned, double *d_cv) {
    if (!c || !d_owned || !d_cv) { metad_set_error("null argument"); return METAD_ERR_ARG; }
    if (!c->has_q6) { metad_set_error("metad_cv_owned_sum: only the Q6 CVs have per-atom values to sum (DESIGN.md section 8)"); return METAD_ERR_STATE; }
    if (!c->have_neighbors) { metad_set_error("metad_build_neighbors / metad_eval_cv have not been called"); return METAD_ERR_STATE; }
    for (int d = 0; d < c->D; ++d)
        if (d != c->q6_mean_dim && d != c->q6_solid_dim) {
            metad_set_error("metad_cv_owned_sum: every CV dimension of the context must be a Q6 CV"); return METAD_ERR_STATE;
        }
    const int N = c->N, nb = std::min(std::min(div_up(N, OWN_THREADS), OWN_MAX_BLOCKS), c->nblocks_atoms);   // the Q6 region of the per-block scratch
    const double qt = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_thresh : 0.0;
    const double qw = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_width : 1.0;
    const double sm = c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0;
    const double ss = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0;
    double *partials = c->d_partials + c->nblocks_atoms;       // free again once eval_cv's kernel has finished (stream order)
    unsigned int *ticket = c->d_tickets + 14;
    if (c->tiled) {
        // the force pass of this step skips the atoms the rank does not own (their rows of F belong to other ranks): it walks
        // the neighbour counts written here, which are 0 for them
        const int *cin = c->skin_on ? c->d_rc_count : c->d_nl_count;
        k_cv_owned_sum<float><<<nb, OWN_THREADS, 0, c->stream>>>(N, c->d_perm, d_owned, c->d_q6, 1, (float)qt, (float)(1.0 / qw), sm, ss,
                                                                 c->q6_mean_dim, c->q6_solid_dim, partials, ticket, d_cv, cin, c->d_own_count);
        c->own_count_valid = c->d_own_count != nullptr;
    }
    else if (c->prec == 32)
        k_cv_owned_sum<float><<<nb, OWN_THREADS, 0, c->stream>>>(N, c->d_perm, d_owned, (const float *)c->d_q6, 1, (float)qt,
                                                                 (float)(1.0 / qw), sm, ss, c->q6_mean_dim, c->q6_solid_dim, partials, ticket, d_cv, nullptr, nullptr);
    else
        k_cv_owned_sum<double><<<nb, OWN_THREADS, 0, c->stream>>>(N, c->d_perm, d_owned, (const double *)c->d_q6, 1, qt, 1.0 / qw,
                                                                  sm, ss, c->q6_mean_dim, c->q6_solid_dim, partials, ticket, d_cv, nullptr, nullptr);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
