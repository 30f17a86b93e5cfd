// cv.cu — a2/a3 CV evaluation and a6 gather-form forces for the neighbour-list CVs
// (coordination number, Steinhardt Q6 mean, solid-like count).  Thread per (cell-sorted) atom;
// pair arithmetic in T, every reduction in fp64 with a fixed order (deterministic).
#include "common.cuh"
#include "cv_q6.cuh"
#include "cv_switch.cuh"

template <typename T> PBox<T> ctx_pbox(const metad_ctx *c);

#define CV_THREADS 128

// ------------------------------------------------------------------------------------------------
// coordination number
template <typename T>
__global__ void __launch_bounds__(CV_THREADS)
k_coord_cv(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ nl_count,
           const int *__restrict__ nl, PBox<T> pb, BoxD bdk, T rc2T, double rc2k /* Verlet skin: keep pairs with r < rc only; 0 = the list is exact */, int fshift /* this CV's bits of the group flags */, T inv_r0, int n, int m, double scale,
           double *__restrict__ partials, unsigned int *__restrict__ ticket, double *__restrict__ cv_out,
           unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg) {
    __shared__ double red[32];
    if (dg) { pb = dg_pb<T>(dg); bdk = dg->bd; }
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    T acc = T(0);
    if (s < N) {
        typename Vec4<T>::type pi = spos[s];
        if ((((int)pi.w) >> fshift) & 1) {
            int cnt = nl_count[s];
            for (int k = 0; k < cnt; ++k) {
                int j = nl[(size_t)k * N + s];
                typename Vec4<T>::type pj = ldg4<T>(spos + j);
                if (!((((int)pj.w) >> fshift) & 2)) continue;
                if (rc2k > 0.0 && !pair_in_range<T>(pb, bdk, rc2T, rc2k, pi, pj)) continue;
                T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                min_image(pb, dx, dy, dz);
                T r = sqrt(dx * dx + dy * dy + dz * dz), dsw;
                acc += switch_fn<T>(r * inv_r0, n, m, dsw);
            }
        }
    }
    double v[1] = { (double)acc };
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

// VIRIAL: the same pass also sums g d_a d_b over the visited pairs (every unordered pair is visited from both ends, hence
// the factor 1/2): W = -1/2 force_scale scale dV/ds sum_k sum_j g d d^T (reading AD).
template <typename T, bool VIRIAL>
__global__ void __launch_bounds__(CV_THREADS)
k_coord_force(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ nl_count,
              const int *__restrict__ nl, const int *__restrict__ perm, PBox<T> pb, BoxD bdk, T rc2T, double rc2k /* Verlet skin: keep pairs with r < rc only; 0 = the list is exact */, int fshift /* this CV's bits of the group flags */, T inv_r0, int n, int m,
              double coef /* force_scale*scale */, const double *__restrict__ dVds, T *__restrict__ F, VirArgs va,
              const DevGeom *__restrict__ dg) {
    __shared__ double vsm[VIRIAL ? 9 * 32 : 1];
    if (dg) { pb = dg_pb<T>(dg); bdk = dg->bd; }
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (!VIRIAL && s >= N) return;
    const bool act = s < N;
    if (!act) s = N - 1;                       // idle thread of the virial instance: valid addresses, zero trip count
    T wv[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) wv[q] = T(0);
    typename Vec4<T>::type pi = spos[s];
    const int fi = ((int)pi.w) >> fshift;
    T ax = T(0), ay = T(0), az = T(0);
    int cnt = act ? nl_count[s] : 0;
    for (int k = 0; k < cnt; ++k) {
        int j = nl[(size_t)k * N + s];
        typename Vec4<T>::type pj = ldg4<T>(spos + j);
        const int fj = ((int)pj.w) >> fshift;
        int mult = ((fi & 1) && (fj & 2)) + ((fi & 2) && (fj & 1));
        if (!mult) continue;
        if (rc2k > 0.0 && !pair_in_range<T>(pb, bdk, rc2T, rc2k, pi, pj)) continue;
        T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        min_image(pb, dx, dy, dz);
        T r = sqrt(dx * dx + dy * dy + dz * dz), dsw;
        switch_fn<T>(r * inv_r0, n, m, dsw);
        T g = T(mult) * dsw * inv_r0 / r;
        ax += g * dx; ay += g * dy; az += g * dz;
        if (VIRIAL) {
            const T gx = g * dx, gy = g * dy, gz = g * dz;
            wv[0] += gx * dx; wv[1] += gx * dy; wv[2] += gx * dz;
            wv[3] += gy * dx; wv[4] += gy * dy; wv[5] += gy * dz;
            wv[6] += gz * dx; wv[7] += gz * dy; wv[8] += gz * dz;
        }
    }
    // ds/dr_k = scale * sum g * (-d)  ->  F_k += -fs*dVds*ds/dr_k = +fs*scale*dVds * sum g*d
    if (act) {
        const double a = coef * dVds[0];
        const int i = perm[s];
        F[3 * i] += (T)(a * (double)ax);
        F[3 * i + 1] += (T)(a * (double)ay);
        F[3 * i + 2] += (T)(a * (double)az);
    }
    if (VIRIAL) {
        double w[9];
#pragma unroll
        for (int q = 0; q < 9; ++q) w[q] = (double)wv[q];
        virial_finish(w, vsm, va, -0.5 * coef, dVds);
    }
}

// Warp-per-atom variants for small systems (N <= METAD_WARP_PER_ATOM_MAX): the lanes share an atom's neighbours, a fixed
// shuffle tree sums the lane partials (deterministic).  Same arithmetic per pair as the thread-per-atom kernels.
template <typename T, int G>
__global__ void __launch_bounds__(CV_THREADS)
k_coord_cv_warp(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ nl_count,
                const int *__restrict__ nl, PBox<T> pb, BoxD bdk, T rc2T, double rc2k /* Verlet skin: keep pairs with r < rc only; 0 = the list is exact */, int fshift /* this CV's bits of the group flags */, T inv_r0, int n, int m, double scale,
                double *__restrict__ partials, unsigned int *__restrict__ ticket, double *__restrict__ cv_out,
                unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg) {
    __shared__ double red[32];
    if (dg) { pb = dg_pb<T>(dg); bdk = dg->bd; }
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int s = gt / G, lane = gt % G;
    T acc = T(0);
    if (s < N) {
        typename Vec4<T>::type pi = spos[s];
        if ((((int)pi.w) >> fshift) & 1) {
            const int cnt = nl_count[s];
            for (int k = lane; k < cnt; k += G) {
                const int j = nl[(size_t)k * N + s];
                typename Vec4<T>::type pj = ldg4<T>(spos + j);
                if (!((((int)pj.w) >> fshift) & 2)) continue;
                if (rc2k > 0.0 && !pair_in_range<T>(pb, bdk, rc2T, rc2k, pi, pj)) continue;
                T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                min_image(pb, dx, dy, dz);
                T r = sqrt(dx * dx + dy * dy + dz * dz), dsw;
                acc += switch_fn<T>(r * inv_r0, n, m, dsw);
            }
        }
    }
    double v[1] = { (double)acc };
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

template <typename T, int G>
__global__ void __launch_bounds__(CV_THREADS)
k_coord_force_warp(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ nl_count,
                   const int *__restrict__ nl, const int *__restrict__ perm, PBox<T> pb, BoxD bdk, T rc2T, double rc2k /* Verlet skin: keep pairs with r < rc only; 0 = the list is exact */, int fshift /* this CV's bits of the group flags */, T inv_r0, int n, int m,
                   double coef /* force_scale*scale */, const double *__restrict__ dVds, T *__restrict__ F,
                   const DevGeom *__restrict__ dg) {
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int s = gt / G, lane = gt % G;
    if (s >= N) return;
    if (dg) { pb = dg_pb<T>(dg); bdk = dg->bd; }
    const unsigned gmask = G == 32 ? 0xffffffffu : (((1u << G) - 1u) << ((threadIdx.x & 31) / G * G));
    typename Vec4<T>::type pi = spos[s];
    const int fi = ((int)pi.w) >> fshift;
    T ax = T(0), ay = T(0), az = T(0);
    const int cnt = (fi & 3) ? nl_count[s] : 0;             // an atom in neither group takes no force
    for (int k = lane; k < cnt; k += G) {
        const int j = nl[(size_t)k * N + s];
        typename Vec4<T>::type pj = ldg4<T>(spos + j);
        const int fj = ((int)pj.w) >> fshift;
        const int mult = ((fi & 1) && (fj & 2)) + ((fi & 2) && (fj & 1));
        if (!mult) continue;
        if (rc2k > 0.0 && !pair_in_range<T>(pb, bdk, rc2T, rc2k, pi, pj)) continue;
        T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        min_image(pb, dx, dy, dz);
        T r = sqrt(dx * dx + dy * dy + dz * dz), dsw;
        switch_fn<T>(r * inv_r0, n, m, dsw);
        T g = T(mult) * dsw * inv_r0 / r;
        ax += g * dx; ay += g * dy; az += g * dz;
    }
#pragma unroll
    for (int o = G / 2; o > 0; o >>= 1) {
        ax += __shfl_down_sync(gmask, ax, o, G);
        ay += __shfl_down_sync(gmask, ay, o, G);
        az += __shfl_down_sync(gmask, az, o, G);
    }
    if (lane == 0 && (fi & 3)) {
        const double a = coef * dVds[0];
        const int i = perm[s];
        F[3 * i] += (T)(a * (double)ax);
        F[3 * i + 1] += (T)(a * (double)ay);
        F[3 * i + 2] += (T)(a * (double)az);
    }
}

// ------------------------------------------------------------------------------------------------
// Q6 pass 1: per-atom q6m accumulation -> record + block partials of (sum q6, sum f(q6))
template <typename T>
__global__ void __launch_bounds__(CV_THREADS, 5)        // fp64: 96 registers instead of 120, five blocks per SM: 0.305 -> 0.262 ms at c3
k_q6_pass1(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ nl_count,
           const int *__restrict__ nl, PBox<T> pb, BoxD bdk, T rc2T, double rc2k /* Verlet skin: keep pairs with r < rc only; 0 = the list is exact */, T q_thresh, T inv_width, T *__restrict__ rec,
           T *__restrict__ q6arr /* [N] q6, then [N] f'(q6) */,
           double scale_mean, double scale_solid, int dim_mean, int dim_solid,
           double *__restrict__ partials, unsigned int *__restrict__ ticket, double *__restrict__ cv_out,
           unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg) {
    __shared__ double red[64];
    if (dg) { pb = dg_pb<T>(dg); bdk = dg->bd; }
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    double v[2] = { 0.0, 0.0 };
    if (s < N) {
        typename Vec4<T>::type pi = spos[s];
        T A[13];
#pragma unroll
        for (int k = 0; k < 13; ++k) A[k] = T(0);
        const int nlist = nl_count[s];
        int cnt = 0;                                     // neighbours within rc (== nlist unless a skin keeps a longer list)
        // list entries are fetched two iterations ahead: the chain entry -> position gather is what a thread waits on
        int e0 = nlist > 0 ? nl[s] : 0, e1 = nlist > 1 ? nl[(size_t)N + s] : 0;
        for (int k = 0; k < nlist; ++k) {
            const int j = e0;
            e0 = e1;
            if (k + 2 < nlist) e1 = nl[(size_t)(k + 2) * N + s];
            typename Vec4<T>::type pj = ldg4<T>(spos + j);
            if (rc2k > 0.0 && !pair_in_range<T>(pb, bdk, rc2T, rc2k, pi, pj)) continue;
            ++cnt;
            T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
            min_image(pb, dx, dy, dz);
            T rinv = T(1) / sqrt(dx * dx + dy * dy + dz * dz);
            Y6<T> y;
            y6_eval<T>(dx * rinv, dy * rinv, dz * rinv, y);
            A[0] += y.E[0];
#pragma unroll
            for (int m = 1; m <= 6; ++m) {
                A[2 * m - 1] += y.E[m] * y.c[m];
                A[2 * m] += y.E[m] * y.s[m];
            }
        }
        T S = T(0);
#pragma unroll
        for (int k = 0; k < 13; ++k) S += A[k] * A[k];
        T q6 = T(0), fsw = T(0), dfsw = T(0), norm = T(0);
        if (cnt > 0 && S > T(0)) {
            T rs = sqrt(S);
            q6 = rs / T(cnt);
            norm = T(1) / (T(cnt) * rs);
        }
        {
            T f = T(1) / (T(1) + exp(-(q6 - q_thresh) * inv_width));
            fsw = f;
            dfsw = f * (T(1) - f) * inv_width;
        }
        // record: B_m = conj(A_m)/(n sqrt(S)); [13..15] = the atom's position (one gather per pair in the force pass)
        T out[METAD_NREC];
        out[0] = A[0] * norm;
#pragma unroll
        for (int m = 1; m <= 6; ++m) { out[2 * m - 1] = A[2 * m - 1] * norm; out[2 * m] = -A[2 * m] * norm; }
        out[13] = pi.x; out[14] = pi.y; out[15] = pi.z;
        q6arr[s] = q6; q6arr[(size_t)N + s] = dfsw;
        typename Vec4<T>::type *r4 = reinterpret_cast<typename Vec4<T>::type *>(rec + (size_t)s * METAD_NREC);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            typename Vec4<T>::type w;
            w.x = out[4 * q]; w.y = out[4 * q + 1]; w.z = out[4 * q + 2]; w.w = out[4 * q + 3];
            st4<T>(r4 + q, w);
        }
        v[0] = (double)q6; v[1] = (double)fsw;
    }
    block_reduce<2>(v, red);
    if (threadIdx.x == 0) { partials[2 * blockIdx.x] = v[0]; partials[2 * blockIdx.x + 1] = v[1]; }
    if (last_block_ticket(ticket)) {
        double t[2] = { 0.0, 0.0 };
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) { t[0] += partials[2 * b]; t[1] += partials[2 * b + 1]; }
        block_reduce<2>(t, red);
        if (threadIdx.x == 0) {
            double a = scale_mean * t[0], b = scale_solid * t[1];
            if (dim_mean >= 0) cv_out[dim_mean] = a;
            if (dim_solid >= 0) cv_out[dim_solid] = b;
            if (!isfinite(a) || !isfinite(b)) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
        }
    }
}

// Q6 pass 2 (gather form, reading E):  F_k += fs * sum_{j in N(k)} grad_d [ (g_k B(k) + g_j B(j)) . y ](d_kj),
// g_i = alpha + beta f'(q6_i), alpha = dVds[mean]*scale_mean, beta = dVds[solid]*scale_solid.
template <typename T, bool VIRIAL>
__global__ void __launch_bounds__(CV_THREADS)
k_q6_force(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ nl_count,
           const int *__restrict__ nl, const int *__restrict__ perm, PBox<T> pb, BoxD bdk, T rc2T, double rc2k /* Verlet skin: keep pairs with r < rc only; 0 = the list is exact */, const T *__restrict__ rec,
           const T *__restrict__ fprime /* [N] f'(q6) */, double scale_mean, double scale_solid, int dim_mean, int dim_solid, double force_scale,
           const double *__restrict__ dVds, T *__restrict__ F, VirArgs va, const DevGeom *__restrict__ dg) {
    typedef typename Vec4<T>::type V4;
    if (dg) { pb = dg_pb<T>(dg); bdk = dg->bd; }
    __shared__ double vsm[VIRIAL ? 9 * 32 : 1];
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (!VIRIAL && s >= N) return;
    const bool act = s < N;
    if (!act) s = N - 1;
    T wv[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) wv[q] = T(0);
    const T alpha = dim_mean >= 0 ? (T)(dVds[dim_mean] * scale_mean) : T(0);
    const T beta = dim_solid >= 0 ? (T)(dVds[dim_solid] * scale_solid) : T(0);
    V4 pi = spos[s];
    T Bk[13];
    {
        const V4 *r4 = reinterpret_cast<const V4 *>(rec + (size_t)s * METAD_NREC);
        V4 a = ldg4<T>(r4), b = ldg4<T>(r4 + 1), c = ldg4<T>(r4 + 2), d = ldg4<T>(r4 + 3);
        T gk = beta != T(0) ? alpha + beta * fprime[s] : alpha;
        Bk[0] = gk * a.x; Bk[1] = gk * a.y; Bk[2] = gk * a.z; Bk[3] = gk * a.w;
        Bk[4] = gk * b.x; Bk[5] = gk * b.y; Bk[6] = gk * b.z; Bk[7] = gk * b.w;
        Bk[8] = gk * c.x; Bk[9] = gk * c.y; Bk[10] = gk * c.z; Bk[11] = gk * c.w;
        Bk[12] = gk * d.x;
    }
    T ax = T(0), ay = T(0), az = T(0);
    int cnt = act ? nl_count[s] : 0;
    int e0 = cnt > 0 ? nl[s] : 0, e1 = cnt > 1 ? nl[(size_t)N + s] : 0;      // entries two iterations ahead (as in pass 1)
    for (int k = 0; k < cnt; ++k) {
        const int j = e0;
        e0 = e1;
        if (k + 2 < cnt) e1 = nl[(size_t)(k + 2) * N + s];
        // the record carries the neighbour's position: four gathers of one array per pair instead of five of two
        const V4 *r4 = reinterpret_cast<const V4 *>(rec + (size_t)j * METAD_NREC);
        V4 d = ldg4<T>(r4 + 3), pj;
        pj.x = d.y; pj.y = d.z; pj.z = d.w; pj.w = T(0);
        if (rc2k > 0.0 && !pair_in_range<T>(pb, bdk, rc2T, rc2k, pi, pj)) continue;
        V4 a = ldg4<T>(r4), b = ldg4<T>(r4 + 1), c = ldg4<T>(r4 + 2);
        T gj = beta != T(0) ? alpha + beta * fprime[j] : alpha;
        T bb[13];
        bb[0] = Bk[0] + gj * a.x; bb[1] = Bk[1] + gj * a.y; bb[2] = Bk[2] + gj * a.z; bb[3] = Bk[3] + gj * a.w;
        bb[4] = Bk[4] + gj * b.x; bb[5] = Bk[5] + gj * b.y; bb[6] = Bk[6] + gj * b.z; bb[7] = Bk[7] + gj * b.w;
        bb[8] = Bk[8] + gj * c.x; bb[9] = Bk[9] + gj * c.y; bb[10] = Bk[10] + gj * c.z; bb[11] = Bk[11] + gj * c.w;
        bb[12] = Bk[12] + gj * d.x;
        T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        min_image(pb, dx, dy, dz);
        T rinv = T(1) / sqrt(dx * dx + dy * dy + dz * dz);
        T ux = dx * rinv, uy = dy * rinv, uz = dz * rinv;
        Y6<T> y;
        y6_eval<T>(ux, uy, uz, y);
        T gx, gy, gz;
        y6_grad<T>(y, bb, gx, gy, gz);
        T gu = gx * ux + gy * uy + gz * uz;     // project onto the tangent plane, divide by r
        const T tx = (gx - gu * ux) * rinv, ty = (gy - gu * uy) * rinv, tz = (gz - gu * uz) * rinv;
        ax += tx; ay += ty; az += tz;
        if (VIRIAL) {
            wv[0] += tx * dx; wv[1] += tx * dy; wv[2] += tx * dz;
            wv[3] += ty * dx; wv[4] += ty * dy; wv[5] += ty * dz;
            wv[6] += tz * dx; wv[7] += tz * dy; wv[8] += tz * dz;
        }
    }
    if (act) {
        const int i = perm[s];
        F[3 * i] += (T)(force_scale * (double)ax);
        F[3 * i + 1] += (T)(force_scale * (double)ay);
        F[3 * i + 2] += (T)(force_scale * (double)az);
    }
    if (VIRIAL) {                               // alpha, beta already carry dV/ds: W = -1/2 force_scale sum t d^T
        double w[9];
#pragma unroll
        for (int q = 0; q < 9; ++q) w[q] = (double)wv[q];
        virial_finish(w, vsm, va, -0.5 * force_scale, nullptr);
    }
}

// ------------------------------------------------------------------------------------------------
// Q6 pass 2 for the tiled fp32 path.  Neighbour entries are (global sorted index | lattice-shift
// code << 27) in the sliced layout written by k_tile_build.  Per pair: one 128-bit load of the
// neighbour position and two 256-bit loads (LDG.E.256, sm_100) of its 64-byte q6 record — half the
// L1 requests of four 128-bit loads, which is what bounds this gather (profiles/r1a_ncu_top3.md).
// Pairs across a periodic boundary (code != 13, a few %) form d in fp64 from the exact inputs.
#define NLG_IDX_MASK ((1 << 27) - 1)
__device__ __forceinline__ void ldg256(const float *p, float4 &a, float4 &b) {
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
                 : "l"(p));
}

#define Q6F_MINB 9             // resident blocks per SM of k_q6_force_g (56 registers)
// SKIN (params.skin): the kept list reaches rc + skin and a neighbour may have crossed a box face since it was built (the caller
// re-wraps), so the shift codes are ignored and the image is found from the current positions.  The raw difference d = pj - pi
// settles almost every pair: with perpendicular box widths W >= 2 (rc + skin) (the box check of this mode) any other image lies
// at |d - t| >= W - |d|, so for |d|^2 <= far2 = (rc + 2 skin)^2 (1 - 1e-4) no other image is within rc — d is the minimum
// image if |d| < rc and the pair is out of range otherwise.  Only pairs beyond far2 (across a periodic face, a few %) take the
// minimum image, in fp64 on the exact fp32 inputs (the fp32 form is not accurate enough for the forces in a 255 A box,
// profiles/r2_experiments.md).  Pass 1 and the force pass share this function, so both see the same displacement.
__device__ __forceinline__ void skin_displacement(const BoxD &b, float far2, const float4 &pi, const float4 &pj,
                                                  float &dx, float &dy, float &dz) {
    if (dx * dx + dy * dy + dz * dz > far2) {
        double ex = (double)pj.x - (double)pi.x, ey = (double)pj.y - (double)pi.y, ez = (double)pj.z - (double)pi.z;
        min_image_d(b, ex, ey, ez);
        dx = (float)ex; dy = (float)ey; dz = (float)ez;
    }
}
// The kernel walks the compacted rc list that pass 1 (k_q6_pass1_g) wrote for this step, so no record of a pair beyond rc is gathered.
template <bool SOLID, bool VIRIAL, bool DEVBOX, bool SKIN>   // DEVBOX: box in device memory (metad_*_dev); the other instances never touch dg
__global__ void __launch_bounds__(CV_THREADS, VIRIAL ? 8 : Q6F_MINB)
k_q6_force_g(int N, int maxn, const float4 *__restrict__ spos, const int *__restrict__ nl_count,
             const int *__restrict__ nl, const int *__restrict__ perm, BoxD bd, const float *__restrict__ rec,
             double scale_mean, double scale_solid, int dim_mean, int dim_solid, double force_scale,
             const double *__restrict__ dVds, float *__restrict__ F, VirArgs va, const float *__restrict__ fprime,
             const DevGeom *__restrict__ dg_arg, float far2 /* SKIN: see skin_displacement */) {
    const DevGeom *dg = DEVBOX ? dg_arg : nullptr;
    __shared__ double vsm[VIRIAL ? 9 * 32 : 1];
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (!VIRIAL && s >= N) return;
    const bool act = s < N;
    if (!act) s = N - 1;                       // idle thread of the virial instance: valid addresses, zero trip count
    float wv[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) wv[q] = 0.f;
    const float alpha = dim_mean >= 0 ? (float)(dVds[dim_mean] * scale_mean) : 0.f;
    const float beta = dim_solid >= 0 ? (float)(dVds[dim_solid] * scale_solid) : 0.f;
    const float4 pi = spos[s];
    const float *__restrict__ recB = rec + (size_t)N * 8;
    float Bk[13];
    {
        float4 a4, b4, c4, d4;
        ldg256(rec + (size_t)s * 8, a4, b4);                 // split layout of the tiled path (tiled.cu: finish_atom)
        ldg256(recB + (size_t)s * 8, c4, d4);
        const float gk = SOLID ? alpha + beta * fprime[s] : alpha;
        Bk[0] = gk * a4.x; Bk[1] = gk * a4.y; Bk[2] = gk * a4.z; Bk[3] = gk * a4.w;
        Bk[4] = gk * b4.x; Bk[5] = gk * b4.y; Bk[6] = gk * b4.z; Bk[7] = gk * b4.w;
        Bk[8] = gk * c4.x; Bk[9] = gk * c4.y; Bk[10] = gk * c4.z; Bk[11] = gk * c4.w;
        Bk[12] = gk * d4.x;
    }
    const int *in = nl + ((size_t)(s >> 5) * maxn) * 32 + (s & 31);
    const int cnt = act ? nl_count[s] : 0;
    float fx = 0.f, fy = 0.f, fz = 0.f;
    // the list entries are fetched two iterations ahead: an entry load (streamed from DRAM) followed by the dependent record
    // gather was 40 % of the stall samples of this kernel (profiles/r1w_ncu.md)
    int e0 = cnt > 0 ? __ldcs(in) : 0, e1 = cnt > 1 ? __ldcs(in + 32) : 0;
    for (int k = 0; k < cnt; ++k) {
        const int e = e0;                              // streamed once: do not displace positions / records in L2
        e0 = e1;
        if (k + 2 < cnt) e1 = __ldcs(in + (k + 2) * 32);
        const int j = e & NLG_IDX_MASK, code = (unsigned)e >> 27;
        float4 a4, b4, c4, d4, pj;
        ldg256(rec + (size_t)j * 8, a4, b4);
        ldg256(recB + (size_t)j * 8, c4, d4);
        pj.x = d4.y; pj.y = d4.z; pj.z = d4.w;               // the record carries the position
        float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        if (SKIN) {
            skin_displacement(dg ? dg->bd : bd, far2, pi, pj, dx, dy, dz);   // the image pass 1 decided r < rc on
        } else if (code != 13) {
            const int wx = code % 3 - 1, wy = (code / 3) % 3 - 1, wz = code / 9 - 1;
            const BoxD &b = dg ? dg->bd : bd;                  // device-resident box (NPT): read at the rare point of use
            dx = (float)(((double)pj.x - (double)pi.x) + (wx * b.ax + wy * b.bx + wz * b.cx));
            dy = (float)(((double)pj.y - (double)pi.y) + (wy * b.by + wz * b.cy));
            dz = (float)(((double)pj.z - (double)pi.z) + (wz * b.cz));
        }
        const float gw = SOLID ? alpha + beta * fprime[j] : alpha;   // 4-byte gather from a dense array: few lines per warp
        float bb[13];
        bb[0] = Bk[0] + gw * a4.x; bb[1] = Bk[1] + gw * a4.y; bb[2] = Bk[2] + gw * a4.z; bb[3] = Bk[3] + gw * a4.w;
        bb[4] = Bk[4] + gw * b4.x; bb[5] = Bk[5] + gw * b4.y; bb[6] = Bk[6] + gw * b4.z; bb[7] = Bk[7] + gw * b4.w;
        bb[8] = Bk[8] + gw * c4.x; bb[9] = Bk[9] + gw * c4.y; bb[10] = Bk[10] + gw * c4.z; bb[11] = Bk[11] + gw * c4.w;
        bb[12] = Bk[12] + gw * d4.x;
        const float rinv = rsqrtf(dx * dx + dy * dy + dz * dz);
        const float ux = dx * rinv, uy = dy * rinv, uz = dz * rinv;
        Y6<float> y;
        y6_eval<float>(ux, uy, uz, y);
        float gx, gy, gz;
        y6_grad<float>(y, bb, gx, gy, gz);
        const float gu = gx * ux + gy * uy + gz * uz;
        const float tx = (gx - gu * ux) * rinv, ty = (gy - gu * uy) * rinv, tz = (gz - gu * uz) * rinv;
        fx += tx; fy += ty; fz += tz;
        if (VIRIAL) {
            // t is tangential in exact arithmetic; in fp32 it keeps a radial residue (g.u)(1 - |u|^2) u / r, and g.u has ONE
            // sign for most pairs (it is 6 x the pair's share of q6), so the residue adds up coherently in the trace of the
            // virial (1.1e-5 against a traceless Q6 virial of 0.27 at 1,024,000 atoms; per atom it is far inside the force
            // tolerance).  Projected out against d itself before the outer product.
            const float td = (tx * dx + ty * dy + tz * dz) * (rinv * rinv);
            const float px = tx - td * dx, py = ty - td * dy, pz = tz - td * dz;
            wv[0] += px * dx; wv[1] += px * dy; wv[2] += px * dz;
            wv[3] += py * dx; wv[4] += py * dy; wv[5] += py * dz;
            wv[6] += pz * dx; wv[7] += pz * dy; wv[8] += pz * dz;
        }
    }
    if (act) {
        const int i = perm[s];
        F[3 * i] += (float)(force_scale * (double)fx);
        F[3 * i + 1] += (float)(force_scale * (double)fy);
        F[3 * i + 2] += (float)(force_scale * (double)fz);
    }
    if (VIRIAL) {                               // alpha, beta already carry dV/ds: W = -1/2 force_scale sum t d^T
        double w[9];
#pragma unroll
        for (int q = 0; q < 9; ++q) w[q] = (double)wv[q];
        virial_finish(w, vsm, va, -0.5 * force_scale, nullptr);
    }
}

// Q6 pass 1 from the KEPT list of the tiled fp32 path (params.skin): thread per atom over the sliced list, one 128-bit
// position gather per entry, image from the current positions (skin_displacement), pairs beyond rc skipped with the
// canonical decision inside the recheck band; writes the same split records, per-atom q6 and f'(q6) as the fused pass of
// k_tile_build and finishes the global sums in its last block.
template <bool DEVBOX>
__global__ void __launch_bounds__(CV_THREADS, 10)
k_q6_pass1_g(int N, int maxn, const float4 *__restrict__ spos, const int *__restrict__ nl_count, const int *__restrict__ nl,
             PBox<float> pb, BoxD bd, float rc2f, double rc2, float q_thresh, float inv_width, float *__restrict__ rec,
             float *__restrict__ q6_out, int solid, double scale_mean, double scale_solid, double *__restrict__ partials,
             unsigned int *__restrict__ ticket, double *__restrict__ cv_q6, double *__restrict__ cv_out, int dim0, int dim1,
             unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg,
             int *__restrict__ rc_count, int *__restrict__ rc_list /* the entries within rc, same sliced layout: read by the force pass */,
             float far2) {
    __shared__ double red[64];
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (DEVBOX) pb = dg->pbf;                      // host-box instance: the box stays in the constant bank
    double v[2] = { 0.0, 0.0 };
    if (s < N) {
        const float4 pi = spos[s];
        const int *in = nl + ((size_t)(s >> 5) * maxn) * 32 + (s & 31);
        const int cnt = nl_count[s];
        float A[13];
#pragma unroll
        for (int k = 0; k < 13; ++k) A[k] = 0.f;
        int n = 0;
        int *out = rc_list + ((size_t)(s >> 5) * maxn) * 32 + (s & 31);
        // entries two iterations ahead, as in k_q6_force_g: the entry load -> position gather chain is the latency to hide
        int e0 = cnt > 0 ? __ldg(in) : 0, e1 = cnt > 1 ? __ldg(in + 32) : 0;
        for (int k = 0; k < cnt; ++k) {
            const int e = e0, j = e0 & NLG_IDX_MASK;
            e0 = e1;
            if (k + 2 < cnt) e1 = __ldg(in + (k + 2) * 32);
            const float4 pj = spos[j];
            float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
            skin_displacement(DEVBOX ? dg->bd : bd, far2, pi, pj, dx, dy, dz);
            const float r2 = dx * dx + dy * dy + dz * dz;
            bool keep = r2 < rc2f;
            if (fabsf(r2 - rc2f) <= pb.band)
                keep = r2_canonical(DEVBOX ? dg->bd : bd, (double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y,
                                    (double)pj.z - (double)pi.z) < rc2;
            if (!keep) continue;
            __stcs(out + n * 32, e);                   // read once, by the force pass of this step
            ++n;
            const float rinv = rsqrtf(r2);
            Y6<float> y;
            y6_eval<float>(dx * rinv, dy * rinv, dz * rinv, y);
            A[0] += y.E[0];
#pragma unroll
            for (int m = 1; m <= 6; ++m) { A[2 * m - 1] += y.E[m] * y.c[m]; A[2 * m] += y.E[m] * y.s[m]; }
        }
        rc_count[s] = n;
        float S = 0.f;
#pragma unroll
        for (int k = 0; k < 13; ++k) S += A[k] * A[k];
        float q6 = 0.f, norm = 0.f;
        if (n > 0 && S > 0.f) { const float rs = sqrtf(S); q6 = rs / (float)n; norm = 1.f / ((float)n * rs); }
        float4 *r4 = reinterpret_cast<float4 *>(rec + (size_t)s * 8);                      // split record layout of tiled.cu
        float4 *r4b = reinterpret_cast<float4 *>(rec + (size_t)N * 8 + (size_t)s * 8) - 2;
        r4[0] = make_float4(A[0] * norm, A[1] * norm, -A[2] * norm, A[3] * norm);
        r4[1] = make_float4(-A[4] * norm, A[5] * norm, -A[6] * norm, A[7] * norm);
        r4b[2] = make_float4(-A[8] * norm, A[9] * norm, -A[10] * norm, A[11] * norm);
        r4b[3] = make_float4(-A[12] * norm, pi.x, pi.y, pi.z);
        const float f = 1.f / (1.f + expf(-(q6 - q_thresh) * inv_width));
        if (solid) q6_out[(size_t)N + s] = f * (1.f - f) * inv_width;
        q6_out[s] = q6;
        v[0] = (double)q6; v[1] = (double)f;
    }
    block_reduce<2>(v, red);
    if (threadIdx.x == 0) { partials[2 * blockIdx.x] = v[0]; partials[2 * blockIdx.x + 1] = v[1]; }
    if (last_block_ticket(ticket)) {
        double u[2] = { 0.0, 0.0 };
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) { u[0] += partials[2 * b]; u[1] += partials[2 * b + 1]; }
        block_reduce<2>(u, red);
        if (threadIdx.x == 0) {
            cv_q6[0] = scale_mean * u[0]; cv_q6[1] = scale_solid * u[1];
            if (dim0 >= 0) cv_out[dim0] = cv_q6[0];
            if (dim1 >= 0) cv_out[dim1] = cv_q6[1];
            if (!isfinite(cv_q6[0]) || !isfinite(cv_q6[1])) atomicOr(sticky, (unsigned)METAD_DEV_NONFINITE);
        }
    }
}

// threshold of skin_displacement: (rc + 2 skin)^2, a little inside
static float skin_far2(const metad_ctx *c) {
    const double r = c->rc + 2.0 * (c->rcl - c->rc);
    return (float)(r * r * (1.0 - 1e-4));
}

int tiled_q6_pass1_skin(metad_ctx *c, double *d_cv) {
    const double qt = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_thresh : 0.0;
    const double qw = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_width : 1.0;
#define P1G_ARGS                                                                                                           \
    c->N, c->maxn, (const float4 *)c->d_spos, c->d_nl_count, c->d_nl, ctx_pbox<float>(c), c->boxd, (float)c->rc2, c->rc2,  \
        (float)qt, (float)(1.0 / qw), (float *)c->d_rec, c->d_q6, c->q6_solid_dim >= 0 ? 1 : 0,                            \
        c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0, c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0, \
        c->d_partials + c->nblocks_atoms, c->d_tickets + 1, c->d_cvq6, d_cv, c->q6_mean_dim, c->q6_solid_dim, c->d_sticky, c->dg, c->d_rc_count, c->d_rc_list, skin_far2(c)
    if (c->dg) k_q6_pass1_g<true><<<div_up(c->N, CV_THREADS), CV_THREADS, 0, c->stream>>>(P1G_ARGS);
    else k_q6_pass1_g<false><<<div_up(c->N, CV_THREADS), CV_THREADS, 0, c->stream>>>(P1G_ARGS);
#undef P1G_ARGS
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

// Coordination-number forces on the tiled fp32 path (ungrouped: every ordered pair counts, i.e. each pair twice in
// d s/d r_k): thread per atom, gather form over the sliced list; per pair one 128-bit position load.
template <bool VIRIAL>
__global__ void __launch_bounds__(CV_THREADS)
k_coord_force_g(int N, int maxn, const float4 *__restrict__ spos, const int *__restrict__ nl_count,
                const int *__restrict__ nl, const int *__restrict__ perm, BoxD bd, float inv_r0, int n, int m,
                double coef /* force_scale * scale */, const double *__restrict__ dVds, float *__restrict__ F, VirArgs va,
                const DevGeom *__restrict__ dg) {
    __shared__ double vsm[VIRIAL ? 9 * 32 : 1];
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (!VIRIAL && s >= N) return;
    const bool act = s < N;
    if (!act) s = N - 1;
    float wv[9];
#pragma unroll
    for (int q = 0; q < 9; ++q) wv[q] = 0.f;
    const float4 pi = spos[s];
    const int *in = nl + ((size_t)(s >> 5) * maxn) * 32 + (s & 31);
    const int cnt = act ? nl_count[s] : 0;
    float ax = 0.f, ay = 0.f, az = 0.f;
    for (int k = 0; k < cnt; ++k) {
        const int e = __ldcs(in + k * 32);            // streamed once: do not displace positions / records in L2
        const int j = e & NLG_IDX_MASK, code = (unsigned)e >> 27;
        const float4 pj = spos[j];
        float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
        if (code != 13) {
            const int wx = code % 3 - 1, wy = (code / 3) % 3 - 1, wz = code / 9 - 1;
            const BoxD &b = dg ? dg->bd : bd;
            dx = (float)(((double)pj.x - (double)pi.x) + (wx * b.ax + wy * b.bx + wz * b.cx));
            dy = (float)(((double)pj.y - (double)pi.y) + (wy * b.by + wz * b.cy));
            dz = (float)(((double)pj.z - (double)pi.z) + (wz * b.cz));
        }
        const float r2 = dx * dx + dy * dy + dz * dz, rinv = rsqrtf(r2);
        float dsw;
        switch_fn<float>(r2 * rinv * inv_r0, n, m, dsw);
        const float g = 2.f * dsw * inv_r0 * rinv;
        ax += g * dx; ay += g * dy; az += g * dz;
        if (VIRIAL) {
            const float gx = g * dx, gy = g * dy, gz = g * dz;
            wv[0] += gx * dx; wv[1] += gx * dy; wv[2] += gx * dz;
            wv[3] += gy * dx; wv[4] += gy * dy; wv[5] += gy * dz;
            wv[6] += gz * dx; wv[7] += gz * dy; wv[8] += gz * dz;
        }
    }
    if (act) {
        const double a = coef * dVds[0];
        const int i = perm[s];
        F[3 * i] += (float)(a * (double)ax);
        F[3 * i + 1] += (float)(a * (double)ay);
        F[3 * i + 2] += (float)(a * (double)az);
    }
    if (VIRIAL) {
        double w[9];
#pragma unroll
        for (int q = 0; q < 9; ++q) w[q] = (double)wv[q];
        virial_finish(w, vsm, va, -0.5 * coef, dVds);
    }
}

// Coalesced force update of the tiled coordination path: F[i] += a * v[i] for a float4 array v in ORIGINAL atom order, one
// thread per force component (F is [N][3], 12-byte rows: consecutive threads touch consecutive floats of F).
// v = the per-atom gradient sum_j 2 sw'(r_ij) d_ij / (r0 r_ij) that k_tile_build<2> accumulated on its exact pass (tiled.cu):
// it does not depend on dV/ds, so the coordination force stage is this one scaled add per atom, no list walk, no gathers;
// a = force_scale * scale * dV/ds.  (The same split for the Q6 forces — k_q6_force_g storing into a scratch array in original
// order, this pass adding it — was measured and dropped: profiles/r1h_rejected.md.)
__global__ void __launch_bounds__(256)
k_force_add(int N, const float *__restrict__ v4, double coef, const double *__restrict__ dVds, float *__restrict__ F) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 3 * N) return;
    const int i = t / 3, k = t - 3 * i;
    const double a = coef * dVds[0];
    F[t] += (float)(a * (double)v4[4 * i + k]);
}

// the same update with 128-bit accesses, four atoms per thread (48 contiguous bytes of F, 64 of v); F must be 16-byte aligned
__global__ void __launch_bounds__(256)
k_force_add4(int N, const float4 *__restrict__ v4, double coef, const double *__restrict__ dVds, float *__restrict__ F) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (4 * t >= N) return;
    const double a = coef * dVds[0];
    if (4 * t + 3 < N) {
        float4 *F4 = reinterpret_cast<float4 *>(F) + 3 * (size_t)t;
        const float4 g0 = v4[4 * t], g1 = v4[4 * t + 1], g2 = v4[4 * t + 2], g3 = v4[4 * t + 3];
        float4 f0 = F4[0], f1 = F4[1], f2 = F4[2];
        f0.x += (float)(a * (double)g0.x); f0.y += (float)(a * (double)g0.y); f0.z += (float)(a * (double)g0.z);
        f0.w += (float)(a * (double)g1.x); f1.x += (float)(a * (double)g1.y); f1.y += (float)(a * (double)g1.z);
        f1.z += (float)(a * (double)g2.x); f1.w += (float)(a * (double)g2.y); f2.x += (float)(a * (double)g2.z);
        f2.y += (float)(a * (double)g3.x); f2.z += (float)(a * (double)g3.y); f2.w += (float)(a * (double)g3.z);
        F4[0] = f0; F4[1] = f1; F4[2] = f2;
    } else {
        for (int i = 4 * t; i < N; ++i) {
            const float4 g = v4[i];
            F[3 * i] += (float)(a * (double)g.x); F[3 * i + 1] += (float)(a * (double)g.y); F[3 * i + 2] += (float)(a * (double)g.z);
        }
    }
}

int tiled_coord_force(metad_ctx *c, const double *d_dVds, void *d_F) {
    const CvDev &d = c->cv[c->coord_dim];
    const VirArgs va = { c->d_vir_partials, c->d_tickets + 12, c->d_virial };
    if (!c->p.want_virial && c->d_cgrad && ((uintptr_t)d_F & 15) == 0)
        k_force_add4<<<div_up(div_up(c->N, 4), 256), 256, 0, c->stream>>>(c->N, (const float4 *)c->d_cgrad, c->p.force_scale * d.scale,
                                                                          d_dVds + c->coord_dim, (float *)d_F);
    else if (!c->p.want_virial && c->d_cgrad)
        k_force_add<<<div_up(3 * c->N, 256), 256, 0, c->stream>>>(c->N, c->d_cgrad, c->p.force_scale * d.scale,
                                                                  d_dVds + c->coord_dim, (float *)d_F);
    else if (c->p.want_virial)
        k_coord_force_g<true><<<div_up(c->N, CV_THREADS), CV_THREADS, 0, c->stream>>>(
            c->N, c->maxn, (const float4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm, c->boxd, (float)(1.0 / d.r0), d.n, d.m,
            c->p.force_scale * d.scale, d_dVds + c->coord_dim, (float *)d_F, va, c->dg);
    else
        k_coord_force_g<false><<<div_up(c->N, CV_THREADS), CV_THREADS, 0, c->stream>>>(
            c->N, c->maxn, (const float4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm, c->boxd, (float)(1.0 / d.r0), d.n, d.m,
            c->p.force_scale * d.scale, d_dVds + c->coord_dim, (float *)d_F, va, c->dg);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int tiled_q6_force(metad_ctx *c, const double *d_dVds, void *d_F) {
    double sm = c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0;
    double ss = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0;
    const VirArgs va = { c->d_vir_partials, c->d_tickets + 12, c->d_virial };
#define Q6FG_ARGS                                                                                                          \
    c->N, c->maxn, (const float4 *)c->d_spos, c->own_count_valid ? c->d_own_count : (c->skin_on ? c->d_rc_count : c->d_nl_count), c->skin_on ? c->d_rc_list : c->d_nl, c->d_perm, c->boxd, (const float *)c->d_rec, sm, ss,  \
        c->q6_mean_dim, c->q6_solid_dim, c->p.force_scale, d_dVds, (float *)d_F, va, c->d_q6 + c->N, c->dg, skin_far2(c)
#define Q6FG_GRID <<<div_up(c->N, CV_THREADS), CV_THREADS, 0, c->stream>>>
#define Q6FG_LAUNCH(SOLID, VIR)                                                                                            \
    do {                                                                                                                   \
        if (c->dg && c->skin_on) k_q6_force_g<SOLID, VIR, true, true> Q6FG_GRID(Q6FG_ARGS);                                \
        else if (c->dg) k_q6_force_g<SOLID, VIR, true, false> Q6FG_GRID(Q6FG_ARGS);                                        \
        else if (c->skin_on) k_q6_force_g<SOLID, VIR, false, true> Q6FG_GRID(Q6FG_ARGS);                                   \
        else k_q6_force_g<SOLID, VIR, false, false> Q6FG_GRID(Q6FG_ARGS);                                                  \
    } while (0)
    if (c->q6_solid_dim >= 0) { if (c->p.want_virial) Q6FG_LAUNCH(true, true); else Q6FG_LAUNCH(true, false); }
    else { if (c->p.want_virial) Q6FG_LAUNCH(false, true); else Q6FG_LAUNCH(false, false); }
#undef Q6FG_LAUNCH
#undef Q6FG_GRID
#undef Q6FG_ARGS
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

template <typename T>
__global__ void k_q6_export_arr(int N, const int *__restrict__ perm, const T *__restrict__ q6s, T *__restrict__ q6) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < N) q6[perm[s]] = q6s[s];
}

// ------------------------------------------------------------------------------------------------
// Distance to the nearest atom of a group (reading AA): arg-min over the neighbour list of (r^2, i, j) in
// ORIGINAL indices (ties -> smallest pair), block partials + last-block pass.  The result record feeds the force kernel.
struct MinKey { double r2; long long ij; };
__device__ __forceinline__ bool min_less(double r2a, long long ija, double r2b, long long ijb) {
    return r2a < r2b || (r2a == r2b && ija < ijb);
}
__device__ __forceinline__ void min_warp(double &r2, long long &ij, int &sj, int &si) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double r2o = __shfl_down_sync(0xffffffffu, r2, o);
        const long long ijo = __shfl_down_sync(0xffffffffu, ij, o);
        const int sjo = __shfl_down_sync(0xffffffffu, sj, o), sio = __shfl_down_sync(0xffffffffu, si, o);
        if (min_less(r2o, ijo, r2, ij)) { r2 = r2o; ij = ijo; sj = sjo; si = sio; }
    }
}

template <typename T>
__global__ void __launch_bounds__(CV_THREADS)
k_mindist_cv(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ nl_count,
             const int *__restrict__ nl, const int *__restrict__ perm, PBox<T> pb, BoxD bdk, T rc2T, double rc2k /* Verlet skin: keep pairs with r < rc only; 0 = the list is exact */, int fshift /* this CV's bits of the group flags */, double rc,
             double *__restrict__ part_r2, long long *__restrict__ part_ij, int *__restrict__ part_s /* [2*nblocks] */,
             unsigned int *__restrict__ ticket, double *__restrict__ rec /* [r, dx, dy, dz, (i, j) as two ints] */,
             double *__restrict__ cv_out, const DevGeom *__restrict__ dg) {
    __shared__ double s_r2[32];
    __shared__ long long s_ij[32];
    __shared__ int s_sj[32], s_si[32];
    if (dg) { pb = dg_pb<T>(dg); bdk = dg->bd; }
    const int s = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double r2 = 1e300; long long ij = 0x7fffffffffffffffll; int sj = -1, si = -1;
    if (s < N) {
        const typename Vec4<T>::type pi = spos[s];
        if ((((int)pi.w) >> fshift) & 1) {
            const int cnt = nl_count[s];
            const long long io = perm[s];
            for (int k = 0; k < cnt; ++k) {
                const int j = nl[(size_t)k * N + s];
                const typename Vec4<T>::type pj = ldg4<T>(spos + j);
                if (!((((int)pj.w) >> fshift) & 2)) continue;
                if (rc2k > 0.0 && !pair_in_range<T>(pb, bdk, rc2T, rc2k, pi, pj)) continue;
                T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                min_image(pb, dx, dy, dz);
                const double q = (double)(dx * dx + dy * dy + dz * dz);
                const long long key = (io << 32) | (long long)perm[j];
                if (min_less(q, key, r2, ij)) { r2 = q; ij = key; sj = j; si = s; }
            }
        }
    }
    min_warp(r2, ij, sj, si);
    if (lane == 0) { s_r2[wid] = r2; s_ij[wid] = ij; s_sj[wid] = sj; s_si[wid] = si; }
    __syncthreads();
    if (wid == 0) {
        const int nw = blockDim.x >> 5;
        r2 = lane < nw ? s_r2[lane] : 1e300; ij = lane < nw ? s_ij[lane] : 0x7fffffffffffffffll;
        sj = lane < nw ? s_sj[lane] : -1; si = lane < nw ? s_si[lane] : -1;
        min_warp(r2, ij, sj, si);
        if (lane == 0) { part_r2[blockIdx.x] = r2; part_ij[blockIdx.x] = ij; part_s[2 * blockIdx.x] = si; part_s[2 * blockIdx.x + 1] = sj; }
    }
    if (last_block_ticket(ticket)) {
        r2 = 1e300; ij = 0x7fffffffffffffffll; sj = -1; si = -1;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x)
            if (min_less(part_r2[b], part_ij[b], r2, ij)) { r2 = part_r2[b]; ij = part_ij[b]; si = part_s[2 * b]; sj = part_s[2 * b + 1]; }
        min_warp(r2, ij, sj, si);
        if (lane == 0) { s_r2[wid] = r2; s_ij[wid] = ij; s_sj[wid] = sj; s_si[wid] = si; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w)
                if (min_less(s_r2[w], s_ij[w], r2, ij)) { r2 = s_r2[w]; ij = s_ij[w]; sj = s_sj[w]; si = s_si[w]; }
            int *pair = reinterpret_cast<int *>(rec + 4);
            if (sj < 0) {                                   // nobody within rc: s = rc, no force
                rec[0] = rc; rec[1] = rec[2] = rec[3] = 0.0; pair[0] = pair[1] = -1;
                *cv_out = rc;
            } else {
                const typename Vec4<T>::type pi = spos[si], pj = spos[sj];
                T dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                min_image(pb, dx, dy, dz);
                const double r = sqrt((double)dx * (double)dx + (double)dy * (double)dy + (double)dz * (double)dz);
                rec[0] = r; rec[1] = (double)dx; rec[2] = (double)dy; rec[3] = (double)dz;
                pair[0] = (int)(ij >> 32); pair[1] = (int)(ij & 0xffffffffll);
                *cv_out = r;
            }
        }
    }
}

template <typename T>
__global__ void k_mindist_force(const double *__restrict__ rec, double force_scale, const double *__restrict__ dVds,
                                T *__restrict__ F, double *__restrict__ virial /* NULL: not wanted */) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const int *pair = reinterpret_cast<const int *>(rec + 4);
    if (pair[0] < 0) return;
    // d s/d r_j = d/r, d s/d r_i = -d/r  ->  F_j += -fs dVds d/r, F_i += +fs dVds d/r
    const double a = force_scale * dVds[0] / rec[0];
    for (int k = 0; k < 3; ++k) {
        F[3 * (size_t)pair[0] + k] += (T)(a * rec[1 + k]);
        F[3 * (size_t)pair[1] + k] += (T)(-a * rec[1 + k]);
    }
    if (virial)                                  // d s/d eps = d d^T / |d| (reading AD)
        for (int p = 0; p < 3; ++p)
            for (int q = 0; q < 3; ++q) virial[3 * p + q] += -a * rec[1 + p] * rec[1 + q];
}

// List-free variant for a few centres (ONE surface oxygen against all hydrogens): thread per group-B atom
// loops over the nA centres with the fp64 minimum image of reading O on the caller's positions; same arg-min reduction.
// Chosen when params.lazy_neighbors is set and MINDIST is the only CV that would read the list.
template <typename T>
__global__ void __launch_bounds__(CV_THREADS)
k_mindist_brute(int nA, const int *__restrict__ ga, int nB, const int *__restrict__ gb, const T *__restrict__ pos, BoxD bd,
                double rc, double *__restrict__ part_r2, long long *__restrict__ part_ij, unsigned int *__restrict__ ticket,
                double *__restrict__ rec, double *__restrict__ cv_out, const DevGeom *__restrict__ dg) {
    __shared__ double s_r2[32];
    __shared__ long long s_ij[32];
    if (dg) bd = dg->bd;
    const int t = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double r2 = 1e300; long long ij = 0x7fffffffffffffffll; int u0 = -1, u1 = -1;     // u0/u1 unused payload of min_warp
    const double rc2 = rc * rc;
    if (t < nB) {
        const int j = gb[t];
        const double xj = (double)pos[3 * (size_t)j], yj = (double)pos[3 * (size_t)j + 1], zj = (double)pos[3 * (size_t)j + 2];
        for (int a = 0; a < nA; ++a) {
            const int i = ga[a];
            if (i == j) continue;
            const double q = r2_canonical(bd, xj - (double)pos[3 * (size_t)i], yj - (double)pos[3 * (size_t)i + 1],
                                          zj - (double)pos[3 * (size_t)i + 2]);
            const long long key = ((long long)i << 32) | (long long)j;
            if (q < rc2 && min_less(q, key, r2, ij)) { r2 = q; ij = key; }
        }
    }
    min_warp(r2, ij, u0, u1);
    if (lane == 0) { s_r2[wid] = r2; s_ij[wid] = ij; }
    __syncthreads();
    if (wid == 0) {
        const int nw = blockDim.x >> 5;
        r2 = lane < nw ? s_r2[lane] : 1e300; ij = lane < nw ? s_ij[lane] : 0x7fffffffffffffffll;
        min_warp(r2, ij, u0, u1);
        if (lane == 0) { part_r2[blockIdx.x] = r2; part_ij[blockIdx.x] = ij; }
    }
    if (last_block_ticket(ticket)) {
        r2 = 1e300; ij = 0x7fffffffffffffffll;
        for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x)
            if (min_less(part_r2[b], part_ij[b], r2, ij)) { r2 = part_r2[b]; ij = part_ij[b]; }
        min_warp(r2, ij, u0, u1);
        if (lane == 0) { s_r2[wid] = r2; s_ij[wid] = ij; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w)
                if (min_less(s_r2[w], s_ij[w], r2, ij)) { r2 = s_r2[w]; ij = s_ij[w]; }
            int *pair = reinterpret_cast<int *>(rec + 4);
            if (!(r2 < 1e299)) {
                rec[0] = rc; rec[1] = rec[2] = rec[3] = 0.0; pair[0] = pair[1] = -1;
                *cv_out = rc;
            } else {
                const int i = (int)(ij >> 32), j = (int)(ij & 0xffffffffll);
                double dx = (double)pos[3 * (size_t)j] - (double)pos[3 * (size_t)i],
                       dy = (double)pos[3 * (size_t)j + 1] - (double)pos[3 * (size_t)i + 1],
                       dz = (double)pos[3 * (size_t)j + 2] - (double)pos[3 * (size_t)i + 2];
                min_image_d(bd, dx, dy, dz);
                const double r = sqrt(dx * dx + dy * dy + dz * dz);
                rec[0] = r; rec[1] = dx; rec[2] = dy; rec[3] = dz; pair[0] = i; pair[1] = j;
                *cv_out = r;
            }
        }
    }
}

template <typename T>
static int mindist_eval_t(metad_ctx *c, double *d_cv, int md) {
    typedef typename Vec4<T>::type V4;
    const CvDev &d = c->cv[md];
    const int nb = div_up(c->N, CV_THREADS);
    double *pr = c->d_partials;
    long long *pk = reinterpret_cast<long long *>(c->d_partials + c->nblocks_atoms);
    int *ps = reinterpret_cast<int *>(c->d_partials + 2 * (size_t)c->nblocks_atoms);
    k_mindist_cv<T><<<nb, CV_THREADS, 0, c->stream>>>(c->N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm, ctx_pbox<T>(c), c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, d.fshift,
                                                     c->rc, pr, pk, ps, c->d_tickets + 0, c->d_mind + 8 * md, d_cv + md, c->dg);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
int mindist_eval(metad_ctx *c, double *d_cv) {
    if (!c->has_mindist) return METAD_OK;
    for (int md = 0; md < c->D; ++md) {
    if (c->cv[md].kind != METAD_CV_MINDIST) continue;
    if (!c->list_built) {                                       // lazy_neighbors: list-free scan of the few centres
        const CvDev &d = c->cv[md];
        const int nb = div_up(d.n_gb, CV_THREADS);
        double *pr = c->d_partials;
        long long *pk = reinterpret_cast<long long *>(c->d_partials + c->nblocks_atoms);
        if (c->prec == 32)
            k_mindist_brute<float><<<nb, CV_THREADS, 0, c->stream>>>(d.n_ga, d.d_ga, d.n_gb, d.d_gb, (const float *)ctx_last_pos(c), c->boxd,
                                                                     c->rc, pr, pk, c->d_tickets + 0, c->d_mind + 8 * md, d_cv + md, c->dg);
        else
            k_mindist_brute<double><<<nb, CV_THREADS, 0, c->stream>>>(d.n_ga, d.d_ga, d.n_gb, d.d_gb, (const double *)ctx_last_pos(c), c->boxd,
                                                                      c->rc, pr, pk, c->d_tickets + 0, c->d_mind + 8 * md, d_cv + md, c->dg);
        c->launches++;
        CUDA_TRY(cudaGetLastError());
        continue;
    }
    const int r = c->prec == 32 ? mindist_eval_t<float>(c, d_cv, md) : mindist_eval_t<double>(c, d_cv, md);
    if (r) return r;
    }
    return METAD_OK;
}
int mindist_forces(metad_ctx *c, const double *d_dVds, void *d_F) {
    if (!c->has_mindist) return METAD_OK;
    for (int md = 0; md < c->D; ++md) {
        if (c->cv[md].kind != METAD_CV_MINDIST) continue;
        if (c->prec == 32) k_mindist_force<float><<<1, 32, 0, c->stream>>>(c->d_mind + 8 * md, c->p.force_scale, d_dVds + md, (float *)d_F,
                                                                       c->p.want_virial ? c->d_virial : nullptr);
        else k_mindist_force<double><<<1, 32, 0, c->stream>>>(c->d_mind + 8 * md, c->p.force_scale, d_dVds + md, (double *)d_F,
                                                             c->p.want_virial ? c->d_virial : nullptr);
        c->launches++;
    }
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

// ------------------------------------------------------------------------------------------------
int chain_eval(metad_ctx *c, int dim, const void *d_pos_unused, double *d_cv);          // cv_chain.cu
int chain_forces(metad_ctx *c, const double *d_dVds, void *d_F);                         // cv_chain.cu

template <typename T>
static int cv_eval_t(metad_ctx *c, double *d_cv) {
    typedef typename Vec4<T>::type V4;
    const int N = c->N, nb = div_up(N, CV_THREADS);
    PBox<T> pb = ctx_pbox<T>(c);
    if (c->has_coord && c->tiled) {                          // the sum ran inside k_tile_build<2>
        int r = tiled_q6_pass1(c, d_cv);
        if (r) return r;
    } else for (int cd = 0; cd < c->D; ++cd) {               // every COORD dimension: its own pass over the list
        if (c->cv[cd].kind != METAD_CV_COORD) continue;
        const CvDev &d = c->cv[cd];
        if (N <= METAD_WARP_PER_ATOM_MAX)
            k_coord_cv_warp<T, 32><<<div_up((long long)N * 32, CV_THREADS), CV_THREADS, 0, c->stream>>>(
                N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, d.fshift, (T)(1.0 / d.r0), d.n, d.m, d.scale, c->d_partials_warp,
                c->d_tickets + 0, d_cv + cd, c->d_sticky, c->dg);
        else
        k_coord_cv<T><<<nb, CV_THREADS, 0, c->stream>>>(N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, d.fshift,
                                                       (T)(1.0 / d.r0), d.n, d.m, d.scale, c->d_partials,
                                                       c->d_tickets + 0, d_cv + cd, c->d_sticky, c->dg);
        c->launches++;
    }
    if (c->has_q6 && (c->tiled || c->tiled64)) {              // tiled64: the fp64 sums ran inside k_tile_build64
        int r = (c->tiled && c->skin_on) ? tiled_q6_pass1_skin(c, d_cv) : tiled_q6_pass1(c, d_cv);
        if (r) return r;
    } else if (c->has_q6) {
        double sm = c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0;
        double ss = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0;
        double qt = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_thresh : 0.0;
        double qw = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].q_width : 1.0;
        k_q6_pass1<T><<<nb, CV_THREADS, 0, c->stream>>>(N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, (T)qt,
                                                       (T)(1.0 / qw), (T *)c->d_rec, (T *)c->d_q6, sm, ss, c->q6_mean_dim,
                                                       c->q6_solid_dim, c->d_partials + c->nblocks_atoms, c->d_tickets + 1,
                                                       d_cv, c->d_sticky, c->dg);
        c->launches++;
    }
    return METAD_OK;
}

int cv_eval_all(metad_ctx *c, double *d_cv) {
    int rcode = c->prec == 32 ? cv_eval_t<float>(c, d_cv) : cv_eval_t<double>(c, d_cv);
    if (rcode) return rcode;
    for (int d = 0; d < c->D; ++d)
        if (c->cv[d].kind == METAD_CV_RGYR || c->cv[d].kind == METAD_CV_CONTACTS) {
            rcode = chain_eval(c, d, nullptr, d_cv);
            if (rcode) return rcode;
        }
    rcode = torsion_eval_all(c, d_cv);
    if (rcode) return rcode;
    rcode = mindist_eval(c, d_cv);
    if (rcode) return rcode;
    rcode = lattice_eval(c, d_cv);
    if (rcode) return rcode;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

template <typename T>
static int cv_forces_t(metad_ctx *c, const double *d_dVds, void *d_F) {
    typedef typename Vec4<T>::type V4;
    const int N = c->N, nb = div_up(N, CV_THREADS);
    PBox<T> pb = ctx_pbox<T>(c);
    if (c->has_coord && c->tiled) {
        int r = tiled_coord_force(c, d_dVds, d_F);
        if (r) return r;
    } else for (int cd = 0; cd < c->D; ++cd) {               // every COORD dimension adds its forces in turn (fixed order)
        if (c->cv[cd].kind != METAD_CV_COORD) continue;
        const CvDev &d = c->cv[cd];
        const VirArgs va = { c->d_vir_partials, c->d_tickets + 12, c->d_virial };
        if (c->p.want_virial)                                 // forces and virial in one thread-per-atom pass
            k_coord_force<T, true><<<nb, CV_THREADS, 0, c->stream>>>(N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm,
                                                                    pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, d.fshift, (T)(1.0 / d.r0), d.n, d.m, c->p.force_scale * d.scale,
                                                                    d_dVds + cd, (T *)d_F, va, c->dg);
        else if (N <= METAD_WARP_PER_ATOM_MAX)
            k_coord_force_warp<T, 32><<<div_up((long long)N * 32, CV_THREADS), CV_THREADS, 0, c->stream>>>(
                N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm, pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, d.fshift, (T)(1.0 / d.r0), d.n, d.m,
                c->p.force_scale * d.scale, d_dVds + cd, (T *)d_F, c->dg);
        else if (d.use_groups && N <= 8 * METAD_WARP_PER_ATOM_MAX)
            k_coord_force_warp<T, 8><<<div_up((long long)N * 8, CV_THREADS), CV_THREADS, 0, c->stream>>>(
                N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm, pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, d.fshift, (T)(1.0 / d.r0), d.n, d.m,
                c->p.force_scale * d.scale, d_dVds + cd, (T *)d_F, c->dg);
        else
            k_coord_force<T, false><<<nb, CV_THREADS, 0, c->stream>>>(N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm,
                                                                     pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0, d.fshift, (T)(1.0 / d.r0), d.n, d.m, c->p.force_scale * d.scale,
                                                                     d_dVds + cd, (T *)d_F, va, c->dg);
        c->launches++;
    }
    if (c->has_q6 && c->tiled) {
        int r = tiled_q6_force(c, d_dVds, d_F);
        if (r) return r;
    } else if (c->has_q6) {
        double sm = c->q6_mean_dim >= 0 ? c->cv[c->q6_mean_dim].scale : 0.0;
        double ss = c->q6_solid_dim >= 0 ? c->cv[c->q6_solid_dim].scale : 0.0;
        const VirArgs va = { c->d_vir_partials, c->d_tickets + 12, c->d_virial };
        if (c->p.want_virial)
            k_q6_force<T, true><<<nb, CV_THREADS, 0, c->stream>>>(N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm, pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0,
                                                                 (const T *)c->d_rec, (const T *)c->d_q6 + c->N, sm, ss, c->q6_mean_dim, c->q6_solid_dim,
                                                                 c->p.force_scale, d_dVds, (T *)d_F, va, c->dg);
        else
            k_q6_force<T, false><<<nb, CV_THREADS, 0, c->stream>>>(N, (const V4 *)c->d_spos, c->d_nl_count, c->d_nl, c->d_perm, pb, c->boxd, (T)c->rc2, c->skin_on ? c->rc2 : 0.0,
                                                                  (const T *)c->d_rec, (const T *)c->d_q6 + c->N, sm, ss, c->q6_mean_dim, c->q6_solid_dim,
                                                                  c->p.force_scale, d_dVds, (T *)d_F, va, c->dg);
        c->launches++;
    }
    return METAD_OK;
}

int cv_forces_all(metad_ctx *c, const double *d_dVds, void *d_F) {
    if (c->p.want_virial) CUDA_TRY(cudaMemsetAsync(c->d_virial, 0, sizeof(double) * 9, c->stream));
    int rcode = c->prec == 32 ? cv_forces_t<float>(c, d_dVds, d_F) : cv_forces_t<double>(c, d_dVds, d_F);
    if (rcode) return rcode;
    rcode = chain_forces(c, d_dVds, d_F);
    if (rcode) return rcode;
    rcode = torsion_forces(c, d_dVds, d_F);
    if (rcode) return rcode;
    rcode = mindist_forces(c, d_dVds, d_F);
    if (rcode) return rcode;
    rcode = lattice_forces(c, d_dVds);
    if (rcode) return rcode;
    rcode = chain_virial(c, d_dVds);
    if (rcode) return rcode;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int q6_export(metad_ctx *c, void *d_q6) {
    if (!c->has_q6) return METAD_ERR_STATE;
    int nb = div_up(c->N, 256);
    if (c->prec == 32) k_q6_export_arr<float><<<nb, 256, 0, c->stream>>>(c->N, c->d_perm, (const float *)c->d_q6, (float *)d_q6);
    else k_q6_export_arr<double><<<nb, 256, 0, c->stream>>>(c->N, c->d_perm, (const double *)c->d_q6, (double *)d_q6);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
