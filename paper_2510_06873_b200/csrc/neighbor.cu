// neighbor.cu — a1: cell-list neighbour build (BASELINE.json north_star).
//   k_bin            cell index per atom + histogram (int atomics give the in-cell slot)
//   k_scan_sums/k_scan_apply   exclusive scan of the histogram over cells (two launches)
//   k_scatter        counting-sort scatter of atom indices
//   k_cell_sort_gather  thread per atom: rank by original index inside the cell (run-to-run determinism,
//                    reading P), gathers positions into the cell-sorted Vec4 array (x, y, z, group flags)
//   k_build_list     per-atom candidate scan of the 27 neighbouring cells; canonical predicate
// Everything downstream works in "sorted space" (indices into the cell-sorted arrays), so that the
// gathers of the CV and force passes touch neighbouring memory.
#include <math.h>
#include "common.cuh"

#define SCAN_THREADS 512
#define SCAN_ITEMS 4
#define SCAN_TILE (SCAN_THREADS * SCAN_ITEMS)

template <typename T>
__global__ void k_bin(int N, const T *__restrict__ pos, CellGrid g, int *__restrict__ cell_of,
                      int *__restrict__ slot, int *__restrict__ cell_count, unsigned int *__restrict__ sticky,
                      const DevGeom *__restrict__ dg, const int *__restrict__ skin_flag, const int *__restrict__ step) {
    pdl_enter();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N || SKIN_SKIP(skin_flag, step)) return;
    if (dg) { g.inv[0] = dg->inv[0]; g.inv[1] = dg->inv[1]; g.inv[2] = dg->inv[2]; g.cx = dg->cx; g.cy = dg->cy; g.bx = dg->bx; }
    double x = (double)pos[3 * i], y = (double)pos[3 * i + 1], z = (double)pos[3 * i + 2];
    double sc = z * g.inv[2];
    double sb = (y - sc * g.cy) * g.inv[1];
    double sa = (x - sb * g.bx - sc * g.cx) * g.inv[0];
    // Positions must lie in the primary cell (include/metad.h).  A coordinate that rounds to the far face (fractional
    // 1.0 + eps, e.g. after fp32 rounding) is CLAMPED into the boundary cell, not wrapped: its cartesian coordinates are
    // next to that cell's atoms, which is what the lattice-shift logic of the tiled path relies on.
    if (!(fabs(sa - 0.5) <= 0.5001) || !(fabs(sb - 0.5) <= 0.5001) || !(fabs(sc - 0.5) <= 0.5001))   // also catches NaN
        atomicOr(sticky, (unsigned)METAD_DEV_POS_RANGE);
    if (g.wlen < 1.0) {              // slab-decomposition rank: only the tiles of its window are launched (params.c_window_lo)
        double u = sc - g.wlo;
        u -= floor(u);
        if (!(u < g.wlen)) atomicOr(sticky, (unsigned)METAD_DEV_POS_RANGE);
    }
    int ia = min(max((int)floor(sa * g.nc[0]), 0), g.nc[0] - 1);
    int ib = min(max((int)floor(sb * g.nc[1]), 0), g.nc[1] - 1);
    int ic = min(max((int)floor(sc * g.nc[2]), 0), g.nc[2] - 1);
    int c = (ic * g.nc[1] + ib) * g.nc[0] + ia;
    cell_of[i] = c;
    slot[i] = atomicAdd(&cell_count[c], 1);
}

__global__ void k_scan_sums(int ncell, const int *__restrict__ cell_count, int *__restrict__ block_sums,
                            const int *__restrict__ skin_flag, const int *__restrict__ step) {
    __shared__ int ws[32];
    pdl_enter();
    if (SKIN_SKIP(skin_flag, step)) return;
    int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) s += (base + k < ncell) ? cell_count[base + k] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        int v = threadIdx.x < SCAN_THREADS / 32 ? ws[threadIdx.x] : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) block_sums[blockIdx.x] = v;
    }
}

// exclusive scan; also zeroes the histogram for the next step and writes cell_start[ncell] = N
__global__ void k_scan_apply(int ncell, int N, int *__restrict__ cell_count, const int *__restrict__ block_sums,
                             int *__restrict__ cell_start, const int *__restrict__ skin_flag, const int *__restrict__ step) {
    __shared__ int ws[32];
    __shared__ int s_prefix;
    pdl_enter();
    if (SKIN_SKIP(skin_flag, step)) return;
    // prefix of the preceding blocks' sums
    int pre = 0;
    for (int b = threadIdx.x; b < (int)blockIdx.x; b += blockDim.x) pre += block_sums[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) pre += __shfl_down_sync(0xffffffffu, pre, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = pre;
    __syncthreads();
    if (threadIdx.x < 32) {
        int v = threadIdx.x < SCAN_THREADS / 32 ? ws[threadIdx.x] : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) s_prefix = v;
    }
    __syncthreads();
    int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS], tsum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < ncell) ? cell_count[base + k] : 0;
        tsum += v[k];
    }
    // inclusive warp scan of thread sums
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int inc = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();
    if (lane == 31) ws[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int w = lane < SCAN_THREADS / 32 ? ws[lane] : 0;
        int winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        ws[lane] = winc - w;  // exclusive warp offsets
    }
    __syncthreads();
    int run = s_prefix + ws[wid] + (inc - tsum);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < ncell) {
            cell_start[base + k] = run;
            cell_count[base + k] = 0;
            run += v[k];
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) cell_start[ncell] = N;
}

// counting-sort scatter: slot a of the raw order receives (atom index, cell) in ONE 8-byte store, so that the ordering pass
// reads its cell from contiguous memory instead of gathering cell_of[i]
__global__ void k_scatter(int N, const int *__restrict__ cell_of, const int *__restrict__ slot,
                          const int *__restrict__ cell_start, int2 *__restrict__ perm,
                          const int *__restrict__ skin_flag, const int *__restrict__ step) {
    pdl_enter();
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N || SKIN_SKIP(skin_flag, step)) return;
    const int c = cell_of[i];
    perm[cell_start[c] + slot[i]] = make_int2(i, c);
}

// Thread per sorted slot: the atom in slot a finds its rank by original index among the atoms of its cell (a handful,
// read from the unsorted permutation through L1) and moves itself to that place: in-cell order = original index, so the
// float summation order downstream is run-to-run deterministic (reading P) no matter how the atomics of k_bin fell.
template <typename T>
__global__ void k_cell_sort_gather(int N, const int *__restrict__ cell_start,
                                   const int2 *__restrict__ perm_in /* (atom, cell) in raw order */, int *__restrict__ perm,
                                   const T *__restrict__ pos, const unsigned char *__restrict__ flags,
                                   typename Vec4<T>::type *__restrict__ spos, int *__restrict__ scell, int index_in_w,
                                   typename Vec4<T>::type *__restrict__ ref /* skin: positions at the build, else NULL */,
                                   const int *__restrict__ skin_flag, const int *__restrict__ step, int *__restrict__ nbuilds) {
    pdl_enter();
    int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= N || SKIN_SKIP(skin_flag, step)) return;
    if (a == 0 && nbuilds) ++*nbuilds;            // list builds so far (metad_get_rebuilds)
    const int2 ic = perm_in[a];
    const int i = ic.x, c = ic.y;
    const int b = cell_start[c], e = cell_start[c + 1];
    int rank = 0;
    for (int q = b; q < e; ++q) rank += perm_in[q].x < i;
    typename Vec4<T>::type v;
    v.x = pos[3 * i]; v.y = pos[3 * i + 1]; v.z = pos[3 * i + 2];
    v.w = (T)(flags ? (int)flags[i] : 3);
    const int d = b + rank;
    // tiled fp32 contexts have no group flags: .w carries (sorted index | no-shift code << 27), the neighbour-list entry of
    // this atom, so that interior tiles can be staged by raw bulk copies (tile.cuh)
    if (index_in_w && sizeof(T) == 4) v.w = (T)__int_as_float(d | (13 << 27));
    perm[d] = i;
    spos[d] = v;
    if (ref) ref[d] = v;
    scell[d] = c;
}

// fp64 contexts on a grid with >= 3 cells per direction take the per-run form of the predicate (common.cuh: r2_shifted)
template <typename T>
__device__ __forceinline__ bool pair_in_run(bool shifted, const RunShift &w, const PBox<T> &pb, const BoxD &bd, T rc2T, double rc2,
                                            const typename Vec4<T>::type &pi, const typename Vec4<T>::type &pj) {
    if (sizeof(T) == 8 && shifted)
        return r2_shifted(w, (double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y, (double)pj.z - (double)pi.z) < rc2;
    return pair_in_range<T>(pb, bd, rc2T, rc2, pi, pj);
}

template <typename T>
__global__ void __launch_bounds__(128)
k_build_list(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ scell,
             const int *__restrict__ cell_start, CellGrid g, PBox<T> pb, BoxD bd, T rc2T, double rc2, int maxn,
             int *__restrict__ nl_count, int *__restrict__ nl, unsigned int *__restrict__ sticky,
             const DevGeom *__restrict__ dg, const int *__restrict__ skin_flag, const int *__restrict__ step) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N || SKIN_SKIP(skin_flag, step)) return;
    if (dg) { pb = dg_pb<T>(dg); bd = dg->bd; }
    typename Vec4<T>::type pi = spos[s];
    int c = scell[s];
    int ia = c % g.nc[0], t = c / g.nc[0];
    int ib = t % g.nc[1], ic = t / g.nc[1];
    // offsets visited along a direction: all distinct cells among {-1,0,+1}
    int za0 = g.nc[0] >= 3 ? -1 : 0, za1 = g.nc[0] >= 2 ? 1 : 0;
    int zb0 = g.nc[1] >= 3 ? -1 : 0, zb1 = g.nc[1] >= 2 ? 1 : 0;
    int zc0 = g.nc[2] >= 3 ? -1 : 0, zc1 = g.nc[2] >= 2 ? 1 : 0;
    int cnt = 0;
    const bool shifted = sizeof(T) == 8 && g.nc[0] >= 3 && g.nc[1] >= 3 && g.nc[2] >= 3;
    RunShift w = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
    for (int oc = zc0; oc <= zc1; ++oc) {
        int jc = ic + oc;
        const double wz = jc < 0 ? -1.0 : (jc >= g.nc[2] ? 1.0 : 0.0);
        jc += jc < 0 ? g.nc[2] : 0; jc -= jc >= g.nc[2] ? g.nc[2] : 0;
        w.zx = wz * bd.cx; w.zy = wz * bd.cy; w.zz = wz * bd.cz;
        for (int ob = zb0; ob <= zb1; ++ob) {
            int jb = ib + ob;
            const double wy = jb < 0 ? -1.0 : (jb >= g.nc[1] ? 1.0 : 0.0);
            jb += jb < 0 ? g.nc[1] : 0; jb -= jb >= g.nc[1] ? g.nc[1] : 0;
            w.yx = wy * bd.bx; w.yy = wy * bd.by;
            int rowbase = (jc * g.nc[1] + jb) * g.nc[0];
            for (int oa = za0; oa <= za1; ++oa) {
                int ja = ia + oa;
                w.xx = ja < 0 ? -bd.ax : (ja >= g.nc[0] ? bd.ax : 0.0);
                ja += ja < 0 ? g.nc[0] : 0; ja -= ja >= g.nc[0] ? g.nc[0] : 0;
                int cb = cell_start[rowbase + ja], ce = cell_start[rowbase + ja + 1];
                for (int j = cb; j < ce; ++j) {
                    typename Vec4<T>::type pj = ldg4<T>(spos + j);
                    if (j != s && pair_in_run<T>(shifted, w, pb, bd, rc2T, rc2, pi, pj)) {
                        if (cnt < maxn) nl[(size_t)cnt * N + s] = j;
                        ++cnt;
                    }
                }
            }
        }
    }
    if (cnt > maxn) { atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW); cnt = maxn; }
    nl_count[s] = cnt;
}

// Warp per atom (systems too small to fill the GPU with one thread per atom: BASELINE.json configs[0]-[2]): the lanes
// share the candidates of each run of cells, a ballot keeps the accepted ones in candidate order (deterministic list).
// A row's three cells are one contiguous run of the cell-sorted order unless the row wraps in x.
template <typename T, int G>
__global__ void __launch_bounds__(128)
k_build_list_warp(int N, const typename Vec4<T>::type *__restrict__ spos, const int *__restrict__ scell,
                  const int *__restrict__ cell_start, CellGrid g, PBox<T> pb, BoxD bd, T rc2T, double rc2, int maxn,
                  int *__restrict__ nl_count, int *__restrict__ nl, unsigned int *__restrict__ sticky,
                  const DevGeom *__restrict__ dg, const int *__restrict__ skin_flag, const int *__restrict__ step) {
    // G lanes per atom (G = 32: one warp per atom; G = 8: four atoms per warp, each group votes under its own mask)
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int s = gt / G, lane = gt % G;
    if (s >= N || SKIN_SKIP(skin_flag, step)) return;
    if (dg) { pb = dg_pb<T>(dg); bd = dg->bd; }
    const unsigned gmask = G == 32 ? 0xffffffffu : (((1u << G) - 1u) << ((threadIdx.x & 31) / G * G));
    const int gshift = (threadIdx.x & 31) / G * G;
    const typename Vec4<T>::type pi = spos[s];
    const int c = scell[s];
    const int ia = c % g.nc[0], t = c / g.nc[0];
    const int ib = t % g.nc[1], ic = t / g.nc[1];
    const int zb0 = g.nc[1] >= 3 ? -1 : 0, zb1 = g.nc[1] >= 2 ? 1 : 0;
    const int zc0 = g.nc[2] >= 3 ? -1 : 0, zc1 = g.nc[2] >= 2 ? 1 : 0;
    // runs along x: [first cell, last cell] pairs, in the visiting order of the thread-per-atom kernel (-1, 0, +1)
    int ra[3], rb[3], nr = 0;
    double rsx[3] = { 0.0, 0.0, 0.0 };                     // lattice shift along a of each run (per-run predicate, fp64)
    if (g.nc[0] >= 3) {
        if (ia == 0) { rsx[nr] = -bd.ax; ra[nr] = g.nc[0] - 1; rb[nr++] = g.nc[0] - 1; ra[nr] = 0; rb[nr++] = 1; }
        else if (ia == g.nc[0] - 1) { ra[nr] = ia - 1; rb[nr++] = ia; rsx[nr] = bd.ax; ra[nr] = 0; rb[nr++] = 0; }
        else { ra[nr] = ia - 1; rb[nr++] = ia + 1; }
    } else if (g.nc[0] == 2) { ra[nr] = ia; rb[nr++] = ia; ra[nr] = 1 - ia; rb[nr++] = 1 - ia; }
    else { ra[nr] = 0; rb[nr++] = 0; }
    int cnt = 0;
    const bool shifted = sizeof(T) == 8 && g.nc[0] >= 3 && g.nc[1] >= 3 && g.nc[2] >= 3;
    RunShift w = { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 };
    for (int oc = zc0; oc <= zc1; ++oc) {
        int jc = ic + oc;
        const double wz = jc < 0 ? -1.0 : (jc >= g.nc[2] ? 1.0 : 0.0);
        jc += jc < 0 ? g.nc[2] : 0; jc -= jc >= g.nc[2] ? g.nc[2] : 0;
        w.zx = wz * bd.cx; w.zy = wz * bd.cy; w.zz = wz * bd.cz;
        for (int ob = zb0; ob <= zb1; ++ob) {
            int jb = ib + ob;
            const double wy = jb < 0 ? -1.0 : (jb >= g.nc[1] ? 1.0 : 0.0);
            jb += jb < 0 ? g.nc[1] : 0; jb -= jb >= g.nc[1] ? g.nc[1] : 0;
            w.yx = wy * bd.bx; w.yy = wy * bd.by;
            const int rowbase = (jc * g.nc[1] + jb) * g.nc[0];
            for (int r = 0; r < nr; ++r) {
                const int cb = cell_start[rowbase + ra[r]], ce = cell_start[rowbase + rb[r] + 1];
                w.xx = rsx[r];
                for (int j0 = cb; j0 < ce; j0 += G) {
                    const int j = j0 + lane;
                    bool hit = false;
                    if (j < ce && j != s) hit = pair_in_run<T>(shifted, w, pb, bd, rc2T, rc2, pi, ldg4<T>(spos + j));
                    const unsigned m = (__ballot_sync(gmask, hit) & gmask) >> gshift;
                    if (hit) {
                        const int k = cnt + __popc(m & ((1u << lane) - 1u));
                        if (k < maxn) nl[(size_t)k * N + s] = j;
                    }
                    cnt += __popc(m);
                }
            }
        }
    }
    if (lane == 0) {
        if (cnt > maxn) { atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW); cnt = maxn; }
        nl_count[s] = cnt;
    }
}

// Systems of at most METAD_SMALL_N atoms: no cells at all.  One warp per atom tests every other atom with the canonical
// predicate (N^2 / 32 tests per lane), the ballot keeps ascending j; the kernel also writes the identity "sort" (spos = the
// positions in their original order, perm = identity), so that the whole of a1 is ONE launch instead of six.
template <typename T>
__global__ void __launch_bounds__(128)
k_build_list_small(int N, const T *__restrict__ pos, const unsigned char *__restrict__ flags,
                   typename Vec4<T>::type *__restrict__ spos, int *__restrict__ perm, int *__restrict__ scell,
                   PBox<T> pb, BoxD bd, T rc2T, double rc2, int maxn, int *__restrict__ nl_count, int *__restrict__ nl,
                   CellGrid g, unsigned int *__restrict__ sticky, const DevGeom *__restrict__ dg,
                   typename Vec4<T>::type *__restrict__ ref, const int *__restrict__ skin_flag, const int *__restrict__ step,
                   int *__restrict__ nbuilds) {
    const int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (s >= N || SKIN_SKIP(skin_flag, step)) return;
    if (dg) {
        pb = dg_pb<T>(dg); bd = dg->bd;
        g.inv[0] = dg->inv[0]; g.inv[1] = dg->inv[1]; g.inv[2] = dg->inv[2]; g.cx = dg->cx; g.cy = dg->cy; g.bx = dg->bx;
    }
    typename Vec4<T>::type pi;
    pi.x = pos[3 * s]; pi.y = pos[3 * s + 1]; pi.z = pos[3 * s + 2];
    pi.w = (T)(flags ? (int)flags[s] : 3);
    if (lane == 0) {
        spos[s] = pi; perm[s] = s; scell[s] = 0;
        if (ref) ref[s] = pi;
        if (s == 0 && nbuilds) ++*nbuilds;
        // positions must lie in the primary cell (same check as k_bin)
        const double sc = (double)pi.z * g.inv[2], sb = ((double)pi.y - sc * g.cy) * g.inv[1],
                     sa = ((double)pi.x - sb * g.bx - sc * g.cx) * g.inv[0];
        if (!(fabs(sa - 0.5) <= 0.5001) || !(fabs(sb - 0.5) <= 0.5001) || !(fabs(sc - 0.5) <= 0.5001))
            atomicOr(sticky, (unsigned)METAD_DEV_POS_RANGE);
    }
    int cnt = 0;
    for (int j0 = 0; j0 < N; j0 += 32) {
        const int j = j0 + lane;
        bool hit = false;
        if (j < N && j != s) {
            typename Vec4<T>::type pj;
            pj.x = pos[3 * j]; pj.y = pos[3 * j + 1]; pj.z = pos[3 * j + 2]; pj.w = T(0);
            hit = pair_in_range<T>(pb, bd, rc2T, rc2, pi, pj);
        }
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (hit) {
            const int k = cnt + __popc(m & ((1u << lane) - 1u));
            if (k < maxn) nl[(size_t)k * N + s] = j;
        }
        cnt += __popc(m);
    }
    if (lane == 0) {
        if (cnt > maxn) { atomicOr(sticky, (unsigned)METAD_DEV_NEIGH_OVERFLOW); cnt = maxn; }
        nl_count[s] = cnt;
    }
}

// metad_get_neighbors: the list in ORIGINAL atom indices.  With a skin the kept list reaches rc + skin; the export applies
// the canonical fp64 predicate (reading O) on the current cell-sorted coordinates, so the caller sees the exact rc list.
// sliced: layout of the tiled path ([N/32][maxn][32], entries carry a shift code) or of the generic path (nl[k N + s]).
template <typename T>
__global__ void k_export_list(int N, int maxn, const int *__restrict__ perm, const int *__restrict__ nl_count,
                              const int *__restrict__ nl, int *__restrict__ out_count, int *__restrict__ out_list, int sliced,
                              const typename Vec4<T>::type *__restrict__ spos, BoxD bd, double rc2, int skin,
                              const DevGeom *__restrict__ dg) {
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    if (dg) bd = dg->bd;
    const int i = perm[s], cnt = nl_count[s];
    const typename Vec4<T>::type pi = spos[s];
    int n = 0;
    for (int k = 0; k < cnt; ++k) {
        const int j = sliced ? (nl[((size_t)(s >> 5) * maxn + k) * 32 + (s & 31)] & ((1 << 27) - 1)) : nl[(size_t)k * N + s];
        if (skin) {
            const typename Vec4<T>::type pj = spos[j];
            if (!(r2_canonical(bd, (double)pj.x - (double)pi.x, (double)pj.y - (double)pi.y, (double)pj.z - (double)pi.z) < rc2)) continue;
        }
        out_list[(size_t)i * maxn + n++] = perm[j];
    }
    out_count[i] = n;
    for (int k = n; k < maxn; ++k) out_list[(size_t)i * maxn + k] = -1;
}

template <typename T>
static PBox<T> make_pbox(const BoxD &b, double rc);
template <>
PBox<double> make_pbox<double>(const BoxD &b, double) {
    PBox<double> p = { b.ax, b.bx, b.by, b.cx, b.cy, b.cz, 0, 0, 0, 0, 0, 0, b.hx, b.hy, b.hz, 0.0 };
    return p;
}
template <>
PBox<float> make_pbox<float>(const BoxD &b, double rc) {
    PBox<float> p;
    const double v[6] = { b.ax, b.bx, b.by, b.cx, b.cy, b.cz };
    float hi[6], lo[6];
    for (int k = 0; k < 6; ++k) { hi[k] = (float)v[k]; lo[k] = (float)(v[k] - (double)hi[k]); }
    p.ax = hi[0]; p.bx = hi[1]; p.by = hi[2]; p.cx = hi[3]; p.cy = hi[4]; p.cz = hi[5];
    p.lax = lo[0]; p.lbx = lo[1]; p.lby = lo[2]; p.lcx = lo[3]; p.lcy = lo[4]; p.lcz = lo[5];
    p.hx = (float)b.hx; p.hy = (float)b.hy; p.hz = (float)b.hz;
    // Recheck band of the fp32 fast test.  Inside the primary cell pj - pi is exact only while the two coordinates are within
    // a factor 2 of one another; across a periodic face the raw difference is of the order of the box and is rounded at
    // ulp_f32(L) / 2 per component before the (hi + lo) lattice shift restores the small vector, so r^2 carries up to
    // 2 sum_c |d_c| ulp(L) / 2 <= sqrt(3) rc ulp(L) on top of the ~4 ulp(rc^2) of the three products.  The band must cover
    // both: max(1e-5 rc^2, 4 rc ulp_f32(L)) with L the largest coordinate a position can take.
    const double L = fmax(fabs(b.ax) + fabs(b.bx) + fabs(b.cx), fmax(fabs(b.by) + fabs(b.cy), fabs(b.cz)));
    const double ulpL = ldexp(1.0, ilogb(fmax(L, 1e-30)) - 23);
    p.band = (float)fmax(1e-5 * rc * rc, 4.0 * rc * ulpL);
    return p;
}
template <typename T> PBox<T> ctx_pbox(const metad_ctx *c) { return make_pbox<T>(c->boxd, c->rc); }
template PBox<float> ctx_pbox<float>(const metad_ctx *);
template PBox<double> ctx_pbox<double>(const metad_ctx *);

// Device-resident box (NEXT-3, PAPER.md:51 NPT): derives everything the kernels need from the 9 box doubles in device memory
// and checks what setup_geometry checks on the host for a host box — here a violation sets the sticky bit METAD_DEV_BOX (the
// step then runs with defined but meaningless neighbour sets).  nc: cell counts frozen at capture (x in sub-cells).
__global__ void k_geom_update(const double *__restrict__ box, double rc, int nc0, int nc1, int nc2, int xsub, float band_rel,
                              DevGeom *__restrict__ out, unsigned int *__restrict__ sticky) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const double ax = box[0], bx = box[3], by = box[4], cx = box[6], cy = box[7], cz = box[8];
    bool ok = box[1] == 0.0 && box[2] == 0.0 && box[5] == 0.0 && ax > 0.0 && by > 0.0 && cz > 0.0;
    const double vol = ax * by * cz;
    const double bxc[3] = { by * cz, -bx * cz, bx * cy - by * cx };
    const double cxa[3] = { 0.0, cz * ax, -cy * ax };
    double w[3];
    w[0] = vol / sqrt(bxc[0] * bxc[0] + bxc[1] * bxc[1] + bxc[2] * bxc[2]);
    w[1] = vol / sqrt(cxa[1] * cxa[1] + cxa[2] * cxa[2]);
    w[2] = cz;
    const int nc[3] = { nc0, nc1, nc2 };
    for (int d = 0; d < 3; ++d) {
        if (!(rc < 0.5 * w[d])) ok = false;
        const int full = d == 0 ? nc[d] / xsub : nc[d];                 // rc-wide cells along this direction
        if (full > 1 && !(w[d] / full >= rc)) ok = false;               // a cell narrower than rc would miss neighbours
    }
    if (!ok) atomicOr(sticky, (unsigned)METAD_DEV_BOX);
    BoxD b = { ax, bx, by, cx, cy, cz, 0.5 * ax, 0.5 * by, 0.5 * cz };
    out->bd = b;
    PBox<double> pd = { ax, bx, by, cx, cy, cz, 0, 0, 0, 0, 0, 0, b.hx, b.hy, b.hz, 0.0 };
    out->pbd = pd;
    PBox<float> pf;
    const double v[6] = { ax, bx, by, cx, cy, cz };
    float hi[6], lo[6];
    for (int k = 0; k < 6; ++k) { hi[k] = (float)v[k]; lo[k] = (float)(v[k] - (double)hi[k]); }
    pf.ax = hi[0]; pf.bx = hi[1]; pf.by = hi[2]; pf.cx = hi[3]; pf.cy = hi[4]; pf.cz = hi[5];
    pf.lax = lo[0]; pf.lbx = lo[1]; pf.lby = lo[2]; pf.lcx = lo[3]; pf.lcy = lo[4]; pf.lcz = lo[5];
    pf.hx = (float)b.hx; pf.hy = (float)b.hy; pf.hz = (float)b.hz;
    const double L = fmax(fabs(ax) + fabs(bx) + fabs(cx), fmax(fabs(by) + fabs(cy), fabs(cz)));
    const double ulpL = ldexp(1.0, ilogb(fmax(L, 1e-30)) - 23);
    pf.band = (float)fmax((double)band_rel * rc * rc, 4.0 * rc * ulpL);      // as make_pbox<float>
    out->pbf = pf;
    out->inv[0] = 1.0 / ax; out->inv[1] = 1.0 / by; out->inv[2] = 1.0 / cz;
    out->inv[3] = out->inv[4] = out->inv[5] = 0.0;
    out->cx = cx; out->cy = cy; out->bx = bx;
    for (int k = 0; k < 9; ++k) out->box[k] = box[k];
}

int geom_update(metad_ctx *c, const double *d_box) {
    k_geom_update<<<1, 32, 0, c->stream>>>(d_box, c->rc, c->grid.nc[0], c->grid.nc[1], c->grid.nc[2], (c->tiled || c->tiled64) ? c->tile_hx : 1,
                                           1e-5f, c->d_geom, c->d_sticky);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

// Verlet-skin reuse (params.skin).  Every step, before the build kernels: has any atom moved more
// than skin / 2 (minimum-image displacement in fp64) from where it was when the list was built?  Then the step's rebuild flag
// is raised and the build kernels that follow in the stream (or in the captured graph) do their work; otherwise they return
// at once and the step works on the kept list, whose cell-sorted positions this kernel refreshes (same slots, current
// coordinates).  The two flags alternate with the parity of the device step counter: the kernel clears the flag of the NEXT
// step, so no memset node is needed and the decision never leaves the device.
template <typename T>
__global__ void k_skin_check(int N, const T *__restrict__ pos, const int *__restrict__ perm,
                             const typename Vec4<T>::type *__restrict__ ref, typename Vec4<T>::type *__restrict__ spos, BoxD bd,
                             double half_skin2, int *__restrict__ skin_flag, const int *__restrict__ step,
                             const DevGeom *__restrict__ dg, cudaGraphConditionalHandle cond, int use_cond) {
    const int cur = *step & 1;
    if (blockIdx.x == 0 && threadIdx.x == 0) skin_flag[cur ^ 1] = 0;
    if (skin_flag[cur]) {                         // already decided (first step, new geometry): perm / ref are about to be rebuilt
        if (use_cond && blockIdx.x == 0 && threadIdx.x == 0) cudaGraphSetConditional(cond, 1);
        return;
    }
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    bool moved = false;
    if (s < N) {
        if (dg) bd = dg->bd;
        const int i = perm[s];
        typename Vec4<T>::type r = ref[s], v;
        v.x = pos[3 * i]; v.y = pos[3 * i + 1]; v.z = pos[3 * i + 2]; v.w = r.w;
        double dx = (double)v.x - (double)r.x, dy = (double)v.y - (double)r.y, dz = (double)v.z - (double)r.z;
        min_image_d(bd, dx, dy, dz);
        moved = !(dx * dx + dy * dy + dz * dz <= half_skin2);       // also catches NaN
        spos[s] = v;
    }
    if (__any_sync(0xffffffffu, moved) && (threadIdx.x & 31) == 0) {
        atomicOr(&skin_flag[cur], 1);
        // inside a captured graph the build kernels are the body of a conditional IF node (default: skipped): switch it on
        if (use_cond) cudaGraphSetConditional(cond, 1);
    }
}

static int skin_check_launch(metad_ctx *c, const void *d_pos, cudaGraphConditionalHandle cond, int use_cond) {
    const double h2 = 0.25 * c->p.skin * c->p.skin;
    if (c->prec == 32)
        k_skin_check<float><<<div_up(c->N, 256), 256, 0, c->stream>>>(c->N, (const float *)d_pos, c->d_perm, (const float4 *)c->d_ref,
                                                                      (float4 *)c->d_spos, c->boxd, h2, c->d_skin_flag, c->d_step, c->dg,
                                                                      cond, use_cond);
    else
        k_skin_check<double><<<div_up(c->N, 256), 256, 0, c->stream>>>(c->N, (const double *)d_pos, c->d_perm, (const double4 *)c->d_ref,
                                                                       (double4 *)c->d_spos, c->boxd, h2, c->d_skin_flag, c->d_step, c->dg,
                                                                       cond, use_cond);
    c->launches++;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

template <typename T> static int nb_build_kernels(metad_ctx *c, const void *d_pos);

// With a skin, inside a stream capture (metad_run), the build kernels become the body of a conditional IF node that
// k_skin_check switches on from the device (cudaGraphSetConditional): a step that keeps its list launches none of them.
// Outside a capture (stage calls) the kernels are launched and return at once when the flag is clear.
template <typename T>
static int nb_build_t(metad_ctx *c, const void *d_pos) {
    const bool tm = c->timing && !c->capturing;
    if (tm) { cudaEventRecord(c->ev[0], c->stream); c->timing_recorded = 1; }
    if (!c->skin_on) return nb_build_kernels<T>(c, d_pos);
    if (!c->capturing) {
        int r = skin_check_launch(c, d_pos, 0, 0);
        return r ? r : nb_build_kernels<T>(c, d_pos);
    }
    cudaStream_t st = c->stream;
    cudaStreamCaptureStatus status;
    unsigned long long id;
    cudaGraph_t graph;
    const cudaGraphNode_t *deps;
    size_t ndeps;
    CUDA_TRY(cudaStreamGetCaptureInfo(st, &status, &id, &graph, &deps, &ndeps));
    cudaGraphConditionalHandle cond;
    CUDA_TRY(cudaGraphConditionalHandleCreate(&cond, graph, 0, cudaGraphCondAssignDefault));
    int r = skin_check_launch(c, d_pos, cond, 1);
    if (r) return r;
    CUDA_TRY(cudaStreamGetCaptureInfo(st, &status, &id, &graph, &deps, &ndeps));      // now: the check kernel
    cudaGraphNodeParams np = {};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = cond;
    np.conditional.type = cudaGraphCondTypeIf;
    np.conditional.size = 1;
    cudaGraphNode_t cnode;
    CUDA_TRY(cudaGraphAddNode(&cnode, graph, deps, ndeps, &np));
    CUDA_TRY(cudaStreamBeginCaptureToGraph(c->copy_stream, np.conditional.phGraph_out[0], nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
    c->stream = c->copy_stream;                   // the build kernels are captured into the body graph
    r = nb_build_kernels<T>(c, d_pos);
    c->stream = st;
    cudaError_t e = cudaStreamEndCapture(c->copy_stream, nullptr);
    if (r) return r;
    CUDA_TRY(e);
    CUDA_TRY(cudaStreamUpdateCaptureDependencies(st, &cnode, 1, cudaStreamSetCaptureDependencies));
    return METAD_OK;
}

template <typename T>
static int nb_build_kernels(metad_ctx *c, const void *d_pos) {
    typedef typename Vec4<T>::type V4;
    const int N = c->N, ncell = c->grid.ncell;
    cudaStream_t st = c->stream;
    const int nsb = div_up(ncell, SCAN_TILE);
    const bool tm = c->timing && !c->capturing;
    const int *sf = c->skin_on ? c->d_skin_flag : nullptr, *stp = c->d_step;
    V4 *ref = c->skin_on ? (V4 *)c->d_ref : nullptr;
    if (N <= METAD_SMALL_N && !c->tiled && !c->tiled64) {                     // the whole neighbour stage in one launch
        if (tm) cudaEventRecord(c->ev[1], st);
        k_build_list_small<T><<<div_up((long long)N * 32, 128), 128, 0, st>>>(N, (const T *)d_pos, c->d_flags, (V4 *)c->d_spos, c->d_perm,
                                                                             c->d_scell, make_pbox<T>(c->boxd, c->rcl), c->boxd, (T)c->rcl2, c->rcl2,
                                                                             c->maxn, c->d_nl_count, c->d_nl, c->grid, c->d_sticky, c->dg, ref, sf, stp, c->d_nbuilds);
        if (tm) cudaEventRecord(c->ev[2], st);
        c->launches += 1;
        CUDA_TRY(cudaGetLastError());
        return METAD_OK;
    }
    // the kernels of the step chain are launched as programmatic dependents of one another (common.cuh: pdl_enter); not in skin
    // mode, where the build sits in the body of a conditional graph node
    const bool pdl = !c->skin_on;
    klaunch_pdl(pdl, k_bin<T>, div_up(N, 256), 256, 0, st, N, (const T *)d_pos, c->grid, c->d_cell_of, c->d_slot, c->d_cell_count,
                c->d_sticky, (const DevGeom *)c->dg, sf, stp);
    klaunch_pdl(pdl, k_scan_sums, nsb, SCAN_THREADS, 0, st, ncell, (const int *)c->d_cell_count, c->d_block_sums, sf, stp);
    klaunch_pdl(pdl, k_scan_apply, nsb, SCAN_THREADS, 0, st, ncell, N, c->d_cell_count, (const int *)c->d_block_sums, c->d_cell_start, sf, stp);
    klaunch_pdl(pdl, k_scatter, div_up(N, 256), 256, 0, st, N, (const int *)c->d_cell_of, (const int *)c->d_slot, (const int *)c->d_cell_start,
                (int2 *)c->d_perm_raw, sf, stp);
    klaunch_pdl(pdl, k_cell_sort_gather<T>, div_up(N, 256), 256, 0, st, N, (const int *)c->d_cell_start,
                (const int2 *)c->d_perm_raw, c->d_perm, (const T *)d_pos,
                (const unsigned char *)c->d_flags,   /* NULL unless a COORD / MINDIST CV has groups */
                (V4 *)c->d_spos, c->d_scell, c->tiled ? 1 : 0, ref, sf, stp, c->d_nbuilds);
    if (tm) cudaEventRecord(c->ev[1], st);
    if ((c->tiled && sizeof(T) == 4) || (c->tiled64 && sizeof(T) == 8)) {
        c->launches += 5;
        int r = sizeof(T) == 4 ? tiled_build(c) : tiled64_build(c);
        if (tm) cudaEventRecord(c->ev[2], st);
        return r;
    }
    PBox<T> pb = make_pbox<T>(c->boxd, c->rcl);
    if (N <= METAD_WARP_PER_ATOM_MAX)
        k_build_list_warp<T, 32><<<div_up((long long)N * 32, 128), 128, 0, st>>>(N, (const V4 *)c->d_spos, c->d_scell, c->d_cell_start,
                                                                                 c->grid, pb, c->boxd, (T)c->rcl2, c->rcl2, c->maxn,
                                                                                 c->d_nl_count, c->d_nl, c->d_sticky, c->dg, sf, stp);
    else if (N <= 8 * METAD_WARP_PER_ATOM_MAX)
        k_build_list_warp<T, 8><<<div_up((long long)N * 8, 128), 128, 0, st>>>(N, (const V4 *)c->d_spos, c->d_scell, c->d_cell_start,
                                                                               c->grid, pb, c->boxd, (T)c->rcl2, c->rcl2, c->maxn,
                                                                               c->d_nl_count, c->d_nl, c->d_sticky, c->dg, sf, stp);
    else
    k_build_list<T><<<div_up(N, 128), 128, 0, st>>>(N, (const V4 *)c->d_spos, c->d_scell, c->d_cell_start, c->grid, pb,
                                                   c->boxd, (T)c->rcl2, c->rcl2, c->maxn, c->d_nl_count, c->d_nl,
                                                   c->d_sticky, c->dg, sf, stp);
    if (tm) cudaEventRecord(c->ev[2], st);
    c->launches += 6;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}

int nb_build(metad_ctx *c, const void *d_pos) {
    return c->prec == 32 ? nb_build_t<float>(c, d_pos) : nb_build_t<double>(c, d_pos);
}

int nb_export(metad_ctx *c, int *d_count, int *d_list) {
    if (c->prec == 32)
        k_export_list<float><<<div_up(c->N, 128), 128, 0, c->stream>>>(c->N, c->maxn, c->d_perm, c->d_nl_count, c->d_nl, d_count, d_list,
                                                                       c->tiled, (const float4 *)c->d_spos, c->boxd, c->rc2, c->skin_on, c->dg);
    else
        k_export_list<double><<<div_up(c->N, 128), 128, 0, c->stream>>>(c->N, c->maxn, c->d_perm, c->d_nl_count, c->d_nl, d_count, d_list,
                                                                        0, (const double4 *)c->d_spos, c->boxd, c->rc2, c->skin_on, c->dg);
    c->launches += 1;
    CUDA_TRY(cudaGetLastError());
    return METAD_OK;
}
