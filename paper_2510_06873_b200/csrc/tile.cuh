// tile.cuh — shared-memory tiling of the cell grid (fp32 fast path).
//
// A thread block owns a tile of Tx x Ty x Tz cells (x counted in sub-cells: the rc-wide cells are split hx-fold along x).
// Its halo = the tile grown by hx sub-cells in x and one cell in y and z = (Ty+2)(Tz+2) "rows", each row a run of Tx+2hx
// sub-cells that is contiguous in the cell-sorted atom order (up to a periodic split into <= 3 pieces A|B|C with lattice
// shift -a|0|+a).  The halo atoms are numbered 0..total-1 in (row, piece, atom) order: the LOCAL index, used by the
// per-thread candidate lists in shared memory (uint16); the neighbour list written to global memory holds global sorted
// indices | lattice-shift code << 27.
//
// Positions are staged in tile-local coordinates  p - origin (+ lattice shift for periodic images):
// for atoms of the primary cell the subtraction is exact in fp32 (origin is the point of the tile's
// coordinate range nearest to 0, on a 2^-6 grid), periodic images are formed in fp64 and rounded
// once.  No per-pair minimum image is needed afterwards.
#pragma once
#include "common.cuh"

#define TILE_THREADS 256
#define TILE_MAXROWS 36          // (Ty+2)(Tz+2), Ty,Tz <= 4
#define TILE_TXMAX 30
#define TILE_HXMAX 4
#define TILE_NSEG (3 * TILE_MAXROWS)
#define TILE_MAXOWN 16           // Ty*Tz

struct TileGeom {
    int Tx, Ty, Tz;              // tile size in cells
    int hx;                      // halo width along x in cells (= the x-subdivision of the rc-wide cells, api.cu)
    int ntx, nty, ntz;           // tiles per direction
    int nc0, nc1, nc2;           // cells per direction
    int cap;                     // halo capacity (atoms) of the shared-memory staging area
    int cshift;                  // log2 of the power of two >= Tx + 2 hx + 1: a halo cell is (row, column) = (i >> cshift, i & mask)
    const int *cuts;             // device: tile boundaries along x [ntx + 1], y [nty + 1], z [ntz + 1] (api.cu: no division in the kernel)
    int natoms;                  // N (the second halves of the q6 records start at rec + 8 N)
    int sparse;                  // params.fill_fraction < 1: most tiles of the box hold no atom (tile_is_empty)
    int tz0, ntz_launch;         // z-tiles launched: tz0, tz0 + 1, ... (mod ntz), ntz_launch of them (all unless sparse)
    double ax, bx, by, cx, cy, cz;   // lattice rows
    double wa, wb, wc;           // cell edge vectors are a/nc0, b/nc1, c/nc2 (used for the tile's coordinate range)
};

// lattice rows of the step: from the device-resident geometry when the box lives in device memory (NPT), else the kernel
// argument (read at the few points of use: the kernel argument itself is never written, it stays in the constant bank)
struct TileBox { double ax, bx, by, cx, cy, cz; };
__device__ __forceinline__ TileBox tile_box(const TileGeom &g, const DevGeom *dg) {
    TileBox b;
    if (dg) { b.ax = dg->bd.ax; b.bx = dg->bd.bx; b.by = dg->bd.by; b.cx = dg->bd.cx; b.cy = dg->bd.cy; b.cz = dg->bd.cz; }
    else { b.ax = g.ax; b.bx = g.bx; b.by = g.by; b.cx = g.cx; b.cy = g.cy; b.cz = g.cz; }
    return b;
}

// A rank of a slab decomposition holds atoms in part of the GLOBAL box only (params.fill_fraction < 1):
// a tile none of whose own rows holds an atom skips set-up, staging and scan.  All threads of the block must call it.
__device__ __forceinline__ bool tile_is_empty(const TileGeom &g, const int *__restrict__ cell_start) {
    const int *cy = g.cuts + g.ntx + 1, *cz = cy + g.nty + 1;
    const int x0 = g.cuts[blockIdx.x], x1 = g.cuts[blockIdx.x + 1];
    int tz = blockIdx.z + g.tz0;
    if (tz >= g.ntz) tz -= g.ntz;
    const int y0 = cy[blockIdx.y], ny = cy[blockIdx.y + 1] - y0, z0 = cz[tz], nz = cz[tz + 1] - z0;
    int n = 0;
    if ((int)threadIdx.x < ny * nz) {                         // an own row = cells [x0, x1) of one (y, z): contiguous in the sort
        const int oz = (int)threadIdx.x / ny, oy = (int)threadIdx.x - oz * ny;
        const int base = ((z0 + oz) * g.nc1 + (y0 + oy)) * g.nc0;
        n = cell_start[base + x1] - cell_start[base + x0];
    }
    return __syncthreads_or(n) == 0;
}

struct TileTables {
    int seg_g[TILE_NSEG];        // global (sorted-space) index of the segment's first atom
    int seg_len[TILE_NSEG];
    int seg_off[TILE_NSEG + 1];  // local index of the segment's first atom
    unsigned char seg_wrapped[TILE_NSEG];
    unsigned char seg_code[TILE_NSEG];  // lattice-shift code (wx+1) + 3(wy+1) + 9(wz+1); 13 = no shift
    unsigned short hcell[TILE_MAXROWS][TILE_TXMAX + 2 * TILE_HXMAX + 1];   // local index where halo cell (row, lx) starts; [Txe+2] = row end
    int own_g[TILE_MAXOWN];      // global index of the first own atom of own-row q
    int own_l[TILE_MAXOWN];      // local index of the same atom
    int own_off[TILE_MAXOWN + 1];
    int own_row[TILE_MAXOWN];    // halo row id of own-row q
    float origin[3];
    int x0, y0, z0, Txe, Tye, Tze, nrows, nown, total, staged;
    int any_wrapped;             // some non-empty segment of the halo is a periodic image (boundary tile)
};

__device__ __forceinline__ int tile_row_id(const TileTables &t, int hy, int hz) {   // hy,hz in [-1, T*e]
    return (hz + 1) * (t.Tye + 2) + (hy + 1);
}

// Builds the tables (all threads of the block must call it).  cell_start: exclusive scan over cells.
// Four barrier-separated phases, none with a serial loop: every global load (two per halo cell) is issued in phase 1
// by a different thread, so the block pays the L2 latency once; the tile origin is worked out by 8 lanes in parallel.
// Tiles partition each direction evenly (tile k covers cells [k nc / nt, (k+1) nc / nt)), so no sliver tiles.
// scratch: >= TILE_SCRATCH_BYTES of shared memory that is free during the setup (the position staging area)
struct TileScratch {
    int hbeg[TILE_MAXROWS][TILE_TXMAX + 2 * TILE_HXMAX + 1];    // cell_start[cell]
    int hend[TILE_MAXROWS][TILE_TXMAX + 2 * TILE_HXMAX + 1];    // cell_start[cell + 1]
    int hrel[TILE_MAXROWS][TILE_TXMAX + 2 * TILE_HXMAX + 1];    // start of the halo cell relative to its segment | piece << 28
};
#define TILE_SCRATCH_BYTES sizeof(TileScratch)
// r / d and r % d for 0 <= r < 64, 3 <= d <= 6 (rows of a halo: d = Ty + 2) by a reciprocal multiplication instead of the
// ~20-instruction integer division
__device__ __forceinline__ int small_div(int r, int d) {
    const int magic = d == 3 ? 21846 : (d == 4 ? 16384 : (d == 5 ? 13108 : 10923));      // ceil(65536 / d)
    return (r * magic) >> 16;
}

__device__ __forceinline__ void tile_setup(const TileGeom &g, const int *__restrict__ cell_start, TileTables &t, TileScratch &w,
                                           const DevGeom *dg) {
    const int tid = threadIdx.x;
    // the launch grid is (ntx, nty, ntz) and the tile boundaries come from a table: no integer division on the way in
    const int tx = blockIdx.x, ty = blockIdx.y;
    int tz = blockIdx.z + g.tz0;                  // tz0 != 0 only on a slab-decomposition rank (its window of z-tiles)
    if (tz >= g.ntz) tz -= g.ntz;
    const int *cy = g.cuts + g.ntx + 1, *cz = cy + g.nty + 1;
    const int x0 = g.cuts[tx], y0 = cy[ty], z0 = cz[tz];
    const int Txe = g.cuts[tx + 1] - x0, Tye = cy[ty + 1] - y0, Tze = cz[tz + 1] - z0;
    const int hx = g.hx;
    const int nrows = (Tye + 2) * (Tze + 2), ncol = Txe + 2 * hx;
    const int xa = x0 - hx, xb = x0 + Txe + hx - 1;
    const int cmask = (1 << g.cshift) - 1, nslot = nrows << g.cshift;
    // ---- phase 1: cell_start of every halo cell (both ends); warp 7 fixes the tile origin
    for (int i = tid; i < nslot; i += blockDim.x) {
        const int r = i >> g.cshift, c = i & cmask;
        if (c >= ncol) continue;
        const int hz = small_div(r, Tye + 2) - 1, hy = r - (hz + 1) * (Tye + 2) - 1;
        const int ly = y0 + hy, lz = z0 + hz, lx = xa + c;
        const int jy = ly < 0 ? ly + g.nc1 : (ly >= g.nc1 ? ly - g.nc1 : ly);
        const int jz = lz < 0 ? lz + g.nc2 : (lz >= g.nc2 ? lz - g.nc2 : lz);
        const int jx = lx < 0 ? lx + g.nc0 : (lx >= g.nc0 ? lx - g.nc0 : lx);
        const int id = (jz * g.nc1 + jy) * g.nc0 + jx;
        w.hbeg[r][c] = cell_start[id];
        w.hend[r][c] = cell_start[id + 1];
    }
    if (tid == 0) { t.x0 = x0; t.y0 = y0; t.z0 = z0; t.Txe = Txe; t.Tye = Tye; t.Tze = Tze; t.nrows = nrows; t.any_wrapped = 0; }
    if (tid >= blockDim.x - 32) {
        // coordinate range of the halo'd tile (8 corners of the parallelepiped, one per lane), origin = point nearest to 0
        const int c = tid & 7;
        const double fa = (double)(x0 - hx + ((c & 1) ? Txe + 2 * hx : 0)) / g.nc0;
        const double fb = (double)(y0 - 1 + ((c & 2) ? Tye + 2 : 0)) / g.nc1;
        const double fc = (double)(z0 - 1 + ((c & 4) ? Tze + 2 : 0)) / g.nc2;
        const TileBox bx = tile_box(g, dg);
        double lo[3] = { fa * bx.ax + fb * bx.bx + fc * bx.cx, fb * bx.by + fc * bx.cy, fc * bx.cz }, hi[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            hi[a] = lo[a];
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                lo[a] = fmin(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
                hi[a] = fmax(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
            }
            const double o = lo[a] > 0.0 ? lo[a] : (hi[a] < 0.0 ? hi[a] : 0.0);
            if ((tid & 31) == 0) t.origin[a] = (float)(trunc(o * 64.0) * (1.0 / 64.0));   // toward zero, on a 2^-6 grid
        }
    }
    for (int s = 3 * nrows + tid; s < TILE_NSEG; s += blockDim.x) t.seg_len[s] = 0;
    __syncthreads();
    // ---- phase 2: the <= 3 segments of every row (thread per segment); halo-cell starts relative to their segment
    //      (thread per halo cell).  Piece p of a row covers halo columns [ls, le]: p = 0 left of x = 0 (shift -a),
    //      p = 1 inside the box, p = 2 right of x = nc0 - 1 (shift +a).
    if (tid < 3 * nrows) {
        const int r = tid / 3, p = tid - 3 * r;
        const int hz = small_div(r, Tye + 2) - 1, hy = r - (hz + 1) * (Tye + 2) - 1;
        const int ly = y0 + hy, lz = z0 + hz;
        const int wy = ly < 0 ? -1 : (ly >= g.nc1 ? 1 : 0), wz = lz < 0 ? -1 : (lz >= g.nc2 ? 1 : 0), wx = p - 1;
        const int ls = p == 0 ? xa : (p == 1 ? max(xa, 0) : max(xa, g.nc0));
        const int le = p == 0 ? min(xb, -1) : (p == 1 ? min(xb, g.nc0 - 1) : xb);
        if (ls <= le) { const int sg = w.hbeg[r][ls - xa]; t.seg_g[tid] = sg; t.seg_len[tid] = w.hend[r][le - xa] - sg; }
        else { t.seg_g[tid] = 0; t.seg_len[tid] = 0; }
        t.seg_wrapped[tid] = (wx | wy | wz) != 0;
        if ((wx | wy | wz) != 0 && ls <= le && t.seg_len[tid] > 0) t.any_wrapped = 1;      // benign race: every writer stores 1
        t.seg_code[tid] = (unsigned char)((wx + 1) + 3 * (wy + 1) + 9 * (wz + 1));
    }
    for (int i = tid; i < nslot; i += blockDim.x) {
        const int r = i >> g.cshift, c = i & cmask;
        if (c >= ncol) continue;
        const int lx = xa + c, p = lx < 0 ? 0 : (lx >= g.nc0 ? 2 : 1);
        const int ls = p == 0 ? xa : (p == 1 ? max(xa, 0) : max(xa, g.nc0));
        w.hrel[r][c] = (w.hbeg[r][c] - w.hbeg[r][ls - xa]) | (p << 28);
    }
    __syncthreads();
    // ---- phase 3: exclusive scan of seg_len (<= 108 entries) by warp 0
    if (tid < 32) {
        int base = tid * 4, v[4], sum = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) { v[k] = (base + k < TILE_NSEG) ? t.seg_len[base + k] : 0; sum += v[k]; }
        int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, inc, o); if (tid >= o) inc += u; }
        int run = inc - sum;
#pragma unroll
        for (int k = 0; k < 4; ++k) { if (base + k < TILE_NSEG) t.seg_off[base + k] = run; run += v[k]; }
        if (tid == 31) { t.seg_off[TILE_NSEG] = inc; t.total = inc; t.staged = inc <= g.cap; }
    }
    __syncthreads();
    // ---- phase 4: local halo-cell starts (thread per halo cell); own rows (last warp, lane per own row)
    for (int i = tid; i < nslot; i += blockDim.x) {
        const int r = i >> g.cshift, c = i & cmask;
        if (c > ncol) continue;
        if (c < ncol) {
            const int v = w.hrel[r][c];
            t.hcell[r][c] = (unsigned short)((v & 0xfffffff) + t.seg_off[3 * r + (v >> 28)]);
        } else {
            t.hcell[r][ncol] = (unsigned short)t.seg_off[3 * r + 3];      // end of the row = start of the next row's piece A
        }
    }
    if (tid >= blockDim.x - 32) {
        const int q = tid & 31, nq = Tye * Tze;
        int len = 0, l0 = 0, r = 0;
        if (q < nq) {
            const int oz = Tye == 1 ? q : (Tye == 2 ? q >> 1 : (Tye == 4 ? q >> 2 : small_div(q, 3))), oy = q - oz * Tye;
            r = (oz + 1) * (Tye + 2) + (oy + 1);
            // column hx (cell x0) always lies in piece 1; column Txe + hx (cell x0 + Txe) in piece 1 or, at the box end, 2
            const int v1 = w.hrel[r][Txe + hx];
            l0 = (w.hrel[r][hx] & 0xfffffff) + t.seg_off[3 * r + 1];
            len = (v1 & 0xfffffff) + t.seg_off[3 * r + (v1 >> 28)] - l0;
        }
        int inc = len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int u = __shfl_up_sync(0xffffffffu, inc, o); if (q >= o) inc += u; }
        if (q < nq) {
            t.own_row[q] = r; t.own_l[q] = l0;
            t.own_g[q] = t.seg_g[3 * r + 1] + (l0 - t.seg_off[3 * r + 1]);
            t.own_off[q] = inc - len;
        }
        const int n = __shfl_sync(0xffffffffu, inc, 31);
        if (q >= nq && q <= TILE_MAXOWN) t.own_off[q] = n;
        if (q == 0) t.nown = n;
    }
    __syncthreads();
}

// local index -> segment (binary search over seg_off; used by the unstaged slow path and the export)
__device__ __forceinline__ int tile_seg_of(const TileTables &t, int li) {
    int lo = 0, hi = 3 * t.nrows;        // seg_off[lo] <= li < seg_off[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (t.seg_off[mid] <= li) lo = mid; else hi = mid;
    }
    return lo;
}
__device__ __forceinline__ int tile_global_of(const TileTables &t, int li) {
    int s = tile_seg_of(t, li);
    return t.seg_g[s] + (li - t.seg_off[s]);
}

// neighbour-list entry of the tiled path: global sorted index | lattice-shift code << 27
#define NL_IDX_BITS 27
#define NL_IDX_MASK ((1 << NL_IDX_BITS) - 1)
#define NL_CODE_NONE 13

// tile-local position of a halo atom: (x, y, z, as_float(global sorted index | shift code << 27))
__device__ __forceinline__ float4 tile_transform(const TileGeom &g, const TileTables &t, int seg, float4 p, int gidx,
                                                 const DevGeom *dg) {
    float4 o;
    if (t.seg_wrapped[seg]) {                  // periodic image: lattice shift - origin added in fp64, rounded once
        const int code = t.seg_code[seg];
        const int wx = code % 3 - 1, wy = (code / 3) % 3 - 1, wz = code / 9 - 1;
        const TileBox b = tile_box(g, dg);
        o.x = (float)((double)p.x + (wx * b.ax + wy * b.bx + wz * b.cx - (double)t.origin[0]));
        o.y = (float)((double)p.y + (wy * b.by + wz * b.cy - (double)t.origin[1]));
        o.z = (float)((double)p.z + (wz * b.cz - (double)t.origin[2]));
    } else {
        o.x = p.x - t.origin[0]; o.y = p.y - t.origin[1]; o.z = p.z - t.origin[2];
    }
    o.w = __int_as_float(gidx | ((int)t.seg_code[seg] << NL_IDX_BITS));
    return o;
}

// Stages all halo positions into pos_s (warp per segment, coalesced).  No-op if the halo does not fit.
__device__ __forceinline__ void tile_stage_pos(const TileGeom &g, const TileTables &t, const float4 *__restrict__ spos, float4 *pos_s,
                                               const DevGeom *dg) {
    if (!t.staged) return;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int s = wid; s < 3 * t.nrows; s += nw) {
        const int len = t.seg_len[s], g0 = t.seg_g[s], l0 = t.seg_off[s];
        for (int i = lane; i < len; i += 32) pos_s[l0 + i] = tile_transform(g, t, s, spos[g0 + i], g0 + i, dg);
    }
}

// Interior tiles (no periodic image in the halo): every segment is a contiguous range of the cell-sorted float4 array whose
// .w already holds (sorted index | no-shift code) (k_cell_sort_gather on tiled contexts), so the staging is a handful of TMA
// bulk copies (cp.async.bulk, one per segment, completion on an mbarrier) of the RAW coordinates — differences of fp32
// inputs inside the primary cell are exact, no origin is needed.  All threads of the block must call it; returns after the
// data has landed.
__device__ __forceinline__ void tile_stage_pos_tma(const TileTables &t, const float4 *__restrict__ spos, float4 *pos_s,
                                                   unsigned long long *bar) {
    const unsigned bar_a = (unsigned)__cvta_generic_to_shared(bar);
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the set-up scratch lived where the copies will land
    __syncthreads();
    if (threadIdx.x == 0)
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"((unsigned)t.total * 16u) : "memory");
    if (threadIdx.x < 3 * t.nrows) {
        const int len = t.seg_len[threadIdx.x];
        if (len > 0) {
            const unsigned dst = (unsigned)__cvta_generic_to_shared(pos_s + t.seg_off[threadIdx.x]);
            const float4 *src = spos + t.seg_g[threadIdx.x];
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(dst), "l"(src), "r"((unsigned)len * 16u), "r"(bar_a) : "memory");
        }
    }
    unsigned done = 0;
    while (!done) {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(bar_a) : "memory");
    }
}

// position accessor that also works when the tile was not staged (slow path, global memory)
__device__ __forceinline__ float4 tile_pos(const TileGeom &g, const TileTables &t, const float4 *__restrict__ spos, const float4 *pos_s, int li,
                                           const DevGeom *dg) {
    if (t.staged) return pos_s[li];
    int s = tile_seg_of(t, li);
    int gi = t.seg_g[s] + (li - t.seg_off[s]);
    return tile_transform(g, t, s, spos[gi], gi, dg);
}

// own atom number a (0..nown-1) -> own-row q
__device__ __forceinline__ int tile_own_row(const TileTables &t, int a) {
    int q = 0;
#pragma unroll 1
    while (a >= t.own_off[q + 1]) ++q;
    return q;
}

// sliced neighbour-list layout: 32 consecutive atoms share a [maxn][32] slab (coalesced for
// thread-per-atom consumers, compact in memory)
__device__ __forceinline__ size_t nl_slot(int s, int k, int maxn) {
    return ((size_t)(s >> 5) * maxn + k) * 32 + (s & 31);
}
