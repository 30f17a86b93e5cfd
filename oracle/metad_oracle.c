/* metad_oracle.c — the CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, fp64 restatement of what the per-step metadynamics hot path computes, written
 * from the paper (PAPER.md, arxiv 2510.06873) and, where the paper is silent, from the readings
 * listed in DESIGN.md §3 (= SURVEY.md §8(c), points A–U).  It shares no code, header, table or
 * constant generator with the CUDA path (paper_2510_06873_b200/csrc/) and neither imports the
 * other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.  Compile with -O2 -ffp-contract=off (no FMA contraction: the neighbour
 * predicate's rounding is part of its definition, reading O).
 *
 * Every exported function cites the passage or reading it follows.  Pins (tests/test_oracle_*.py,
 * -m "not gpu") are listed in DESIGN.md §4; no function here is "parity unpinned".
 *
 * Conventions: positions pos[N][3] (row-major doubles), box[9] = rows a=(ax,0,0), b=(bx,by,0),
 * c=(cx,cy,cz); neighbour lists are row-major list[i*maxn + k], k < count[i], ascending j.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * Box checks (reading O): lower-triangular, positive diagonal, rc < half of every perpendicular
 * width.  Returns 0 if valid.  Widths: V/|b x c|, V/|c x a|, V/|a x b|.                        */
int orc_box_check(const double *box, double rc, double *widths /*[3] or NULL*/) {
    if (box[1] != 0.0 || box[2] != 0.0 || box[5] != 0.0) return 1;
    if (!(box[0] > 0.0) || !(box[4] > 0.0) || !(box[8] > 0.0)) return 1;
    const double *a = box, *b = box + 3, *c = box + 6;
    double vol = a[0] * b[1] * c[2];
    double bxc[3] = { b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0] };
    double cxa[3] = { c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0] };
    double axb[3] = { a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0] };
    double w[3];
    w[0] = vol / sqrt(bxc[0] * bxc[0] + bxc[1] * bxc[1] + bxc[2] * bxc[2]);
    w[1] = vol / sqrt(cxa[0] * cxa[0] + cxa[1] * cxa[1] + cxa[2] * cxa[2]);
    w[2] = vol / sqrt(axb[0] * axb[0] + axb[1] * axb[1] + axb[2] * axb[2]);
    if (widths) { widths[0] = w[0]; widths[1] = w[1]; widths[2] = w[2]; }
    if (!(rc > 0.0)) return 2;
    if (!(rc < 0.5 * w[0]) || !(rc < 0.5 * w[1]) || !(rc < 0.5 * w[2])) return 2;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Minimum-image displacement d = r_j - r_i (reading O): componentwise difference, then in this
 * order: z against c, y against b, x against a, each a single +/- lattice-vector shift.        */
void orc_delta(const double *box, const double *ri, const double *rj, double *d) {
    double dx = rj[0] - ri[0], dy = rj[1] - ri[1], dz = rj[2] - ri[2];
    double hz = 0.5 * box[8], hy = 0.5 * box[4], hx = 0.5 * box[0];
    if (dz > hz) { dx -= box[6]; dy -= box[7]; dz -= box[8]; }
    else if (dz < -hz) { dx += box[6]; dy += box[7]; dz += box[8]; }
    if (dy > hy) { dx -= box[3]; dy -= box[4]; }
    else if (dy < -hy) { dx += box[3]; dy += box[4]; }
    if (dx > hx) { dx -= box[0]; }
    else if (dx < -hx) { dx += box[0]; }
    d[0] = dx; d[1] = dy; d[2] = dz;
}

/* r^2 with the canonical rounding order (reading O): (dx*dx + dy*dy) + dz*dz, no FMA. */
static double r2_of(const double *d) { return (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]; }

/* Neighbour predicate (reading O, B: strict r < rc, plain truncation). */
static int is_neighbor(const double *box, const double *ri, const double *rj, double rc2) {
    double d[3];
    orc_delta(box, ri, rj, d);
    return r2_of(d) < rc2;
}

/* ---------------------------------------------------------------------------------------------
 * Neighbour lists.  Full lists (i->j and j->i), j != i (reading C, P), ascending j.
 * All three return the largest per-atom count; entries beyond maxn are dropped (count keeps the
 * true number so the caller can see the overflow).                                            */

/* O(N^2) with the canonical predicate. */
int orc_neighbors_brute(int N, const double *pos, const double *box, double rc, int maxn,
                        int *count, int *list) {
    double rc2 = rc * rc;
    int mx = 0;
    for (int i = 0; i < N; ++i) {
        int c = 0;
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            if (is_neighbor(box, pos + 3 * i, pos + 3 * j, rc2)) {
                if (c < maxn) list[(size_t)i * maxn + c] = j;
                ++c;
            }
        }
        count[i] = c;
        if (c > mx) mx = c;
    }
    return mx;
}

/* O(N^2 * 125 images): the DEFINITION the predicate must reproduce — j is a neighbour of i iff
 * some periodic image of r_j lies at Euclidean distance < rc from r_i.  Used only as a pin.    */
int orc_neighbors_images(int N, const double *pos, const double *box, double rc, int maxn,
                         int *count, int *list) {
    double rc2 = rc * rc;
    int mx = 0;
    for (int i = 0; i < N; ++i) {
        int c = 0;
        for (int j = 0; j < N; ++j) {
            if (j == i) continue;
            int hit = 0;
            for (int na = -2; na <= 2 && !hit; ++na)
            for (int nb = -2; nb <= 2 && !hit; ++nb)
            for (int nc = -2; nc <= 2 && !hit; ++nc) {
                double dx = pos[3 * j] - pos[3 * i] + na * box[0] + nb * box[3] + nc * box[6];
                double dy = pos[3 * j + 1] - pos[3 * i + 1] + nb * box[4] + nc * box[7];
                double dz = pos[3 * j + 2] - pos[3 * i + 2] + nc * box[8];
                if (dx * dx + dy * dy + dz * dz < rc2) hit = 1;
            }
            if (hit) {
                if (c < maxn) list[(size_t)i * maxn + c] = j;
                ++c;
            }
        }
        count[i] = c;
        if (c > mx) mx = c;
    }
    return mx;
}

static int cmp_int(const void *a, const void *b) {
    int x = *(const int *)a, y = *(const int *)b;
    return (x > y) - (x < y);
}

/* Cell list, O(N * 27 * atoms-per-cell), same predicate; for large N.  Cells are an acceleration
 * structure only: bins in fractional coordinates with perpendicular width >= rc, so every pair
 * with r < rc lies in adjacent bins.  With fewer than 3 bins along a direction the duplicate
 * bins are visited once.                                                                        */
int orc_neighbors_cells(int N, const double *pos, const double *box, double rc, int maxn,
                        int *count, int *list) {
    double w[3];
    if (orc_box_check(box, rc, w) != 0) return -1;
    int nc[3];
    for (int d = 0; d < 3; ++d) {
        nc[d] = (int)floor(w[d] / (rc * 1.000001));
        if (nc[d] < 1) nc[d] = 1;
        if (nc[d] > 512) nc[d] = 512;
    }
    long ncell = (long)nc[0] * nc[1] * nc[2];
    int *head = (int *)malloc(sizeof(int) * ncell), *next = (int *)malloc(sizeof(int) * N);
    int *cell = (int *)malloc(sizeof(int) * 3 * (size_t)N);
    for (long c = 0; c < ncell; ++c) head[c] = -1;
    for (int i = 0; i < N; ++i) {
        const double *r = pos + 3 * i;
        double s[3];
        s[2] = r[2] / box[8];
        s[1] = (r[1] - s[2] * box[7]) / box[4];
        s[0] = (r[0] - s[1] * box[3] - s[2] * box[6]) / box[0];
        for (int d = 0; d < 3; ++d) {
            s[d] -= floor(s[d]);
            int ic = (int)(s[d] * nc[d]);
            if (ic >= nc[d]) ic = nc[d] - 1;
            if (ic < 0) ic = 0;
            cell[3 * i + d] = ic;
        }
        long c = ((long)cell[3 * i + 2] * nc[1] + cell[3 * i + 1]) * nc[0] + cell[3 * i];
        next[i] = head[c]; head[c] = i;
    }
    double rc2 = rc * rc;
    int mx = 0;
#pragma omp parallel for schedule(dynamic, 256) reduction(max : mx)
    for (int i = 0; i < N; ++i) {
        int c = 0;
        int *li = list + (size_t)i * maxn;
        int seen[27], nseen = 0;
        for (int oz = -1; oz <= 1; ++oz)
        for (int oy = -1; oy <= 1; ++oy)
        for (int ox = -1; ox <= 1; ++ox) {
            int jc0 = (cell[3 * i] + ox + nc[0]) % nc[0];
            int jc1 = (cell[3 * i + 1] + oy + nc[1]) % nc[1];
            int jc2 = (cell[3 * i + 2] + oz + nc[2]) % nc[2];
            int cid = (jc2 * nc[1] + jc1) * nc[0] + jc0;
            int dup = 0;
            for (int q = 0; q < nseen; ++q) if (seen[q] == cid) dup = 1;
            if (dup) continue;
            seen[nseen++] = cid;
            for (int j = head[cid]; j >= 0; j = next[j]) {
                if (j == i) continue;
                if (is_neighbor(box, pos + 3 * i, pos + 3 * j, rc2)) {
                    if (c < maxn) li[c] = j;
                    ++c;
                }
            }
        }
        qsort(li, c < maxn ? c : maxn, sizeof(int), cmp_int);
        count[i] = c;
        if (c > mx) mx = c;
    }
    free(head); free(next); free(cell);
    return mx;
}

/* ---------------------------------------------------------------------------------------------
 * Rational switching function (BASELINE.json configs[0]: s(r) = (1-(r/r0)^n)/(1-(r/r0)^m);
 * reading A: x = r/r0, d0 = 0; at the removable singularity x = 1 the value is n/m and the
 * slope n(n-m)/(2m); a 2-term Taylor expansion is used for |x-1| < 1e-6).
 * Returns sw(x); *dsw = d sw / d x.                                                            */
double orc_switch(double x, int n, int m, double *dsw) {
    double e = x - 1.0;
    if (fabs(e) < 1e-6) {
        double s0 = (double)n / (double)m;
        double s1 = (double)n * (double)(n - m) / (2.0 * (double)m);
        if (dsw) *dsw = s1;
        return s0 + s1 * e;
    }
    double xn = pow(x, (double)n), xm = pow(x, (double)m);
    double num = 1.0 - xn, den = 1.0 - xm;
    double f = num / den;
    if (dsw) {
        double dnum = -(double)n * pow(x, (double)(n - 1));
        double dden = -(double)m * pow(x, (double)(m - 1));
        *dsw = (dnum * den - num * dden) / (den * den);
    }
    return f;
}

/* ---------------------------------------------------------------------------------------------
 * Coordination-number CV ("coordination number (C.N.)"; BASELINE.json configs[0],[2];
 * readings A–D): s = scale * sum_{i in A} sum_{j in B, j != i, r_ij < rc} sw(r_ij / r0).
 * Ordered pairs, each (i in A, j in B) once (reading C); plain truncation at rc (reading B) — the
 * list already encodes r < rc.  flags[i] bit0 = i in A, bit1 = i in B (NULL: every atom in both).
 * grad (N*3, may be NULL) receives d s / d r_k, accumulated pair by pair.                       */
double orc_cv_coord(int N, const double *pos, const double *box, const int *count, const int *list,
                    int maxn, const unsigned char *flags, double r0, int n, int m, double scale,
                    double *grad) {
    double s = 0.0;
    if (grad) memset(grad, 0, sizeof(double) * 3 * (size_t)N);
    for (int i = 0; i < N; ++i) {
        if (flags && !(flags[i] & 1)) continue;
        int c = count[i] < maxn ? count[i] : maxn;
        for (int k = 0; k < c; ++k) {
            int j = list[(size_t)i * maxn + k];
            if (flags && !(flags[j] & 2)) continue;
            double d[3];
            orc_delta(box, pos + 3 * i, pos + 3 * j, d);
            double r = sqrt(r2_of(d));
            double dsw, sw = orc_switch(r / r0, n, m, &dsw);
            s += sw;
            if (grad) {
                /* d sw(r/r0)/d r_j = dsw/r0 * d/r ; d/d r_i = minus that */
                double g = scale * dsw / (r0 * r);
                for (int a = 0; a < 3; ++a) {
                    grad[3 * j + a] += g * d[a];
                    grad[3 * i + a] -= g * d[a];
                }
            }
        }
    }
    return scale * s;
}

/* ---------------------------------------------------------------------------------------------
 * Steinhardt q6 per atom (BASELINE.json north_star / configs[3],[4]; reading E).
 * Primary route = the rotation-invariant double sum obtained from the addition theorem
 *   q6(i)^2 = (1/n_i^2) sum_{j,k in N(i)} P6(u_ij . u_ik),   P6(x) = (231x^6-315x^4+105x^2-5)/16,
 * which needs no spherical harmonics (so it shares not even a formula with the CUDA path's Y6m
 * recurrence).  n_i = 0 => q6 = 0.                                                              */
static double P6(double x) {
    double x2 = x * x;
    return (((231.0 * x2 - 315.0) * x2 + 105.0) * x2 - 5.0) / 16.0;
}
static double dP6(double x) {
    double x2 = x * x;
    return ((1386.0 * x2 - 1260.0) * x2 + 210.0) * x / 16.0;
}

void orc_q6_atoms(int N, const double *pos, const double *box, const int *count, const int *list,
                  int maxn, double *q6) {
#pragma omp parallel for schedule(dynamic, 256)
    for (int i = 0; i < N; ++i) {
        int c = count[i] < maxn ? count[i] : maxn;
        if (c == 0) { q6[i] = 0.0; continue; }
        double u[64][3];
        double (*uu)[3] = u;
        if (c > 64) uu = (double (*)[3])malloc(sizeof(double) * 3 * c);
        for (int k = 0; k < c; ++k) {
            int j = list[(size_t)i * maxn + k];
            double d[3];
            orc_delta(box, pos + 3 * i, pos + 3 * j, d);
            double r = sqrt(r2_of(d));
            uu[k][0] = d[0] / r; uu[k][1] = d[1] / r; uu[k][2] = d[2] / r;
        }
        double S = 0.0;
        for (int j = 0; j < c; ++j)
            for (int k = 0; k < c; ++k)
                S += P6(uu[j][0] * uu[k][0] + uu[j][1] * uu[k][1] + uu[j][2] * uu[k][2]);
        if (S < 0.0) S = 0.0;
        q6[i] = sqrt(S) / (double)c;
        if (uu != u) free(uu);
    }
}

/* Gradient of E = sum_i w_i q6(i) with respect to all positions (reading E), from the same double
 * sum: with S_i = n_i^2 q6_i^2,  dS_i/du_ij = 2 sum_{k != j} P6'(u_ij.u_ik) u_ik, projected onto
 * the tangent plane and divided by r_ij (u = d/|d|), and dq6_i = dS_i / (2 n_i^2 q6_i).
 * d_ij = r_j - r_i, so the term is added to atom j and subtracted from atom i.  Atoms with
 * n_i = 0 or q6_i = 0 contribute nothing.  The hard-cutoff delta term is ignored (reading E).
 * grad must hold N*3 doubles; it is overwritten.  Serial scatter (deterministic).               */
void orc_q6_grad(int N, const double *pos, const double *box, const int *count, const int *list,
                 int maxn, const double *q6, const double *w, double *grad) {
    memset(grad, 0, sizeof(double) * 3 * (size_t)N);
    double (*uu)[3] = (double (*)[3])malloc(sizeof(double) * 3 * (maxn > 0 ? maxn : 1));
    double *rr = (double *)malloc(sizeof(double) * (maxn > 0 ? maxn : 1));
    for (int i = 0; i < N; ++i) {
        int c = count[i] < maxn ? count[i] : maxn;
        if (c == 0 || !(q6[i] > 0.0) || w[i] == 0.0) continue;
        for (int k = 0; k < c; ++k) {
            int j = list[(size_t)i * maxn + k];
            double d[3];
            orc_delta(box, pos + 3 * i, pos + 3 * j, d);
            double r = sqrt(r2_of(d));
            rr[k] = r;
            uu[k][0] = d[0] / r; uu[k][1] = d[1] / r; uu[k][2] = d[2] / r;
        }
        double pref = w[i] / (2.0 * (double)c * (double)c * q6[i]);
        for (int j = 0; j < c; ++j) {
            double g[3] = { 0.0, 0.0, 0.0 };
            for (int k = 0; k < c; ++k) {
                if (k == j) continue;
                double x = uu[j][0] * uu[k][0] + uu[j][1] * uu[k][1] + uu[j][2] * uu[k][2];
                double dp = 2.0 * dP6(x);
                g[0] += dp * uu[k][0]; g[1] += dp * uu[k][1]; g[2] += dp * uu[k][2];
            }
            double gu = g[0] * uu[j][0] + g[1] * uu[j][1] + g[2] * uu[j][2];
            int ja = list[(size_t)i * maxn + j];
            for (int a = 0; a < 3; ++a) {
                double t = pref * (g[a] - gu * uu[j][a]) / rr[j];
                grad[3 * ja + a] += t;
                grad[3 * i + a] -= t;
            }
        }
    }
    free(uu); free(rr);
}

/* Secondary route for q6 (tiny inputs; a pin for the primary route): explicit l = 6 spherical
 * harmonics on the unit vector, q6m = (1/n) sum_j Y6m, q6 = sqrt(4pi/13 * sum_{m=-6..6} |q6m|^2),
 * with |q6,-m| = |q6m|.  ylm_out (may be NULL) receives, for atom i, 7 complex numbers
 * (re,im) = q6m, m = 0..6, i.e. 14 doubles per atom.  The table is the textbook one. */
void orc_y6(const double *u, double *y /*[14]*/) {
    double x = u[0], yy = u[1], z = u[2];
    double z2 = z * z;
    double pi = 3.14159265358979323846;
    double c1r = x, c1i = yy;                    /* (x+iy)^m by repeated multiplication */
    double pr[7], pim[7];
    pr[0] = 1.0; pim[0] = 0.0;
    for (int m = 1; m <= 6; ++m) {
        pr[m] = pr[m - 1] * c1r - pim[m - 1] * c1i;
        pim[m] = pr[m - 1] * c1i + pim[m - 1] * c1r;
    }
    double f[7];
    f[0] = (1.0 / 32.0) * sqrt(13.0 / pi) * (231.0 * z2 * z2 * z2 - 315.0 * z2 * z2 + 105.0 * z2 - 5.0);
    f[1] = -(1.0 / 16.0) * sqrt(273.0 / (2.0 * pi)) * z * (33.0 * z2 * z2 - 30.0 * z2 + 5.0);
    f[2] = (1.0 / 64.0) * sqrt(1365.0 / pi) * (33.0 * z2 * z2 - 18.0 * z2 + 1.0);
    f[3] = -(1.0 / 32.0) * sqrt(1365.0 / pi) * z * (11.0 * z2 - 3.0);
    f[4] = (3.0 / 32.0) * sqrt(91.0 / (2.0 * pi)) * (11.0 * z2 - 1.0);
    f[5] = -(3.0 / 32.0) * sqrt(1001.0 / pi) * z;
    f[6] = (1.0 / 64.0) * sqrt(3003.0 / pi);
    for (int m = 0; m <= 6; ++m) { y[2 * m] = f[m] * pr[m]; y[2 * m + 1] = f[m] * pim[m]; }
}

void orc_q6_atoms_ylm(int N, const double *pos, const double *box, const int *count, const int *list,
                      int maxn, double *q6, double *ylm_out) {
    double pi = 3.14159265358979323846;
    for (int i = 0; i < N; ++i) {
        int c = count[i] < maxn ? count[i] : maxn;
        double q[14];
        for (int t = 0; t < 14; ++t) q[t] = 0.0;
        for (int k = 0; k < c; ++k) {
            int j = list[(size_t)i * maxn + k];
            double d[3], u[3], y[14];
            orc_delta(box, pos + 3 * i, pos + 3 * j, d);
            double r = sqrt(r2_of(d));
            u[0] = d[0] / r; u[1] = d[1] / r; u[2] = d[2] / r;
            orc_y6(u, y);
            for (int t = 0; t < 14; ++t) q[t] += y[t];
        }
        if (c > 0) for (int t = 0; t < 14; ++t) q[t] /= (double)c;
        double s = q[0] * q[0] + q[1] * q[1];
        for (int m = 1; m <= 6; ++m) s += 2.0 * (q[2 * m] * q[2 * m] + q[2 * m + 1] * q[2 * m + 1]);
        q6[i] = sqrt(4.0 * pi / 13.0 * s);
        if (ylm_out) memcpy(ylm_out + 14 * (size_t)i, q, sizeof(q));
    }
}

/* ---------------------------------------------------------------------------------------------
 * Radius of gyration of an ordered chain (BASELINE.json configs[1]; reading G):
 * unwrap by sequential minimum image along the index list, u_0 = r_c0, u_k = u_{k-1} + delta(r_c(k-1), r_ck);
 * Rg = sqrt( sum m_k |u_k - u_com|^2 / M ); dRg/dr_ck = m_k (u_k - u_com) / (M Rg).
 * grad (nchain*3, may be NULL) is indexed by chain position k.                                  */
double orc_cv_rgyr(int nchain, const int *chain, const double *mass, const double *pos,
                   const double *box, double *grad) {
    double *u = (double *)malloc(sizeof(double) * 3 * (size_t)nchain);
    for (int a = 0; a < 3; ++a) u[a] = pos[3 * chain[0] + a];
    for (int k = 1; k < nchain; ++k) {
        double d[3];
        orc_delta(box, pos + 3 * chain[k - 1], pos + 3 * chain[k], d);
        for (int a = 0; a < 3; ++a) u[3 * k + a] = u[3 * (k - 1) + a] + d[a];
    }
    double M = 0.0, com[3] = { 0.0, 0.0, 0.0 };
    for (int k = 0; k < nchain; ++k) {
        double mk = mass ? mass[k] : 1.0;
        M += mk;
        for (int a = 0; a < 3; ++a) com[a] += mk * u[3 * k + a];
    }
    for (int a = 0; a < 3; ++a) com[a] /= M;
    double s = 0.0;
    for (int k = 0; k < nchain; ++k) {
        double mk = mass ? mass[k] : 1.0;
        for (int a = 0; a < 3; ++a) { double t = u[3 * k + a] - com[a]; s += mk * t * t; }
    }
    double rg = sqrt(s / M);
    if (grad) {
        for (int k = 0; k < nchain; ++k) {
            double mk = mass ? mass[k] : 1.0;
            for (int a = 0; a < 3; ++a)
                grad[3 * k + a] = rg > 0.0 ? mk * (u[3 * k + a] - com[a]) / (M * rg) : 0.0;
        }
    }
    free(u);
    return rg;
}

/* ---------------------------------------------------------------------------------------------
 * Native-contact fraction (BASELINE.json configs[1]; reading H):
 * Qc = scale * sum_p sw(r_p / r0_p), r_p = minimum-image distance of pair p, scale = 1/P,
 * r0_p = 1.5 * reference distance, n = 6, m = 12.  grad (N*3, may be NULL) is overwritten.      */
double orc_cv_contacts(int N, int npairs, const int *pairs, const double *pair_r0, int n, int m,
                       double scale, const double *pos, const double *box, double *grad) {
    double s = 0.0;
    if (grad) memset(grad, 0, sizeof(double) * 3 * (size_t)N);
    for (int p = 0; p < npairs; ++p) {
        int i = pairs[2 * p], j = pairs[2 * p + 1];
        double d[3];
        orc_delta(box, pos + 3 * i, pos + 3 * j, d);
        double r = sqrt(r2_of(d));
        double dsw, sw = orc_switch(r / pair_r0[p], n, m, &dsw);
        s += sw;
        if (grad) {
            double g = scale * dsw / (pair_r0[p] * r);
            for (int a = 0; a < 3; ++a) { grad[3 * j + a] += g * d[a]; grad[3 * i + a] -= g * d[a]; }
        }
    }
    return scale * s;
}

/* ---------------------------------------------------------------------------------------------
 * Metadynamics bias (Methods): V_b(s) = sum_tau w_tau exp(-(s - s_tau)^2 / (2 sigma^2)),
 * for a D-dimensional s a product of 1-D Gaussians with per-dimension sigma (reading L), summed
 * over ALL hills with no truncation.  dV/ds_d = sum_tau -w_tau (s_d - c_tau,d)/sigma_d^2 * (...).
 * centers is [H][D] row-major.                                                                  */
void orc_bias(int D, int H, const double *centers, const double *heights, const double *sigma,
              const double *s, double *V, double *dVds) {
    double v = 0.0, dv[8];
    for (int d = 0; d < D; ++d) dv[d] = 0.0;
    for (int k = 0; k < H; ++k) {
        double e = 0.0;
        for (int d = 0; d < D; ++d) {
            double t = (s[d] - centers[(size_t)k * D + d]) / sigma[d];
            e += t * t;
        }
        double g = heights[k] * exp(-0.5 * e);
        v += g;
        for (int d = 0; d < D; ++d)
            dv[d] += -g * (s[d] - centers[(size_t)k * D + d]) / (sigma[d] * sigma[d]);
    }
    *V = v;
    for (int d = 0; d < D; ++d) dVds[d] = dv[d];
}

/* Well-tempered height (PAPER.md:43 names the method, ref. [16] PAPER.md:121; reading I):
 * w = w0 exp(-V(s)/(kB dT)), dT = (gamma - 1) T, i.e. kB dT = (gamma-1) kT.  gamma <= 1: w = w0. */
double orc_wt_height(double w0, double V, double kT, double gamma) {
    if (!(gamma > 1.0)) return w0;
    return w0 * exp(-V / ((gamma - 1.0) * kT));
}

/* ---------------------------------------------------------------------------------------------
 * Grid-tabulated 2-D bias (BASELINE.json configs[4]; reading M): at the n0 x n1 nodes of
 * [lo0,hi0] x [lo1,hi1] store the analytic V, dV/ds0, dV/ds1, d2V/ds0ds1 of the hill sum;
 * table layout [4][n0][n1].  Evaluation = bicubic Hermite on the enclosing cell.
 * orc_grid_add adds hills k0..k1-1 to an existing table (deposition adds one hill).             */
void orc_grid_add(int n0, int n1, const double *lo, const double *hi, int k0, int k1,
                  const double *centers /*[H][2]*/, const double *heights, const double *sigma,
                  double *table) {
    double h0 = (hi[0] - lo[0]) / (n0 - 1), h1 = (hi[1] - lo[1]) / (n1 - 1);
    size_t plane = (size_t)n0 * n1;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n0; ++i) {
        double x = lo[0] + i * h0;
        for (int j = 0; j < n1; ++j) {
            double y = lo[1] + j * h1;
            double v = 0.0, v0 = 0.0, v1 = 0.0, v01 = 0.0;
            for (int k = k0; k < k1; ++k) {
                double a = (x - centers[2 * k]) / sigma[0], b = (y - centers[2 * k + 1]) / sigma[1];
                double g = heights[k] * exp(-0.5 * (a * a + b * b));
                double ga = -a / sigma[0], gb = -b / sigma[1];
                v += g; v0 += g * ga; v1 += g * gb; v01 += g * ga * gb;
            }
            size_t o = (size_t)i * n1 + j;
            table[o] += v; table[plane + o] += v0; table[2 * plane + o] += v1; table[3 * plane + o] += v01;
        }
    }
}

/* cubic Hermite basis on t in [0,1]: value weights (h00,h01) and slope weights (h10,h11), and
 * their t-derivatives. */
static void hermite(double t, double *h, double *dh) {
    double t2 = t * t, t3 = t2 * t;
    h[0] = 2 * t3 - 3 * t2 + 1;  h[1] = -2 * t3 + 3 * t2;  h[2] = t3 - 2 * t2 + t;  h[3] = t3 - t2;
    dh[0] = 6 * t2 - 6 * t;      dh[1] = -6 * t2 + 6 * t;  dh[2] = 3 * t2 - 4 * t + 1; dh[3] = 3 * t2 - 2 * t;
}

/* returns 0, or 1 if s is outside the table (caller falls back to the exact sum, reading M). */
int orc_grid_eval(int n0, int n1, const double *lo, const double *hi, const double *table,
                  const double *s, double *V, double *dVds) {
    double h0 = (hi[0] - lo[0]) / (n0 - 1), h1 = (hi[1] - lo[1]) / (n1 - 1);
    if (!(s[0] >= lo[0]) || !(s[0] <= hi[0]) || !(s[1] >= lo[1]) || !(s[1] <= hi[1])) return 1;
    double fx = (s[0] - lo[0]) / h0, fy = (s[1] - lo[1]) / h1;
    int i = (int)floor(fx), j = (int)floor(fy);
    if (i > n0 - 2) i = n0 - 2;
    if (j > n1 - 2) j = n1 - 2;
    double tx = fx - i, ty = fy - j;
    double hx[4], dhx[4], hy[4], dhy[4];
    hermite(tx, hx, dhx); hermite(ty, hy, dhy);
    size_t plane = (size_t)n0 * n1;
    double v = 0.0, vx = 0.0, vy = 0.0;
    for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) {
        size_t o = (size_t)(i + a) * n1 + (j + b);
        double f = table[o], f0 = table[plane + o] * h0, f1 = table[2 * plane + o] * h1,
               f01 = table[3 * plane + o] * h0 * h1;
        /* value / x-slope / y-slope / cross weights */
        double wx = hx[a], wxs = hx[2 + a], wy = hy[b], wys = hy[2 + b];
        double dwx = dhx[a], dwxs = dhx[2 + a], dwy = dhy[b], dwys = dhy[2 + b];
        v  += f * wx * wy + f0 * wxs * wy + f1 * wx * wys + f01 * wxs * wys;
        vx += f * dwx * wy + f0 * dwxs * wy + f1 * dwx * wys + f01 * dwxs * wys;
        vy += f * wx * dwy + f0 * wxs * dwy + f1 * wx * dwys + f01 * wxs * dwys;
    }
    *V = v; dVds[0] = vx / h0; dVds[1] = vy / h1;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Bias forces (PAPER.md:77 U_b = U_0 + V_b => forces add; "bias-driven forces";
 * reading N): F_k += -force_scale * sum_d dVds[d] * grad_d[k].  grads is [D][N*3].              */
void orc_apply_forces(int N, int D, const double *dVds, const double *grads, double force_scale,
                      double *F) {
    for (size_t t = 0; t < (size_t)3 * N; ++t) {
        double acc = 0.0;
        for (int d = 0; d < D; ++d) acc += dVds[d] * grads[(size_t)d * 3 * N + t];
        F[t] += -force_scale * acc;
    }
}

/* =============================================================================================
 * NEXT-1: the paper's first workload — backbone torsions Phi, Psi of alanine
 * dipeptide as CVs, sigma = 0.35 rad, W = 1.2 kJ/mol — needs a torsion CV and a
 * bias that is periodic in the CV.  The paper gives neither formula; readings V, W, X of DESIGN.md.
 * ============================================================================================= */

/* Torsion (dihedral) angle of atoms i-j-k-l ("Phi(C-N-Ca-C) and Psi(N-Ca-C-N)";
 * reading V): IUPAC convention, bond vectors by minimum image,
 *     b1 = r_j - r_i, b2 = r_k - r_j, b3 = r_l - r_k,  n1 = b1 x b2,  n2 = b2 x b3,
 *     phi = atan2( |b2| b1.n2 , n1.n2 )  in (-pi, pi];   cis = 0, trans = pi.
 * Gradient (grad[4][3], may be NULL), written with F = -b1, G = -b2, H = b3, A = F x G = n1,
 * B = H x G = -n2 (the textbook form of Blondel & Karplus):
 *     dphi/dr_i = -|G|/A^2 A,   dphi/dr_l = +|G|/B^2 B,
 *     dphi/dr_j = +|G|/A^2 A + (F.G)/(A^2 |G|) A - (H.G)/(B^2 |G|) B,
 *     dphi/dr_k = -|G|/B^2 B - (F.G)/(A^2 |G|) A + (H.G)/(B^2 |G|) B.                            */
static void cross3(const double *a, const double *b, double *c) {
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}
static double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

double orc_cv_torsion(const int *idx, const double *pos, const double *box, double *grad) {
    double b1[3], b2[3], b3[3], n1[3], n2[3];
    orc_delta(box, pos + 3 * idx[0], pos + 3 * idx[1], b1);
    orc_delta(box, pos + 3 * idx[1], pos + 3 * idx[2], b2);
    orc_delta(box, pos + 3 * idx[2], pos + 3 * idx[3], b3);
    cross3(b1, b2, n1);
    cross3(b2, b3, n2);
    double lb2 = sqrt(dot3(b2, b2));
    double phi = atan2(lb2 * dot3(b1, n2), dot3(n1, n2));
    if (grad) {
        double F[3], G[3], H[3], A[3], B[3];
        for (int a = 0; a < 3; ++a) { F[a] = -b1[a]; G[a] = -b2[a]; H[a] = b3[a]; }
        cross3(F, G, A);
        cross3(H, G, B);
        double A2 = dot3(A, A), B2 = dot3(B, B), lG = sqrt(dot3(G, G));
        double FG = dot3(F, G), HG = dot3(H, G);
        for (int a = 0; a < 3; ++a) {
            double gi = -lG / A2 * A[a];
            double gl = lG / B2 * B[a];
            double gj = lG / A2 * A[a] + FG / (A2 * lG) * A[a] - HG / (B2 * lG) * B[a];
            double gk = -lG / B2 * B[a] - FG / (A2 * lG) * A[a] + HG / (B2 * lG) * B[a];
            grad[a] = gi; grad[3 + a] = gj; grad[6 + a] = gk; grad[9 + a] = gl;
        }
    }
    return phi;
}

/* Periodic difference (reading W): x - c brought to the nearest periodic image, in [-P/2, P/2];
 * P <= 0 means the dimension is not periodic. */
double orc_pdiff(double x, double c, double P) {
    double d = x - c;
    if (P > 0.0) d -= P * rint(d / P);
    return d;
}

/* Wraps x into [lo, lo + P). */
double orc_wrap(double x, double lo, double P) {
    double y = x - P * floor((x - lo) / P);
    if (y >= lo + P) y -= P;
    if (y < lo) y += P;
    return y;
}

/* Hill sum with periodic CV dimensions (PAPER.md:81 with (s - s_tau) read as the nearest-image
 * difference, reading W): one image per hill, no sum over images (the next image of a
 * sigma = 0.35 rad hill is below e^-40 at the discontinuity).  period[d] <= 0: not periodic.     */
void orc_bias_periodic(int D, int H, const double *centers, const double *heights, const double *sigma,
                       const double *period, const double *s, double *V, double *dVds) {
    double v = 0.0, dv[8];
    for (int d = 0; d < D; ++d) dv[d] = 0.0;
    for (int k = 0; k < H; ++k) {
        double e = 0.0, t[8];
        for (int d = 0; d < D; ++d) {
            t[d] = orc_pdiff(s[d], centers[(size_t)k * D + d], period[d]) / sigma[d];
            e += t[d] * t[d];
        }
        double g = heights[k] * exp(-0.5 * e);
        v += g;
        for (int d = 0; d < D; ++d) dv[d] += -g * t[d] / sigma[d];
    }
    *V = v;
    for (int d = 0; d < D; ++d) dVds[d] = dv[d];
}

/* Grid-tabulated 2-D bias with periodic dimensions (reading X): a periodic dimension d has n_d
 * nodes at lo_d + i * P_d / n_d (P_d = hi_d - lo_d; node n_d coincides with node 0), a
 * non-periodic one n_d nodes at lo_d + i (hi_d - lo_d)/(n_d - 1) as in orc_grid_add.  Node data
 * and interpolant as in reading M; a periodic dimension has no "outside".                        */
static double grid_h(int n, double lo, double hi, int periodic) { return periodic ? (hi - lo) / n : (hi - lo) / (n - 1); }

void orc_grid_add_p(int n0, int n1, const double *lo, const double *hi, const int *periodic, int k0, int k1,
                    const double *centers /*[H][2]*/, const double *heights, const double *sigma,
                    double *table) {
    double h0 = grid_h(n0, lo[0], hi[0], periodic[0]), h1 = grid_h(n1, lo[1], hi[1], periodic[1]);
    double P0 = periodic[0] ? hi[0] - lo[0] : 0.0, P1 = periodic[1] ? hi[1] - lo[1] : 0.0;
    size_t plane = (size_t)n0 * n1;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n0; ++i) {
        double x = lo[0] + i * h0;
        for (int j = 0; j < n1; ++j) {
            double y = lo[1] + j * h1;
            double v = 0.0, v0 = 0.0, v1 = 0.0, v01 = 0.0;
            for (int k = k0; k < k1; ++k) {
                double a = orc_pdiff(x, centers[2 * k], P0) / sigma[0], b = orc_pdiff(y, centers[2 * k + 1], P1) / sigma[1];
                double g = heights[k] * exp(-0.5 * (a * a + b * b));
                double ga = -a / sigma[0], gb = -b / sigma[1];
                v += g; v0 += g * ga; v1 += g * gb; v01 += g * ga * gb;
            }
            size_t o = (size_t)i * n1 + j;
            table[o] += v; table[plane + o] += v0; table[2 * plane + o] += v1; table[3 * plane + o] += v01;
        }
    }
}

int orc_grid_eval_p(int n0, int n1, const double *lo, const double *hi, const int *periodic, const double *table,
                    const double *s, double *V, double *dVds) {
    int n[2] = { n0, n1 }, i0[2], i1[2];
    double h[2], t[2];
    for (int d = 0; d < 2; ++d) {
        h[d] = grid_h(n[d], lo[d], hi[d], periodic[d]);
        if (periodic[d]) {
            double x = orc_wrap(s[d], lo[d], hi[d] - lo[d]);
            double f = (x - lo[d]) / h[d];
            int i = (int)floor(f);
            if (i > n[d] - 1) i = n[d] - 1;
            if (i < 0) i = 0;
            t[d] = f - i; i0[d] = i; i1[d] = (i + 1) % n[d];
        } else {
            if (!(s[d] >= lo[d]) || !(s[d] <= hi[d])) return 1;
            double f = (s[d] - lo[d]) / h[d];
            int i = (int)floor(f);
            if (i > n[d] - 2) i = n[d] - 2;
            t[d] = f - i; i0[d] = i; i1[d] = i + 1;
        }
    }
    double hx[4], dhx[4], hy[4], dhy[4];
    hermite(t[0], hx, dhx); hermite(t[1], hy, dhy);
    size_t plane = (size_t)n0 * n1;
    double v = 0.0, vx = 0.0, vy = 0.0;
    for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) {
        size_t o = (size_t)(a ? i1[0] : i0[0]) * n1 + (b ? i1[1] : i0[1]);
        double f = table[o], f0 = table[plane + o] * h[0], f1 = table[2 * plane + o] * h[1],
               f01 = table[3 * plane + o] * h[0] * h[1];
        double wx = hx[a], wxs = hx[2 + a], wy = hy[b], wys = hy[2 + b];
        double dwx = dhx[a], dwxs = dhx[2 + a], dwy = dhy[b], dwys = dhy[2 + b];
        v  += f * wx * wy + f0 * wxs * wy + f1 * wx * wys + f01 * wxs * wys;
        vx += f * dwx * wy + f0 * dwxs * wy + f1 * dwx * wys + f01 * dwxs * wys;
        vy += f * wx * dwy + f0 * wxs * dwy + f1 * wx * dwys + f01 * wxs * dwys;
    }
    *V = v; dVds[0] = vx / h[0]; dVds[1] = vy / h[1];
    return 0;
}

/* =============================================================================================
 * NEXT-2: free-energy reconstruction by reweighting:
 *     P_unbias(s) = < delta[s - s(R)] e^{beta V_b(s)} >_{U_b} / < e^{beta V_b(s)} >_{U_b},
 *     F(s) = -(1/beta) log P_unbias(s),
 * the averages running over the frames of the biased trajectory, V_b the (final) bias potential.
 * Reading Z: the delta function is a histogram on uniform bins (bin b of dimension d covers
 * [lo_d + b h_d, lo_d + (b+1) h_d), h_d = (hi_d - lo_d)/nb_d; a periodic dimension is wrapped into
 * [lo_d, hi_d) first); P is the bin average divided by the bin volume; frames outside the range of
 * a non-periodic dimension count in the denominator only; empty bins give F = +inf.
 * traj [T][D] row-major, D = 1 or 2 (nb[1] = 1, lo/hi[1] ignored for D = 1); P, F [nb0][nb1].       */
void orc_reweight(int D, int T, const double *traj, int H, const double *centers, const double *heights,
                  const double *sigma, const double *period, double kT, const int *nb, const double *lo,
                  const double *hi, double *P, double *F) {
    int n0 = nb[0], n1 = D > 1 ? nb[1] : 1;
    double vol = 1.0;
    for (int d = 0; d < D; ++d) vol *= (hi[d] - lo[d]) / nb[d];
    for (int b = 0; b < n0 * n1; ++b) P[b] = 0.0;
    double den = 0.0;
    for (int t = 0; t < T; ++t) {
        const double *s = traj + (size_t)t * D;
        double V, dV[8];
        orc_bias_periodic(D, H, centers, heights, sigma, period, s, &V, dV);
        double w = exp(V / kT);
        den += w;
        int idx[2] = { 0, 0 }, inside = 1;
        for (int d = 0; d < D; ++d) {
            double x = s[d];
            if (period[d] > 0.0) x = orc_wrap(x, lo[d], period[d]);
            double f = (x - lo[d]) / ((hi[d] - lo[d]) / nb[d]);
            int b = (int)floor(f);
            if (period[d] > 0.0 && b >= nb[d]) b = nb[d] - 1;
            if (b < 0 || b >= nb[d] || !(x >= lo[d])) inside = 0;
            idx[d] = b;
        }
        if (inside) P[(size_t)idx[0] * n1 + idx[1]] += w;
    }
    for (int b = 0; b < n0 * n1; ++b) {
        P[b] = P[b] / (den * vol);
        F[b] = P[b] > 0.0 ? -kT * log(P[b]) : INFINITY;
    }
}

/* =============================================================================================
 * NEXT-2b: the paper's second workload biases "the distance between a surface
 * oxygen atom and its nearest hydrogen atom".  Reading AA: s = min over i in A,
 * j in B, j != i, r_ij < rc of the minimum-image distance r_ij (A = the surface oxygen(s), B = the
 * hydrogens); the paper obtains forces by automatic differentiation, and the
 * derivative of a minimum is the derivative of its arg-min: d s/d r_j = d/r, d s/d r_i = -d/r for
 * the nearest pair (i, j), zero for every other atom.  Ties: the pair with the smallest (i, j) in
 * lexicographic order.  No pair within rc: s = rc, zero gradient.  The neighbour list (r < rc)
 * restricts the search exactly as in orc_cv_coord.  pair_out[2] (may be NULL) receives (i, j) or (-1,-1). */
double orc_cv_mindist(int N, const double *pos, const double *box, const int *count, const int *list,
                      int maxn, const unsigned char *flags, double rc, double *grad, int *pair_out) {
    double best = INFINITY, bd[3] = { 0, 0, 0 };
    int bi = -1, bj = -1;
    if (grad) memset(grad, 0, sizeof(double) * 3 * (size_t)N);
    for (int i = 0; i < N; ++i) {
        if (flags && !(flags[i] & 1)) continue;
        int c = count[i] < maxn ? count[i] : maxn;
        for (int k = 0; k < c; ++k) {
            int j = list[(size_t)i * maxn + k];
            if (flags && !(flags[j] & 2)) continue;
            double d[3];
            orc_delta(box, pos + 3 * i, pos + 3 * j, d);
            double r2 = r2_of(d);
            if (r2 < best || (r2 == best && (i < bi || (i == bi && j < bj)))) {
                best = r2; bi = i; bj = j; bd[0] = d[0]; bd[1] = d[1]; bd[2] = d[2];
            }
        }
    }
    if (pair_out) { pair_out[0] = bi; pair_out[1] = bj; }
    if (bi < 0) return rc;
    double r = sqrt(best);
    if (grad)
        for (int a = 0; a < 3; ++a) { grad[3 * bj + a] += bd[a] / r; grad[3 * bi + a] -= bd[a] / r; }
    return r;
}

/* =============================================================================================
 * NEXT-3: "We selected the coordination number (C.N.) and the triaxial lattice
 * parameters as CVs and ran NPT simulation".  Reading AB: the lattice parameter of
 * axis k is the length of box row k, s = |h_k| (a, b, c of the supercell); it does not depend on
 * the atomic positions, its gradient is taken with respect to the box matrix:
 * d s/d h_k = h_k/|h_k| (row k of grad9, other rows zero).  The bias then acts on the cell:
 * F_h = -force_scale * sum_d dV/ds_d * d s_d/d h (what an NPT integrator adds to its box force).   */
double orc_cv_lattice(const double *box, int axis, double *grad9) {
    const double *h = box + 3 * axis;
    double s = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
    if (grad9) {
        for (int k = 0; k < 9; ++k) grad9[k] = 0.0;
        for (int a = 0; a < 3; ++a) grad9[3 * axis + a] = h[a] / s;
    }
    return s;
}

/* =============================================================================================
 * NEXT-3b: bias virial for NPT runs ("ran NPT simulation at 300K and 50 GPa" with the
 * coordination number and the lattice parameters as CVs).  Reading AD: under a homogeneous strain
 * eps (r -> r + eps r, box rows h_k -> h_k + eps h_k) every pair vector changes as d -> d + eps d,
 * so for a CV that is a function of the pair vectors
 *     d s / d eps_ab = sum over ordered pairs (d s / d d_ij)_a (d_ij)_b ,
 * and the bias virial is W_ab = - sum_d dV/ds_d * d s_d / d eps_ab (energy units; its contribution
 * to the pressure tensor is W / volume).  The functions below return d s / d eps (3x3, row-major).  */

/* coordination number: d s/d d_ij = scale * sw'(r/r0)/(r0 r) d_ij for every ordered pair (i in A, j in B). */
void orc_cv_coord_strain(int N, const double *pos, const double *box, const int *count, const int *list,
                         int maxn, const unsigned char *flags, double r0, int n, int m, double scale,
                         double *dsde /*[9]*/) {
    for (int k = 0; k < 9; ++k) dsde[k] = 0.0;
    for (int i = 0; i < N; ++i) {
        if (flags && !(flags[i] & 1)) continue;
        int c = count[i] < maxn ? count[i] : maxn;
        for (int k = 0; k < c; ++k) {
            int j = list[(size_t)i * maxn + k];
            if (flags && !(flags[j] & 2)) continue;
            double d[3];
            orc_delta(box, pos + 3 * i, pos + 3 * j, d);
            double r = sqrt(r2_of(d));
            double dsw;
            orc_switch(r / r0, n, m, &dsw);
            double g = scale * dsw / (r0 * r);
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) dsde[3 * a + b] += g * d[a] * d[b];
        }
    }
}

/* E = sum_i w_i q6(i): the per-pair derivative dE/d d_ij is the vector t of orc_q6_grad (same formula). */
void orc_q6_strain(int N, const double *pos, const double *box, const int *count, const int *list,
                   int maxn, const double *q6, const double *w, double *dsde /*[9]*/) {
    for (int k = 0; k < 9; ++k) dsde[k] = 0.0;
    double (*uu)[3] = (double (*)[3])malloc(sizeof(double) * 3 * (maxn > 0 ? maxn : 1));
    double *rr = (double *)malloc(sizeof(double) * (maxn > 0 ? maxn : 1));
    for (int i = 0; i < N; ++i) {
        int c = count[i] < maxn ? count[i] : maxn;
        if (c == 0 || !(q6[i] > 0.0) || w[i] == 0.0) continue;
        for (int k = 0; k < c; ++k) {
            int j = list[(size_t)i * maxn + k];
            double d[3];
            orc_delta(box, pos + 3 * i, pos + 3 * j, d);
            double r = sqrt(r2_of(d));
            rr[k] = r;
            uu[k][0] = d[0] / r; uu[k][1] = d[1] / r; uu[k][2] = d[2] / r;
        }
        double pref = w[i] / (2.0 * (double)c * (double)c * q6[i]);
        for (int j = 0; j < c; ++j) {
            double g[3] = { 0.0, 0.0, 0.0 };
            for (int k = 0; k < c; ++k) {
                if (k == j) continue;
                double x = uu[j][0] * uu[k][0] + uu[j][1] * uu[k][1] + uu[j][2] * uu[k][2];
                double dp = 2.0 * dP6(x);
                g[0] += dp * uu[k][0]; g[1] += dp * uu[k][1]; g[2] += dp * uu[k][2];
            }
            double gu = g[0] * uu[j][0] + g[1] * uu[j][1] + g[2] * uu[j][2];
            for (int a = 0; a < 3; ++a) {
                double t = pref * (g[a] - gu * uu[j][a]) / rr[j];
                for (int b = 0; b < 3; ++b) dsde[3 * a + b] += t * rr[j] * uu[j][b];
            }
        }
    }
    free(uu); free(rr);
}

/* lattice parameter s = |h_k|: h_k -> h_k + eps h_k  =>  d s/d eps_ab = h_a h_b / |h_k|. */
void orc_cv_lattice_strain(const double *box, int axis, double *dsde /*[9]*/) {
    const double *h = box + 3 * axis;
    double s = sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]);
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) dsde[3 * a + b] = h[a] * h[b] / s;
}

/* Strain derivatives of the remaining CVs (reading AD), each a function of a few minimum-image vectors. */

/* Rg^2 = sum m |u - com|^2 / M on the unwrapped chain; u - com scales with the strain:
 * d Rg/d eps_ab = sum m (u - com)_a (u - com)_b / (M Rg). */
void orc_cv_rgyr_strain(int nchain, const int *chain, const double *mass, const double *pos,
                        const double *box, double *dsde) {
    double *g = (double *)malloc(sizeof(double) * 3 * (size_t)nchain);
    double rg = orc_cv_rgyr(nchain, chain, mass, pos, box, g);      /* g_k = m_k (u_k - com) / (M Rg) */
    double M = 0.0;
    for (int k = 0; k < nchain; ++k) M += mass ? mass[k] : 1.0;
    for (int k = 0; k < 9; ++k) dsde[k] = 0.0;
    for (int k = 0; k < nchain; ++k) {
        double mk = mass ? mass[k] : 1.0;
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b)
                dsde[3 * a + b] += rg > 0.0 ? g[3 * k + a] * (g[3 * k + b] * M * rg / mk) : 0.0;
    }
    free(g);
}

/* Qc = scale sum_p sw(r_p / r0_p):  d Qc/d eps = scale sum_p sw'/(r0_p r_p) d_p d_p^T. */
void orc_cv_contacts_strain(int npairs, const int *pairs, const double *pair_r0, int n, int m, double scale,
                            const double *pos, const double *box, double *dsde) {
    for (int k = 0; k < 9; ++k) dsde[k] = 0.0;
    for (int p = 0; p < npairs; ++p) {
        double d[3];
        orc_delta(box, pos + 3 * pairs[2 * p], pos + 3 * pairs[2 * p + 1], d);
        double r = sqrt(r2_of(d)), dsw;
        orc_switch(r / pair_r0[p], n, m, &dsw);
        double g = scale * dsw / (pair_r0[p] * r);
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) dsde[3 * a + b] += g * d[a] * d[b];
    }
}

/* s = |d| of the nearest pair: d s/d eps = d d^T / |d| (zero if nobody is within rc). */
void orc_cv_mindist_strain(int N, const double *pos, const double *box, const int *count, const int *list,
                           int maxn, const unsigned char *flags, double rc, double *dsde) {
    int pair[2];
    double s = orc_cv_mindist(N, pos, box, count, list, maxn, flags, rc, NULL, pair);
    for (int k = 0; k < 9; ++k) dsde[k] = 0.0;
    if (pair[0] < 0) return;
    double d[3];
    orc_delta(box, pos + 3 * pair[0], pos + 3 * pair[1], d);
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) dsde[3 * a + b] = d[a] * d[b] / s;
}

/* phi(b1, b2, b3): d phi/d eps = sum_k (d phi/d b_k) b_k^T with d phi/d b1 = -g_i, d phi/d b2 = -(g_i + g_j),
 * d phi/d b3 = g_l (g = the atom gradients of orc_cv_torsion, b1 = r_j - r_i, ...). */
void orc_cv_torsion_strain(const int *idx, const double *pos, const double *box, double *dsde) {
    double g[12], b[3][3];
    orc_cv_torsion(idx, pos, box, g);
    for (int k = 0; k < 3; ++k) orc_delta(box, pos + 3 * idx[k], pos + 3 * idx[k + 1], b[k]);
    for (int a = 0; a < 3; ++a)
        for (int c = 0; c < 3; ++c)
            dsde[3 * a + c] = -g[a] * b[0][c] - (g[a] + g[3 + a]) * b[1][c] + g[9 + a] * b[2][c];
}
