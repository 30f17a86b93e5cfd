/* gen.c — seeded synthetic input generators (compiled helper of paper_2510_06873_b200.inputs).
 *
 * Holds NONE of the method's arithmetic (no switching function, no Q6, no bias): only the
 * geometric placement that numpy would be too slow for — random sequential addition (RSA) of
 * points with a minimum separation inside a periodic (possibly triclinic) box.  Used to make
 * the "random liquid" of BASELINE.json configs 3/4 and the water oxygens of config 2.
 * Both the oracle tests and the CUDA tests/bench read the SAME arrays produced here.
 *
 * Box convention (same as the library): rows a=(ax,0,0), b=(bx,by,0), c=(cx,cy,cz).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint64_t s; } rng_t;

static uint64_t rng_next(rng_t *r) { /* splitmix64 */
    uint64_t z = (r->s += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static double rng_uni(rng_t *r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }

/* fractional -> cartesian for a lower-triangular row box */
static void frac2cart(const double *box, const double *s, double *r) {
    r[0] = s[0] * box[0] + s[1] * box[3] + s[2] * box[6];
    r[1] = s[1] * box[4] + s[2] * box[7];
    r[2] = s[2] * box[8];
}
static void cart2frac(const double *box, const double *r, double *s) {
    s[2] = r[2] / box[8];
    s[1] = (r[1] - s[2] * box[7]) / box[4];
    s[0] = (r[0] - s[1] * box[3] - s[2] * box[6]) / box[0];
}

/* Random sequential addition.
 *  n_new        points to place
 *  box[9]       lower-triangular row box
 *  periodic[3]  1 = wrap along that lattice direction
 *  flo/fhi[3]   fractional sub-region new points are drawn from (uniform in fractional coordinates)
 *  sph_c[3],sph_r   new points are rejected if inside this sphere (cartesian; sph_r<=0: no sphere)
 *  min_sep      minimum distance to every other point (existing and new), periodic images included
 *  existing     n_existing*3 cartesian positions already present (must lie in the primary cell)
 *  out          n_new*3 cartesian positions
 * returns the number actually placed (== n_new unless max_trials total draws were used up).
 */
long gen_rsa(long n_new, const double *box, const int *periodic, const double *flo, const double *fhi,
             const double *sph_c, double sph_r, double min_sep, const double *existing, long n_existing,
             uint64_t seed, double *out, long max_trials) {
    rng_t rng = { seed };
    double vol = box[0] * box[4] * box[8];
    /* perpendicular widths of the three lattice directions */
    double bxc[3] = { box[4] * box[8], -(box[3] * box[8]), box[3] * box[7] - box[4] * box[6] };
    double cxa[3] = { 0.0, box[8] * box[0], -(box[7] * box[0]) };
    double wa = vol / sqrt(bxc[0] * bxc[0] + bxc[1] * bxc[1] + bxc[2] * bxc[2]);
    double wb = vol / sqrt(cxa[0] * cxa[0] + cxa[1] * cxa[1] + cxa[2] * cxa[2]);
    double wc = box[8];
    double w[3] = { wa, wb, wc };
    int nc[3];
    for (int d = 0; d < 3; ++d) {
        nc[d] = (int)floor(w[d] / min_sep);
        if (nc[d] < 1) nc[d] = 1;
        if (nc[d] > 400) nc[d] = 400;
    }
    long ncell = (long)nc[0] * nc[1] * nc[2];
    long ntot = n_existing + n_new;
    int *head = (int *)malloc(sizeof(int) * ncell);
    int *next = (int *)malloc(sizeof(int) * (ntot > 0 ? ntot : 1));
    double *fr = (double *)malloc(sizeof(double) * 3 * (ntot > 0 ? ntot : 1));
    for (long c = 0; c < ncell; ++c) head[c] = -1;
    long np = 0;
    for (long i = 0; i < n_existing; ++i) {
        double s[3];
        cart2frac(box, existing + 3 * i, s);
        int ic[3];
        for (int d = 0; d < 3; ++d) {
            s[d] -= floor(s[d]);
            ic[d] = (int)(s[d] * nc[d]);
            if (ic[d] >= nc[d]) ic[d] = nc[d] - 1;
        }
        long c = ((long)ic[2] * nc[1] + ic[1]) * nc[0] + ic[0];
        fr[3 * np] = s[0]; fr[3 * np + 1] = s[1]; fr[3 * np + 2] = s[2];
        next[np] = head[c]; head[c] = (int)np; ++np;
    }
    double ms2 = min_sep * min_sep;
    long placed = 0, trials = 0;
    while (placed < n_new && trials < max_trials) {
        ++trials;
        double s[3], r[3];
        for (int d = 0; d < 3; ++d) s[d] = flo[d] + (fhi[d] - flo[d]) * rng_uni(&rng);
        frac2cart(box, s, r);
        if (sph_r > 0.0) {
            double dx = r[0] - sph_c[0], dy = r[1] - sph_c[1], dz = r[2] - sph_c[2];
            if (dx * dx + dy * dy + dz * dz < sph_r * sph_r) continue;
        }
        int ic[3];
        for (int d = 0; d < 3; ++d) {
            ic[d] = (int)(s[d] * nc[d]);
            if (ic[d] >= nc[d]) ic[d] = nc[d] - 1;
            if (ic[d] < 0) ic[d] = 0;
        }
        int ok = 1;
        for (int oz = -1; oz <= 1 && ok; ++oz)
        for (int oy = -1; oy <= 1 && ok; ++oy)
        for (int ox = -1; ox <= 1 && ok; ++ox) {
            int o[3] = { ox, oy, oz }, jc[3], skip = 0;
            for (int d = 0; d < 3; ++d) {
                jc[d] = ic[d] + o[d];
                if (jc[d] < 0 || jc[d] >= nc[d]) {
                    if (!periodic[d]) { skip = 1; break; }
                    jc[d] = (jc[d] + nc[d]) % nc[d];
                }
                /* with <3 cells an offset can alias a cell already visited: harmless (re-check) */
            }
            if (skip) continue;
            long c = ((long)jc[2] * nc[1] + jc[1]) * nc[0] + jc[0];
            for (int j = head[c]; j >= 0; j = next[j]) {
                double df[3], dc[3];
                for (int d = 0; d < 3; ++d) {
                    df[d] = fr[3 * j + d] - s[d];
                    if (periodic[d]) df[d] -= floor(df[d] + 0.5);
                }
                frac2cart(box, df, dc);
                if (dc[0] * dc[0] + dc[1] * dc[1] + dc[2] * dc[2] < ms2) { ok = 0; break; }
            }
        }
        if (!ok) continue;
        long c = ((long)ic[2] * nc[1] + ic[1]) * nc[0] + ic[0];
        fr[3 * np] = s[0]; fr[3 * np + 1] = s[1]; fr[3 * np + 2] = s[2];
        next[np] = head[c]; head[c] = (int)np; ++np;
        out[3 * placed] = r[0]; out[3 * placed + 1] = r[1]; out[3 * placed + 2] = r[2];
        ++placed;
    }
    free(head); free(next); free(fr);
    return placed;
}
