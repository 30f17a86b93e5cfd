// cv_torsion.cuh — torsion (dihedral) angle and its gradient for the four atoms i-j-k-l (NEXT-1:
// PAPER.md:37 "Phi(C-N-Ca-C) and Psi(N-Ca-C-N) serve as the CVs"; reading V).
// IUPAC sign: b1 = r_j - r_i, b2 = r_k - r_j, b3 = r_l - r_k, n1 = b1 x b2, n2 = b2 x b3,
//     phi = atan2(|b2| b1.n2, n1.n2),
// gradient in the bond-vector form (p = b1.b2/|b2|^2, q = b3.b2/|b2|^2):
//     g_i = -|b2|/|n1|^2 n1,  g_l = |b2|/|n2|^2 n2,  g_j = -(1+p) g_i + q g_l,  g_k = p g_i - (1+q) g_l.
#pragma once
#include <math.h>

#ifdef __CUDACC__
#define TORS_HD __host__ __device__ __forceinline__
#else
#define TORS_HD inline
#endif

// b1, b2, b3: minimum-image bond vectors; g: [4][3] (i, j, k, l)
TORS_HD double torsion_eval(const double *b1, const double *b2, const double *b3, double *g) {
    const double n1[3] = { b1[1] * b2[2] - b1[2] * b2[1], b1[2] * b2[0] - b1[0] * b2[2], b1[0] * b2[1] - b1[1] * b2[0] };
    const double n2[3] = { b2[1] * b3[2] - b2[2] * b3[1], b2[2] * b3[0] - b2[0] * b3[2], b2[0] * b3[1] - b2[1] * b3[0] };
    const double l2 = b2[0] * b2[0] + b2[1] * b2[1] + b2[2] * b2[2], l = sqrt(l2);
    const double y = l * (b1[0] * n2[0] + b1[1] * n2[1] + b1[2] * n2[2]);
    const double x = n1[0] * n2[0] + n1[1] * n2[1] + n1[2] * n2[2];
    if (g) {
        const double ci = -l / (n1[0] * n1[0] + n1[1] * n1[1] + n1[2] * n1[2]);
        const double cl = l / (n2[0] * n2[0] + n2[1] * n2[1] + n2[2] * n2[2]);
        const double p = (b1[0] * b2[0] + b1[1] * b2[1] + b1[2] * b2[2]) / l2;
        const double q = (b3[0] * b2[0] + b3[1] * b2[1] + b3[2] * b2[2]) / l2;
        for (int a = 0; a < 3; ++a) {
            const double gi = ci * n1[a], gl = cl * n2[a];
            g[a] = gi;
            g[3 + a] = -(1.0 + p) * gi + q * gl;
            g[6 + a] = p * gi - (1.0 + q) * gl;
            g[9 + a] = gl;
        }
    }
    return atan2(y, x);
}
