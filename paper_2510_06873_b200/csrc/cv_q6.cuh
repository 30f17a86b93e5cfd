// cv_q6.cuh — device math for the l=6 Steinhardt order parameter.
//
// With u = d/|d| = (x,y,z):  Y6m(u) = N_m P6^(m)(z) (x+iy)^m,  P6^(m) = m-th derivative of the
// Legendre polynomial P6, N_m^2 = (13/4pi)(6-m)!/(6+m)!.  Folding 4pi/13, the m<0 mirror weight
// (w_0=1, w_m=2) and N_m into the polynomials gives  E_m(z) = sqrt(w_m (6-m)!/(6+m)!) P6^(m)(z)  and
//     S_i = n_i^2 q6_i^2 = sum_{m=0..6} | sum_j E_m(z_ij) (x_ij + i y_ij)^m |^2 .
// dE_m/dz = rho_m E_{m+1} with rho_m = sqrt((6-m)(7+m) w_m/w_{m+1}) = sqrt(21,40,36,30,22,12).
#pragma once

template <typename T>
struct Y6 {
    T E[7];   // E_m(z)
    T c[7];   // Re (x+iy)^m
    T s[7];   // Im (x+iy)^m
};

template <typename T>
__device__ __forceinline__ void y6_eval(T x, T y, T z, Y6<T> &o) {
    const T t = z * z;
    // Horner forms with the prefactors folded into the coefficients (13 instead of 18 operations per direction):
    //   E0 = (231 t^3 - 315 t^2 + 105 t - 5)/16,            E1 = 0.57282196186948 z (33 t^2 - 30 t + 5),
    //   E2 = 0.45285552331841994 (33 t^2 - 18 t + 1),        E3 = 0.9057110466368399 z (11 t - 3),
    //   E4 = 0.4960783708246107 (11 t - 1)
    o.E[0] = ((T(14.4375) * t - T(19.6875)) * t + T(6.5625)) * t - T(0.3125);
    o.E[1] = z * ((T(18.90312474169284) * t - T(17.1846588560844)) * t + T(2.8641098093474));
    o.E[2] = (T(14.944232269507857) * t - T(8.15139941973156)) * t + T(0.45285552331841994);
    o.E[3] = z * (T(9.962821513005238) * t - T(2.7171331399105196));
    o.E[4] = T(5.456862079070718) * t - T(0.4960783708246107);
    o.E[5] = T(2.3268138086232857) * z;
    o.E[6] = T(0.6716932893813962);
    o.c[0] = T(1); o.s[0] = T(0);
    o.c[1] = x;    o.s[1] = y;
#pragma unroll
    for (int m = 2; m <= 6; ++m) {
        o.c[m] = o.c[m - 1] * x - o.s[m - 1] * y;
        o.s[m] = o.s[m - 1] * x + o.c[m - 1] * y;
    }
}

// gradient with respect to the (unconstrained) unit-vector components of
//   f(u) = sum_m E_m(z) (br_m c_m - bi_m s_m),   b = (br0, br1, bi1, ..., br6, bi6)
template <typename T>
__device__ __forceinline__ void y6_grad(const Y6<T> &o, const T *b, T &gx, T &gy, T &gz) {
    const T rho[6] = { T(4.58257569495584), T(6.324555320336759), T(6.0), T(5.477225575051661),
                       T(4.69041575982343), T(3.4641016151377544) };
    gz = rho[0] * o.E[1] * b[0];
    gx = T(0); gy = T(0);
#pragma unroll
    for (int m = 1; m <= 6; ++m) {
        const T br = b[2 * m - 1], bi = b[2 * m];
        if (m < 6) gz += rho[m] * o.E[m + 1] * (br * o.c[m] - bi * o.s[m]);
        const T em = T(m) * o.E[m];
        gx += em * (br * o.c[m - 1] - bi * o.s[m - 1]);
        gy -= em * (br * o.s[m - 1] + bi * o.c[m - 1]);
    }
}
