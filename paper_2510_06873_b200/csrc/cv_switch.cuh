// cv_switch.cuh — rational switching function shared by the coordination kernels (reading A).
#pragma once

// ------------------------------------------------------------------------------------------------
// switching function sw(x) = (1-x^n)/(1-x^m) and d sw/dx (reading A).  m == 2n -> 1/(1+x^n).
template <typename T>
__device__ __forceinline__ T ipow(T x, int n) {
    T r = T(1);                                   // square and multiply: log2(n) steps instead of n
    while (n > 0) {
        if (n & 1) r *= x;
        x *= x;
        n >>= 1;
    }
    return r;
}
template <typename T>
__device__ __forceinline__ T switch_fn(T x, int n, int m, T &dsw) {
    if (m == 2 * n) {
        T xn1 = ipow(x, n - 1), xn = xn1 * x;
        T inv = T(1) / (T(1) + xn);
        dsw = -T(n) * xn1 * inv * inv;
        return inv;
    }
    T e = x - T(1);
    if (fabs((double)e) < 1e-6) {
        T s0 = T(n) / T(m), s1 = T(n) * T(n - m) / (T(2) * T(m));
        dsw = s1;
        return s0 + s1 * e;
    }
    T xn1 = ipow(x, n - 1), xm1 = ipow(x, m - 1);
    T num = T(1) - xn1 * x, den = T(1) - xm1 * x;
    T f = num / den;
    dsw = (-T(n) * xn1 * den + num * T(m) * xm1) / (den * den);
    return f;
}

