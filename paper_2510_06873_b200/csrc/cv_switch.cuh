// cv_switch.cuh — rational switching function shared by the coordination kernels (reading A).
#pragma once

// ------------------------------------------------------------------------------------------------
// switching function sw(x) = (1-x^n)/(1-x^m) and d sw/dx (reading A).  m == 2n -> 1/(1+x^n); else the quotient of the
// two geometric sums, which is the same function with the x = 1 limit built in.
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
    // general exponents: (1 - x^n) / (1 - x^m) = P_n(x) / P_m(x) with P_k(x) = 1 + x + ... + x^(k-1).  All terms are positive,
    // so nothing cancels near x = 1 (the quotient of the two differences loses every digit of sw' there in fp32: with
    // |x - 1| = 1e-3 the numerator of sw' is a difference of order 1e-6 between terms of order 1e-2), and the limit
    // n / m with slope n (n - m) / 2m of reading A comes out of the same expression.  P_k and P_k' by one Horner sweep.
    T p = T(1), dp = T(0), pn = T(1), dpn = T(0), pm = T(1), dpm = T(0);
    const int top = n > m ? n : m;
    for (int j = 1; j < top; ++j) {
        dp = dp * x + p;
        p = p * x + T(1);
        if (j == n - 1) { pn = p; dpn = dp; }
        if (j == m - 1) { pm = p; dpm = dp; }
    }
    const T inv = T(1) / pm;
    dsw = (dpn * pm - pn * dpm) * inv * inv;
    return pn * inv;
}

