// gl_tables.h -- HOST-side generator of the quadrature tables the kernels read from constant
// memory.  Computed at library load, never transcribed.  (The oracle has its own generator in its
// own file; the two share nothing.)
//
// For an N-point Gauss-Legendre rule on z in [-1, 1] (N even) and the end-point-smoothing map
//     phi(z) = (3 z - z^3) / 2,   phi'(z) = 1.5 (1 - z^2)
// the kernels need, for the N/2 positive nodes only (the rule is symmetric):
//     qphi[k] = phi(z_k),   qom[k] = w_k * phi'(z_k).
#pragma once
#include <cmath>

namespace glt {

// Legendre P_n(z) and P_{n-1}(z) by Bonnet's recurrence, in long double.
inline void legendre_pair(int n, long double z, long double* pn, long double* pnm1) {
    long double pm = 1.0L, p = z;
    for (int j = 1; j < n; ++j) {
        const long double nx = ((2 * j + 1) * z * p - j * pm) / (j + 1);
        pm = p;
        p = nx;
    }
    *pn = p;
    *pnm1 = pm;
}

// Fills qphi[0..n/2) and qom[0..n/2) (positive nodes, ascending).  n must be even.
template <typename T> inline void smoothed_gauss_legendre(int n, T* qphi, T* qom) {
    const long double PI = 3.141592653589793238462643383279502884L;
    const int half = n / 2;
    for (int k = 0; k < half; ++k) {
        // k-th positive root, counted from the centre; Tricomi-type starting value
        const int idx = half - k;   // 1 = largest root
        long double z = cosl(PI * (idx - 0.25L) / (n + 0.5L));
        long double dp = 1.0L;
        for (int it = 0; it < 60; ++it) {
            long double pn, pm;
            legendre_pair(n, z, &pn, &pm);
            dp = n * (pm - z * pn) / (1.0L - z * z);   // P_n'(z)
            const long double step = pn / dp;
            z -= step;
            if (fabsl(step) < 1e-19L) break;
        }
        long double pn, pm;
        legendre_pair(n, z, &pn, &pm);
        dp = n * (pm - z * pn) / (1.0L - z * z);
        const long double w = 2.0L / ((1.0L - z * z) * dp * dp);
        qphi[k] = static_cast<T>(0.5L * z * (3.0L - z * z));
        qom[k] = static_cast<T>(w * 1.5L * (1.0L - z * z));
    }
}

}  // namespace glt
