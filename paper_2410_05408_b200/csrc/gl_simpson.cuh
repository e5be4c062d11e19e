// gl_simpson.cuh -- NEXT-1 of SURVEY.md 8(f): the PAPER'S OWN algorithm for steps a3 + a4, as a kernel.
//
// PAPER.md:108-125 (eqs. 16-20): a point of the outline that falls outside the stellar disc is
// "snapped" radially onto the limb, lambda = atan(y_e / x_e), (x_d, y_d) = (cos, sin) lambda, with
// d(lambda)/d(theta) = (-y_e x_e' + x_e y_e') / (x_e^2 + y_e^2) carrying the parametrisation -- no
// intersection is ever solved.  PAPER.md:127-135 (eqs. 21-23): the three integrands.  PAPER.md:147:
// "numerically summed" over theta in [0, 2 pi] with Simpson's rule, and PAPER.md:149: the sum is
// spread over a group of work items ("hierarchical parallelism").  Here: one WARP per geometry,
// lanes stride over the Simpson nodes, fixed xor-tree reduction.
//
// It exists to be MEASURED beside the production kernel on the same box (accuracy versus node
// count, and time), and as a third route to the same numbers; it shares the row format and the
// validity rules of gl_flux_geometry.  The outline is parametrised exactly as the paper does
// (eqs. 7-8 with the Cholesky amplitudes of eqs. 11-13), so that it can be compared node for node
// with the oracle's transcription of the same algorithm.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace gls {

template <typename T> struct trig;
template <> struct trig<float> {
    static __device__ __forceinline__ void sincos2pi(float u, float* s, float* c) { sincospif(2.f * u, s, c); }
    static __device__ __forceinline__ float rsq(float x) { return rsqrtf(x); }
    static __device__ __forceinline__ float root(float x) { return sqrtf(x); }
};
template <> struct trig<double> {
    static __device__ __forceinline__ void sincos2pi(double u, double* s, double* c) { sincospi(2.0 * u, s, c); }
    static __device__ __forceinline__ double rsq(double x) { return rsqrt(x); }
    static __device__ __forceinline__ double root(double x) { return sqrt(x); }
};

// The three integrands of eqs. 21-23 at one (possibly snapped) node, times the Simpson weight w.
// r^2 of a node, on which the snap decision r^2 > 1 hangs.  The integrand of eq. 23 is discontinuous across
// the snap, so a node within rounding of the limb (a tangent outline) must be judged with the SAME arithmetic
// by everyone who evaluates the definition: in fp64 plain IEEE products and sums in the written order, no
// contraction into FMAs (fp32 is a different precision anyway: its nodes may flip).
__device__ __forceinline__ float node_r2(float x, float y) { return x * x + y * y; }
__device__ __forceinline__ double node_r2(double x, double y) { return __dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)); }

template <typename T>
__device__ __forceinline__ void add_node(T x, T y, T xp, T yp, T w, T* acc) {
    T r2 = node_r2(x, y);
    if (r2 > T(1)) {
        // eqs. 16-19: snap radially onto the limb; cos(lambda) = x / r, sin(lambda) = y / r
        const T dlam = (x * yp - y * xp) / r2;
        const T ir = trig<T>::rsq(r2);
        x *= ir;
        y *= ir;
        xp = -y * dlam;
        yp = x * dlam;
        r2 = T(1);
    }
    const T fflat = T(0.5) * (x * yp - y * xp);                              // eq. 21
    const T m2 = T(1) - r2 > T(0) ? T(1) - r2 : T(0);                        // R11
    const T m = trig<T>::root(m2);
    const T W = T(1) + m2 / (T(1) + m);   // [1 - (1 - r^2)^{3/2}] / r^2 without the 0/0 at r = 0 (R9)
    const T flin = (T(2) / T(3)) * W * fflat;                                // eq. 22
    const T x2 = x * x, y2 = y * y;
    const T fquad = T(0.5) * (x * (x2 * (T(1) / T(3)) + y2) * yp - y * (x2 + y2 * (T(1) / T(3))) * xp);   // eq. 23
    acc[0] += w * fflat;
    acc[1] += w * flin;
    acc[2] += w * fquad;
}

// One warp per row of geom (d, Rp, f_proj, PA, u1, u2); n_int = number of Simpson intervals (even).
template <typename T>
__global__ void __launch_bounds__(128)
simpson_kernel(const double* __restrict__ geom, long long N, int n_int, T* __restrict__ out) {
    const long long row = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (row >= N) return;   // whole warps leave together
    const double* g = geom + row * 6;
    const double d = g[0], Rp = g[1], fp = g[2], pa = g[3], u1 = g[4], u2 = g[5];
    const double norm = 1.0 - u1 / 3.0 - u2 / 6.0;
    const bool ok = isfinite(d) && isfinite(Rp) && isfinite(fp) && isfinite(pa) && isfinite(u1) &&
                    isfinite(u2) && (d >= 0.0) && (Rp > 0.0) && (Rp < 0.5) && (fp >= 0.0) &&
                    (fp < 1.0) && (norm > 0.0);
    if (!ok) {
        if (lane == 0) out[row] = T(NAN);
        return;
    }
    // eqs. 11-13 for a flat ellipse: (dx, dy1, dy2) = lower-Cholesky factor of its covariance
    const double a = Rp, b = Rp * (1.0 - fp);
    double sp, cp;
    sincos(pa, &sp, &cp);
    const double dxd = sqrt(a * a * cp * cp + b * b * sp * sp);
    const T x0 = T(d), dx = T(dxd), dy1 = T((a * a - b * b) * cp * sp / dxd), dy2 = T(a * b / dxd);
    T acc[3] = {T(0), T(0), T(0)};
    const T inv_n = T(1) / T(n_int);
    // composite Simpson on the closed contour: node 0 = node n_int carries weight 1 + 1 = 2
    for (int k = lane; k < n_int; k += 32) {
        T s, c, x, y;
        if (sizeof(T) == 8) {
            // fp64 (validation path): theta_k = k h with h = 2 pi / n as the definition writes it (at a tangent
            // node the last bit of sin(theta_k) decides the snap: sin(pi) must be 1.2e-16, not sinpi(1) = 0),
            // and eqs. 7-8 in plain IEEE operations in the written order (see node_r2)
            const double h = 2.0 * 3.14159265358979323846 / (double)n_int;
            double sd, cd;
            sincos((double)k * h, &sd, &cd);
            s = (T)sd;
            c = (T)cd;
            x = (T)__dadd_rn((double)x0, __dmul_rn((double)dx, cd));
            y = (T)__dadd_rn(__dmul_rn((double)dy1, cd), __dmul_rn((double)dy2, sd));
        } else {
            trig<T>::sincos2pi(T(k) * inv_n, &s, &c);
            x = x0 + dx * c;                                    // eqs. 7-8
            y = dy1 * c + dy2 * s;
        }
        const T xp = -dx * s, yp = dy2 * c - dy1 * s;           // eqs. 14-15
        add_node<T>(x, y, xp, yp, (k & 1) ? T(4) : T(2), acc);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        acc[0] += __shfl_xor_sync(0xffffffffu, acc[0], off);
        acc[1] += __shfl_xor_sync(0xffffffffu, acc[1], off);
        acc[2] += __shfl_xor_sync(0xffffffffu, acc[2], off);
    }
    if (lane == 0) {
        const double h3 = 6.28318530717958647692 / (3.0 * (double)n_int);
        const double pn = 3.14159265358979323846 * norm;
        const double delta = ((1.0 - u1 - 2.0 * u2) * (double)acc[0] + (u1 + 2.0 * u2) * (double)acc[1] +
                              u2 * (double)acc[2]) * h3 / pn;
        out[row] = T(1.0 - delta);
    }
}

}  // namespace gls
