// gl_gp.cuh -- NEXT-4 of SURVEY.md 8(f): the paper's actual objective, a Gaussian-process likelihood of
// the residuals: covariance = Matern-3/2 kernel + diagonal "jitter",
//   K_ij = s^2 (1 + sqrt(3) |t_i - t_j| / rho) exp(-sqrt(3) |t_i - t_j| / rho) + delta_ij (sigma_i^2 + jit^2),
//   ln L = -1/2 r^T K^-1 r - 1/2 ln det K - (T/2) ln 2 pi,      r_i = obs_i - F(t_i).
// The paper evaluates it with celerite's O(T) semiseparable solver; here the SAME likelihood is
// computed exactly, also in O(T), from the state-space form of the Matern-3/2 process (a 2-state
// linear stochastic differential equation, Hartikainen & Sarkka 2010): with lambda = sqrt(3)/rho and
// state (f, f'),
//   stationary covariance  Pinf = diag(s^2, lambda^2 s^2),
//   transition over dt     A = exp(-lambda dt) [[1 + lambda dt, dt], [-lambda^2 dt, 1 - lambda dt]],
//   process noise          Q = Pinf - A Pinf A^T,
// and a Kalman filter over the sorted series gives the innovations v_i and their variances S_i:
//   ln L = -1/2 sum_i (v_i^2 / S_i + ln S_i + ln 2 pi).
// This header holds what the likelihood kernels share (the process noise in closed form); the kernel is
// gl_gp_scan.cuh (parallel in time).  The plain one-thread-per-walker filter it is checked against lives
// with the tests (tests/gp_serial_harness.cu).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace glg {

// Process noise of the Matern-3/2 state-space model over a step x = lambda dt, in closed form:
//   Q = Pinf - A Pinf A^T,   q00 = s^2 [1 - e^{-2x} (1 + 2x + 2x^2)],   q01 = 2 s^2 lambda x^2 e^{-2x},
//   q11 = s^2 lambda^2 [1 - e^{-2x} (1 - 2x + 2x^2)].
// Formed from the matrices, q00 = O(x^3) comes out of O(1) terms (relative error eps / x^3: 1e-3 for a
// 5-second cadence against a 2-day timescale); here 1 - e^{-2x}(1 + 2x + 2x^2) = e^{-2x} sum_{k>=3}
// (2x)^k / k! is summed as a series for small x.  e2 = e^{-2x}.
__device__ __forceinline__ void matern32_q(double x, double e2, double p0, double lam, double* q00,
                                           double* q01, double* q11) {
    double g0;
    if (x < 0.5) {
        const double y = 2.0 * x;   // sum_{k=3}^{20} y^k / k!  (y < 1: last term < 1e-19)
        double t = 0.0;
        for (int k = 20; k >= 3; --k) t = (t + 1.0) * y / (double)k;   // Horner from the tail
        // t = y/3 (1 + y/4 (1 + ...)): multiply by y^2 / 2 to restore the first two factors
        g0 = e2 * t * y * y * 0.5;
    } else {
        g0 = 1.0 - e2 * (1.0 + 2.0 * x + 2.0 * x * x);
    }
    *q00 = p0 * g0;
    *q01 = 2.0 * p0 * lam * x * x * e2;
    // 1 - e^{-2x}(1 - 2x + 2x^2) = g0 + 4 x e^{-2x}: no cancellation
    *q11 = p0 * lam * lam * (g0 + 4.0 * x * e2);
}

}  // namespace glg
