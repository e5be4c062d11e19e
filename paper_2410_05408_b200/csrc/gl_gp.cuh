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
// One thread per walker, fp64, sequential in time: a LATENCY-bound first version.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace glg {

// flux [B, T] (float or double), gp [B, 3] = (s, rho, jit), times sorted ascending.
template <typename T>
__global__ void __launch_bounds__(32)
gp_kernel(const T* __restrict__ flux, int B, const double* __restrict__ times, int nT,
          const double* __restrict__ obs, const double* __restrict__ sigma,
          const double* __restrict__ gp, double* __restrict__ out) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    const double s = gp[3 * b], rho = gp[3 * b + 1], jit = gp[3 * b + 2];
    if (!(s >= 0.0) || !(rho > 0.0) || !(jit >= 0.0) || !isfinite(s) || !isfinite(rho) || !isfinite(jit)) {
        out[b] = NAN;
        return;
    }
    const T* frow = flux + (size_t)b * nT;
    const double lam = 1.7320508075688772935 / rho;
    const double p0 = s * s, p1 = lam * lam * p0;   // Pinf = diag(p0, p1)
    double m0 = 0.0, m1 = 0.0, P00 = p0, P01 = 0.0, P11 = p1;
    double a00 = 1.0, a01 = 0.0, a10 = 0.0, a11 = 1.0, q00 = 0.0, q01 = 0.0, q11 = 0.0;
    double quad = 0.0, logdet = 0.0, prod = 1.0, tprev = 0.0, dtprev = -1.0;
    bool bad = false, invalid_walker = false;
    for (int i = 0; i < nT; ++i) {
        const double t = times[i];
        if (i > 0) {
            const double dt = t - tprev;
            if (dt < 0.0) bad = true;   // the series must be sorted
            if (dt != dtprev) {         // a uniform cadence pays for exp() once
                const double e = exp(-lam * dt), ld = lam * dt;
                a00 = e * (1.0 + ld);
                a01 = e * dt;
                a10 = -e * lam * lam * dt;
                a11 = e * (1.0 - ld);
                // Q = Pinf - A Pinf A^T
                q00 = p0 - (a00 * a00 * p0 + a01 * a01 * p1);
                q01 = -(a00 * a10 * p0 + a01 * a11 * p1);
                q11 = p1 - (a10 * a10 * p0 + a11 * a11 * p1);
                dtprev = dt;
            }
            // predict: m = A m, P = A P A^T + Q
            const double n0 = a00 * m0 + a01 * m1, n1 = a10 * m0 + a11 * m1;
            const double b00 = a00 * P00 + a01 * P01, b01 = a00 * P01 + a01 * P11;
            const double b10 = a10 * P00 + a11 * P01, b11 = a10 * P01 + a11 * P11;
            m0 = n0;
            m1 = n1;
            P00 = b00 * a00 + b01 * a01 + q00;
            P01 = b00 * a10 + b01 * a11 + q01;
            P11 = b10 * a10 + b11 * a11 + q11;
        }
        tprev = t;
        // update with r_i = obs_i - F_i, observation noise sigma_i^2 + jit^2
        const double sg = sigma[i];
        const double fi = (double)frow[i];
        if (fi != fi) invalid_walker = true;   // NaN row = out-of-domain walker
        const double r = obs[i] - fi;
        const double S = P00 + sg * sg + jit * jit;
        if (!(S > 0.0) || !(sg >= 0.0)) bad = true;
        const double v = r - m0, iS = 1.0 / S;
        quad += v * v * iS;
        prod *= S;
        if ((i & 7) == 7) {   // ln det K = sum ln S_i, eight factors per logarithm
            logdet += log(prod);
            prod = 1.0;
        }
        const double k0 = P00 * iS, k1 = P01 * iS;
        m0 += k0 * v;
        m1 += k1 * v;
        P11 -= k1 * P01;
        P01 -= k1 * P00;
        P00 -= k0 * P00;
    }
    logdet += log(prod);
    const double ll = -0.5 * (quad + logdet + (double)nT * 1.8378770664093454836);
    out[b] = invalid_walker ? -INFINITY : ((bad || !isfinite(ll)) ? NAN : ll);
}

}  // namespace glg
