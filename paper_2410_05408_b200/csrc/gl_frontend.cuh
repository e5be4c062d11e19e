// gl_frontend.cuh -- NEXT-3 of SURVEY.md 8(f): the paper's SAMPLING parameters (App. A,
// PAPER.md:366-430) turned into the model rows the transit kernel takes, on the device, so that an
// MCMC caller can hand over walkers in the parametrisation the paper samples in.
//   (mu, nu) -> (f, eta): f_min = 1 - sqrt((mu + 1)/2) (A2), f = f_min + (1 - f_min) nu (A3), and A1,
//       mu = (f-1)^2 + f (f-2) cos 2 eta, solved for eta in [0, pi/2];
//   ln p(mu, nu) of eq. A6 (it makes p(f, eta) = cos eta, eq. A7);
//   mean radius r -> equatorial radius: R_eq = r / (1 - f)^(1/3) (volume-equivalent sphere, a b c =
//       R_eq^3 (1 - f); SURVEY.md ambiguity 22);
//   (q1, q2) -> (u1, u2) = (2 sqrt(q1) q2, sqrt(q1) (1 - 2 q2))   (Kipping's triangular map, as in
//       BASELINE.json config 3);
//   (u, w) uniform -> (mu, nu) ~ A6 by inverse-transform sampling (A10, A12).
// fp64 throughout: B rows of a dozen numbers, far off any roofline.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace glm {

// sampling row: t0, P, a/R*, b, e, omega, r_mean, mu, nu, xi, q1, q2
// model row:    t0, P, a/R*, b, e, omega, Rp_eq, f, xi, eta, u1, u2
__global__ void __launch_bounds__(128)
params_from_munu_kernel(const double* __restrict__ sampling, int B, double* __restrict__ params,
                        double* __restrict__ logprior) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= B) return;
    const double* s = sampling + (size_t)k * 12;
    double* p = params + (size_t)k * 12;
    const double r = s[6], mu = s[7], nu = s[8], q1 = s[10], q2 = s[11];
    bool ok = (r > 0.0) && (mu > -1.0) && (mu < 1.0) && (nu > 0.0) && (nu <= 1.0) && (q1 >= 0.0) &&
              (q1 <= 1.0) && (q2 >= 0.0) && (q2 <= 1.0);
    for (int j = 0; j < 12; ++j) ok = ok && isfinite(s[j]);
    const double nm1 = nu - 1.0, n2 = nu * (nu - 2.0);
    const double q = n2 * (mu * nm1 * nm1 + n2 - 1.0);   // eq. A6: p = 2^{-3/2} q^{-1/2}
    ok = ok && (q > 0.0);
    if (!ok) {
        for (int j = 0; j < 12; ++j) p[j] = NAN;
        if (logprior) logprior[k] = -INFINITY;
        return;
    }
    const double f_lo = 1.0 - sqrt(0.5 * (mu + 1.0));   // A2
    const double f = f_lo + (1.0 - f_lo) * nu;           // A3
    double c2 = (f > 0.0) ? (mu - (f - 1.0) * (f - 1.0)) / (f * (f - 2.0)) : 1.0;   // A1
    c2 = fmin(fmax(c2, -1.0), 1.0);
    const double sq = sqrt(q1);
    for (int j = 0; j < 6; ++j) p[j] = s[j];
    p[6] = r / cbrt(1.0 - f);
    p[7] = f;
    p[8] = s[9];
    p[9] = 0.5 * acos(c2);
    p[10] = 2.0 * sq * q2;
    p[11] = sq * (1.0 - 2.0 * q2);
    if (logprior) logprior[k] = -1.5 * 0.69314718055994530942 - 0.5 * log(q);
}

// uw [B, 2] uniform variates in [0, 1] -> munu [B, 2]
__global__ void __launch_bounds__(128)
munu_from_uniform_kernel(const double* __restrict__ uw, int B, double* __restrict__ munu) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= B) return;
    const double u = uw[2 * k], w = uw[2 * k + 1];
    const double nu = u * u / (u * u - 2.0 * u + 2.0);                 // A10
    const double s = sqrt(nu * (2.0 - nu)), d = (nu - 1.0) * (nu - 1.0);
    munu[2 * k] = (4.0 * w + 4.0 * (w * w - w) * s + 2.0 * (nu * (nu - 2.0) - 1.0) * w * w - d) / d;   // A12
    munu[2 * k + 1] = nu;
}

}  // namespace glm
