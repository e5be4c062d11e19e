// gp_serial_harness.cu -- TEST INFRASTRUCTURE: the plain Kalman-filter likelihood of the Matern-3/2 +
// jitter process, one thread per walker, sequential in time.  The product computes
// the same number with a parallel-in-time scan (csrc/gl_gp_scan.cuh); tests/test_gpu_parity.py builds
// this file with nvcc and checks the two against each other (and both against the dense definition of
// the oracle).  Not part of the library.
#include <cuda_runtime.h>
#include <math.h>

#include "../paper_2410_05408_b200/csrc/gl_gp.cuh"

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
    // steady state of the covariance recursion (see the loop): cached gains and innovation variance
    bool steady = false;
    double sgprev = -1.0, S_c = 1.0, iS_c = 1.0, k0_c = 0.0, k1_c = 0.0, lnS_c = 0.0;
    double P00s = 0.0, P01s = 0.0, P11s = 0.0;   // predicted covariance in the steady state
    int nsteady = 0;
    // The recursion is a serial dependent chain per walker; what can be taken off it are the memory
    // round trips: the inputs of CH steps are loaded in one batch, then the CH steps run from registers.
    constexpr int CH = 8;
    for (int i0 = 0; i0 < nT; i0 += CH) {
        double tv[CH], sv[CH], rv[CH];
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const int i = min(i0 + c, nT - 1);
            tv[c] = times[i];
            sv[c] = sigma[i];
            const double fi = (double)frow[i];
            if (fi != fi) invalid_walker = true;   // NaN row = out-of-domain walker
            rv[c] = obs[i] - fi;
        }
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            const int i = i0 + c;
            if (i >= nT) break;
            const double t = tv[c], sg = sv[c];
            const double dt = (i > 0) ? t - tprev : 0.0;
            tprev = t;
            if (dt < 0.0) bad = true;   // the series must be sorted
            // time stamps i * cadence carry rounding noise: steps equal to 1e-9 relative share one
            // transition matrix (an error of <= 1e-9 lambda dt in one exponent: ~1e-12 on ln L)
            const bool same_dt = fabs(dt - dtprev) <= 1e-9 * dtprev;
            if (steady && same_dt && sg == sgprev) {
                // Uniform cadence and equal error bars: the covariance recursion (a Riccati map that
                // does not see the data) has reached its fixed point, so P, S and the gain repeat and
                // only the mean has to be advanced -- a 3-deep chain instead of ~20.
                const double n0 = a00 * m0 + a01 * m1, n1 = a10 * m0 + a11 * m1;
                const double v = rv[c] - n0;
                quad += v * v * iS_c;
                m0 = n0 + k0_c * v;
                m1 = n1 + k1_c * v;
                ++nsteady;
                continue;
            }
            if (steady) {   // leaving the steady state: restore the posterior covariance it stood for
                P11 = P11s - k1_c * P01s;
                P01 = P01s - k1_c * P00s;
                P00 = P00s - k0_c * P00s;
                steady = false;
            }
            const bool same = (i > 1) && same_dt && sg == sgprev;
            const double o00 = P00, o01 = P01, o11 = P11;   // posterior of the previous step
            if (i > 0) {
                if (!same_dt) {             // a uniform cadence pays for exp() once
                    const double e = exp(-lam * dt), ld = lam * dt;
                    a00 = e * (1.0 + ld);
                    a01 = e * dt;
                    a10 = -e * lam * lam * dt;
                    a11 = e * (1.0 - ld);
                    matern32_q(ld, e * e, p0, lam, &q00, &q01, &q11);   // Q = Pinf - A Pinf A^T
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
            sgprev = sg;
            // update with r_i = obs_i - F_i, observation noise sigma_i^2 + jit^2
            const double S = P00 + sg * sg + jit * jit;
            if (!(S > 0.0) || !(sg >= 0.0)) bad = true;
            const double v = rv[c] - m0, iS = 1.0 / S;
            quad += v * v * iS;
            prod *= S;
            const double k0 = P00 * iS, k1 = P01 * iS;
            const double pp00 = P00, pp01 = P01, pp11 = P11;   // predicted covariance of this step
            m0 += k0 * v;
            m1 += k1 * v;
            P11 -= k1 * P01;
            P01 -= k1 * P00;
            P00 -= k0 * P00;
            // fixed point reached?  (same dt and sigma as the step before, posterior unchanged to 1e-13: ln L moves by < T 1e-13)
            if (same && fabs(P00 - o00) <= 1e-13 * fabs(P00) && fabs(P01 - o01) <= 1e-13 * fabs(P00) * lam &&
                fabs(P11 - o11) <= 1e-13 * fabs(P11)) {
                steady = true;
                S_c = S;
                iS_c = iS;
                k0_c = k0;
                k1_c = k1;
                P00s = pp00;
                P01s = pp01;
                P11s = pp11;
                if (nsteady) logdet += (double)nsteady * lnS_c;   // a previous steady stretch
                nsteady = 0;
                lnS_c = log(S);
            }
        }
        logdet += log(prod);   // ln det K = sum ln S_i, CH factors per logarithm
        prod = 1.0;
    }
    logdet += log(prod) + (double)nsteady * lnS_c;
    const double ll = -0.5 * (quad + logdet + (double)nT * 1.8378770664093454836);
    out[b] = invalid_walker ? -INFINITY : ((bad || !isfinite(ll)) ? NAN : ll);
}

}  // namespace glg

// flux: [B, T] device, float (dtype 0) or double (dtype 1); everything else fp64 device.  Synchronises.
extern "C" int gp_serial_loglike(const void* flux, int B, const double* times, int T, const double* obs,
                                 const double* sigma, const double* gp, double* out, int dtype) {
    const unsigned blocks = (unsigned)((B + 31) / 32);
    if (dtype == 0)
        glg::gp_kernel<float><<<blocks, 32>>>((const float*)flux, B, times, T, obs, sigma, gp, out);
    else
        glg::gp_kernel<double><<<blocks, 32>>>((const double*)flux, B, times, T, obs, sigma, gp, out);
    return (int)cudaDeviceSynchronize();
}
