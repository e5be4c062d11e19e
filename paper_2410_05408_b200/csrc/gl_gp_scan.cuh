// gl_gp_scan.cuh -- the GP likelihood of gl_gp.cuh, PARALLEL IN TIME: one CTA of 256 threads per walker.
//
// The Kalman filter is a scan: Sarkka & Garcia-Fernandez (2021, "Temporal parallelization of Bayesian
// smoothers") write step k as an element a_k = (A, b, C, eta, J) -- the conditional
// p(x_k | x_{k-1}, y_k) = N(A x_{k-1} + b, C) and the likelihood p(y_k | x_{k-1}) ~ N_I(eta, J) in
// information form -- with an ASSOCIATIVE combination a_i (x) a_j, such that a_1 (x) ... (x) a_k carries
// the filtered mean (b) and covariance (C) at step k.  Here each thread (1) combines the elements of
// its contiguous chunk of the series, (2) an inclusive scan of the 256 chunk aggregates (shuffles
// within a warp, shared memory across the 8 warps) hands every thread the filtered state at the end
// of the previous chunk, and (3) each thread runs the ordinary filter over its own chunk from that
// state, accumulating its part of
//   ln L = -1/2 sum_i (v_i^2 / S_i + ln S_i + ln 2 pi).
// The serial chain per walker drops from T steps to ~2 T / 256 + 13 combinations.  fp64; H = (1, 0).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#include "gl_gp.cuh"

namespace glg {

struct Elem {
    double a00, a01, a10, a11;   // A
    double b0, b1;               // b
    double cxx, cxy, cyy;        // C (symmetric)
    double e0, e1;               // eta
    double jxx, jxy, jyy;        // J (symmetric)
};

__device__ __forceinline__ Elem identity_elem() {
    return Elem{1.0, 0.0, 0.0, 1.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
}

// a_i (x) a_j, i the EARLIER stretch.
__device__ __forceinline__ Elem combine(const Elem& i, const Elem& j) {
    // M = I + C_i J_j and its inverse
    const double m00 = 1.0 + i.cxx * j.jxx + i.cxy * j.jxy, m01 = i.cxx * j.jxy + i.cxy * j.jyy;
    const double m10 = i.cxy * j.jxx + i.cyy * j.jxy, m11 = 1.0 + i.cxy * j.jxy + i.cyy * j.jyy;
    const double idet = 1.0 / (m00 * m11 - m01 * m10);
    const double n00 = m11 * idet, n01 = -m01 * idet, n10 = -m10 * idet, n11 = m00 * idet;   // M^-1
    // T1 = A_j M^-1
    const double t00 = j.a00 * n00 + j.a01 * n10, t01 = j.a00 * n01 + j.a01 * n11;
    const double t10 = j.a10 * n00 + j.a11 * n10, t11 = j.a10 * n01 + j.a11 * n11;
    Elem o;
    o.a00 = t00 * i.a00 + t01 * i.a10;
    o.a01 = t00 * i.a01 + t01 * i.a11;
    o.a10 = t10 * i.a00 + t11 * i.a10;
    o.a11 = t10 * i.a01 + t11 * i.a11;
    const double u0 = i.b0 + i.cxx * j.e0 + i.cxy * j.e1, u1 = i.b1 + i.cxy * j.e0 + i.cyy * j.e1;
    o.b0 = t00 * u0 + t01 * u1 + j.b0;
    o.b1 = t10 * u0 + t11 * u1 + j.b1;
    // C = T1 C_i A_j^T + C_j
    const double w00 = t00 * i.cxx + t01 * i.cxy, w01 = t00 * i.cxy + t01 * i.cyy;
    const double w10 = t10 * i.cxx + t11 * i.cxy, w11 = t10 * i.cxy + t11 * i.cyy;
    o.cxx = w00 * j.a00 + w01 * j.a01 + j.cxx;
    o.cxy = 0.5 * ((w00 * j.a10 + w01 * j.a11) + (w10 * j.a00 + w11 * j.a01)) + j.cxy;
    o.cyy = w10 * j.a10 + w11 * j.a11 + j.cyy;
    // T2 = A_i^T (I + J_j C_i)^-1 = (M^-1 A_i)^T
    const double g00 = n00 * i.a00 + n01 * i.a10, g01 = n00 * i.a01 + n01 * i.a11;   // G = M^-1 A_i
    const double g10 = n10 * i.a00 + n11 * i.a10, g11 = n10 * i.a01 + n11 * i.a11;
    const double z0 = j.e0 - (j.jxx * i.b0 + j.jxy * i.b1), z1 = j.e1 - (j.jxy * i.b0 + j.jyy * i.b1);
    o.e0 = g00 * z0 + g10 * z1 + i.e0;
    o.e1 = g01 * z0 + g11 * z1 + i.e1;
    // J = G^T J_j A_i + J_i
    const double h00 = g00 * j.jxx + g10 * j.jxy, h01 = g00 * j.jxy + g10 * j.jyy;   // G^T J_j
    const double h10 = g01 * j.jxx + g11 * j.jxy, h11 = g01 * j.jxy + g11 * j.jyy;
    o.jxx = h00 * i.a00 + h01 * i.a10 + i.jxx;
    o.jxy = 0.5 * ((h00 * i.a01 + h01 * i.a11) + (h10 * i.a00 + h11 * i.a10)) + i.jxy;
    o.jyy = h10 * i.a01 + h11 * i.a11 + i.jyy;
    return o;
}

__device__ __forceinline__ Elem shfl_up_elem(const Elem& e, int delta) {
    Elem o;
    const double* s = reinterpret_cast<const double*>(&e);
    double* d = reinterpret_cast<double*>(&o);
#pragma unroll
    for (int k = 0; k < 14; ++k) d[k] = __shfl_up_sync(0xffffffffu, s[k], delta);
    return o;
}

// Transition over dt of the Matern-3/2 state-space model (see gl_gp.cuh).
struct Trans {
    double f00, f01, f10, f11, q00, q01, q11;
};
__device__ __forceinline__ Trans transition(double dt, double lam, double p0, double p1) {
    const double e = exp(-lam * dt), ld = lam * dt;
    Trans t;
    t.f00 = e * (1.0 + ld);
    t.f01 = e * dt;
    t.f10 = -e * lam * lam * dt;
    t.f11 = e * (1.0 - ld);
    (void)p1;
    matern32_q(ld, e * e, p0, lam, &t.q00, &t.q01, &t.q11);   // Q = Pinf - A Pinf A^T, no cancellation
    return t;
}

// agg (x) (element of one filter step), using the structure of a step element instead of the general
// combination: with f = F^T H^T = (F00, F01), the step has J = f f^T / Se, eta = f y / Se, A = (I - K H) F,
// b = K y, C = (I - K H) Q, K = Q H^T / Se, Se = Q00 + R.  Then I + C_agg J = I + u f^T / Se with
// u = C_agg f, whose inverse is I - u f^T / D, D = Se + f^T C_agg f (Sherman-Morrison), and
//   A' = Ae (A - u (f^T A) / D),   b' = Ae (b + u (y - f^T b) / D) + K y,
//   C' = Ae (C - u u^T / D) Ae^T + Ce,   eta' = eta + g (y - f^T b) / D,   J' = J + g g^T / D,   g = A^T f.
// Two divisions and ~70 multiply-adds instead of ~140 and a 2x2 inverse.
__device__ __forceinline__ Elem append_step(const Elem& a, const Trans& tr, double R, double y) {
    const double f0 = tr.f00, f1 = tr.f01;
    const double iSe = 1.0 / (tr.q00 + R), k0 = tr.q00 * iSe, k1 = tr.q01 * iSe;
    // Ae = (I - K H) F
    const double e00 = (1.0 - k0) * tr.f00, e01 = (1.0 - k0) * tr.f01;
    const double e10 = tr.f10 - k1 * tr.f00, e11 = tr.f11 - k1 * tr.f01;
    const double u0 = a.cxx * f0 + a.cxy * f1, u1 = a.cxy * f0 + a.cyy * f1;   // u = C f
    const double iD = 1.0 / ((tr.q00 + R) + f0 * u0 + f1 * u1);
    const double g0 = a.a00 * f0 + a.a10 * f1, g1 = a.a01 * f0 + a.a11 * f1;   // g = A^T f
    const double nu = y - (f0 * a.b0 + f1 * a.b1);                             // y - f^T b
    Elem o;
    // A' = Ae (A - u g^T / D)
    const double m00 = a.a00 - u0 * g0 * iD, m01 = a.a01 - u0 * g1 * iD;
    const double m10 = a.a10 - u1 * g0 * iD, m11 = a.a11 - u1 * g1 * iD;
    o.a00 = e00 * m00 + e01 * m10;
    o.a01 = e00 * m01 + e01 * m11;
    o.a10 = e10 * m00 + e11 * m10;
    o.a11 = e10 * m01 + e11 * m11;
    // b' = Ae (b + u nu / D) + K y
    const double w0 = a.b0 + u0 * nu * iD, w1 = a.b1 + u1 * nu * iD;
    o.b0 = e00 * w0 + e01 * w1 + k0 * y;
    o.b1 = e10 * w0 + e11 * w1 + k1 * y;
    // C' = Ae (C - u u^T / D) Ae^T + (I - K H) Q
    const double n00 = a.cxx - u0 * u0 * iD, n01 = a.cxy - u0 * u1 * iD, n11 = a.cyy - u1 * u1 * iD;
    const double r00 = e00 * n00 + e01 * n01, r01 = e00 * n01 + e01 * n11;
    const double r10 = e10 * n00 + e11 * n01, r11 = e10 * n01 + e11 * n11;
    o.cxx = r00 * e00 + r01 * e01 + (1.0 - k0) * tr.q00;
    o.cxy = r00 * e10 + r01 * e11 + (1.0 - k0) * tr.q01;
    o.cyy = r10 * e10 + r11 * e11 + (tr.q11 - k1 * tr.q01);
    o.e0 = a.e0 + g0 * nu * iD;
    o.e1 = a.e1 + g1 * nu * iD;
    o.jxx = a.jxx + g0 * g0 * iD;
    o.jxy = a.jxy + g0 * g1 * iD;
    o.jyy = a.jyy + g1 * g1 * iD;
    return o;
}


}  // namespace glg

namespace glg {

constexpr int GP_NT = 256;   // threads per walker
constexpr int CH = 4;        // filter steps whose inputs are loaded together

// One CTA per walker.  flux [B, T] (float or double), gp [B, 3] = (s, rho, jit), times ascending.
template <typename T>
__global__ void __launch_bounds__(GP_NT)
gp_scan_kernel(const T* __restrict__ flux, int B, const double* __restrict__ times, int nT,
               const double* __restrict__ obs, const double* __restrict__ sigma,
               const double* __restrict__ gp, double* __restrict__ out) {
    const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NWG = GP_NT / 32;
    __shared__ Elem s_wagg[NWG];
    __shared__ double s_part[NWG];
    __shared__ int s_flags[2];
    if (b >= B) return;
    const double s = gp[3 * b], rho = gp[3 * b + 1], jit = gp[3 * b + 2];
    if (!(s >= 0.0) || !(rho > 0.0) || !(jit >= 0.0) || !isfinite(s) || !isfinite(rho) || !isfinite(jit)) {
        if (tid == 0) out[b] = NAN;
        return;
    }
    const T* frow = flux + (size_t)b * nT;
    const double lam = 1.7320508075688772935 / rho;
    const double p0 = s * s, p1 = lam * lam * p0, jit2 = jit * jit;
    // launched behind the transit kernel with programmatic dependent launch: everything above ran while
    // that kernel was still finishing; its flux rows are read only from here on
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // contiguous chunks: thread k owns steps [k len, min((k+1) len, nT))
    const int len = (nT + GP_NT - 1) / GP_NT;
    const int i_lo = min(tid * len, nT), i_hi = min(i_lo + len, nT);
    bool bad = false, invalid_walker = false;

    // ---- (1) aggregate of this lane's chunk
    Elem agg = identity_elem();
    {
        Trans tr = {};
        double dtprev = -1.0;
        // the inputs of CH steps are loaded in one batch (the loop is a dependent chain: a load
        // inside it costs a full memory round trip per step)
        for (int i0 = i_lo; i0 < i_hi; i0 += CH) {
            double tv[CH + 1], sv[CH], yv[CH];
            tv[0] = times[max(i0 - 1, 0)];
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const int i = min(i0 + c, nT - 1);
                tv[c + 1] = times[i];
                sv[c] = sigma[i];
                const double fi = (double)frow[i];
                if (fi != fi && i0 + c < i_hi) invalid_walker = true;
                yv[c] = obs[i] - fi;
            }
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const int i = i0 + c;
                if (i >= i_hi) break;
                const double sg = sv[c], R = sg * sg + jit2, y = yv[c];
                if (!(sg >= 0.0)) bad = true;
                if (i == 0) {
                    // prior N(0, Pinf) updated with y_0: no dependence on an earlier state
                    const double S = p0 + R, k0 = p0 / S;
                    const Elem e = Elem{0.0, 0.0, 0.0, 0.0, k0 * y, 0.0, p0 - k0 * p0, 0.0, p1,
                                        0.0, 0.0, 0.0, 0.0, 0.0};
                    agg = combine(agg, e);
                    continue;
                }
                const double dt = tv[c + 1] - tv[c];
                if (dt < 0.0) bad = true;
                if (!(fabs(dt - dtprev) <= 1e-9 * dtprev)) {
                    tr = transition(dt, lam, p0, p1);
                    dtprev = dt;
                }
                agg = append_step(agg, tr, R, y);
            }
        }
    }
    // ---- (2) inclusive scan: Hillis-Steele within the warp, the warps' totals through shared memory
    Elem inc = agg;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const Elem left = shfl_up_elem(inc, d);
        if (lane >= d) inc = combine(left, inc);
    }
    if (tid == 0) s_flags[0] = s_flags[1] = 0;
    if (lane == 31) s_wagg[warp] = inc;
    __syncthreads();
    Elem before = identity_elem();   // everything owned by the warps in front of this one
    for (int w = 0; w < warp; ++w) before = combine(before, s_wagg[w]);
    if (warp > 0) inc = combine(before, inc);
    Elem prev = shfl_up_elem(inc, 1);   // filtered state at the end of the previous thread's chunk
    if (lane == 0) prev = before;
    // ---- (3) ordinary filter over the chunk, from that state
    double m0 = 0.0, m1 = 0.0, P00 = p0, P01 = 0.0, P11 = p1;
    if (tid > 0) {
        m0 = prev.b0;
        m1 = prev.b1;
        P00 = prev.cxx;
        P01 = prev.cxy;
        P11 = prev.cyy;
    }
    double quad = 0.0, logdet = 0.0, prod = 1.0;
    {
        Trans tr = {};
        double dtprev = -1.0;
        for (int i0 = i_lo; i0 < i_hi; i0 += CH) {
            double tv[CH + 1], sv[CH], yv[CH];
            tv[0] = times[max(i0 - 1, 0)];
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const int i = min(i0 + c, nT - 1);
                tv[c + 1] = times[i];
                sv[c] = sigma[i];
                yv[c] = obs[i] - (double)frow[i];
            }
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                const int i = i0 + c;
                if (i >= i_hi) break;
                if (i > 0) {
                    const double dt = tv[c + 1] - tv[c];
                    if (!(fabs(dt - dtprev) <= 1e-9 * dtprev)) {
                        tr = transition(dt, lam, p0, p1);
                        dtprev = dt;
                    }
                    const double n0 = tr.f00 * m0 + tr.f01 * m1, n1 = tr.f10 * m0 + tr.f11 * m1;
                    const double b00 = tr.f00 * P00 + tr.f01 * P01, b01 = tr.f00 * P01 + tr.f01 * P11;
                    const double b10 = tr.f10 * P00 + tr.f11 * P01, b11 = tr.f10 * P01 + tr.f11 * P11;
                    m0 = n0;
                    m1 = n1;
                    P00 = b00 * tr.f00 + b01 * tr.f01 + tr.q00;
                    P01 = b00 * tr.f10 + b01 * tr.f11 + tr.q01;
                    P11 = b10 * tr.f10 + b11 * tr.f11 + tr.q11;
                }
                const double sg = sv[c];
                const double S = P00 + sg * sg + jit2;
                if (!(S > 0.0)) bad = true;
                const double v = yv[c] - m0, iS = 1.0 / S;
                quad += v * v * iS;
                prod *= S;
                const double k0 = P00 * iS, k1 = P01 * iS;
                m0 += k0 * v;
                m1 += k1 * v;
                P11 -= k1 * P01;
                P01 -= k1 * P00;
                P00 -= k0 * P00;
            }
            logdet += log(prod);   // ln det K = sum ln S_i, CH factors per logarithm
            prod = 1.0;
        }
        logdet += log(prod);
    }
    double part = quad + logdet;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) part += __shfl_xor_sync(0xffffffffu, part, off);
    if (lane == 0) s_part[warp] = part;
    if (bad) s_flags[0] = 1;
    if (invalid_walker) s_flags[1] = 1;
    __syncthreads();
    if (tid == 0) {
        double tot = 0.0;
        for (int w = 0; w < NWG; ++w) tot += s_part[w];
        const double ll = -0.5 * (tot + (double)nT * 1.8378770664093454836);
        out[b] = s_flags[1] ? -INFINITY : ((s_flags[0] || !isfinite(ll)) ? NAN : ll);
    }
}

}  // namespace glg
