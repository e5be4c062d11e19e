// greenlantern_b200.cu -- kernels and C ABI of the B200 oblate-transit library (sm_100a).
//
// transit_kernel<T, EX> does the whole hot path of DESIGN.md section 1 for a batch of walkers:
//   a0 per-walker prelude                    -> shared memory (fp32 path: outline and window in fp32)
//   a1 Kepler + sky position per sub-sample  (phase formed and reduced in fp64, then the compute type)
//   a2 projected-outline geometry            (in the prelude; per sub-sample for tidally locked rows)
//   a3 outline/limb crossings, a4 boundary integrals   (fp64: gl_core.cuh, fp32: gl_fast32.cuh)
//   a5 exposure mean, residual^2, deterministic block + cluster reduction of chi^2
// Work layout: one thread-block CLUSTER per walker (1..8 CTAs of 128 threads, no
// atomics, no scratch in HBM); each CTA classifies its tile of the series against the walker's
// transit window and lists the in-window exposures in shared memory; after one cluster barrier the
// cluster's warps share the whole list over DSMEM, ingress/egress first.
// Also here: the bare-geometry kernels (config 5), the ceiling probes, the host-pointer wrappers and
// the C ABI.  Other kernels live in gl_simpson.cuh (the paper's snap + Simpson scheme),
// gl_frontend.cuh (App. A sampling parameters), gl_gp.cuh / gl_gp_scan.cuh (GP likelihood).
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <atomic>
#include <chrono>
#include <new>

#include <mutex>

#include "../../include/greenlantern_b200.h"
#include "gl_core.cuh"
#include "gl_fast32.cuh"
#include "gl_hot.cuh"
#include "gl_simpson.cuh"
#include "gl_frontend.cuh"
#include "gl_gp.cuh"
#include "gl_gp_scan.cuh"
#include "gl_tables.h"

namespace cg = cooperative_groups;

namespace {

constexpr int NQ32 = 16;   // Gauss-Legendre points per outline arc, fp32 production path
constexpr int NQ64 = 48;   // ... fp64 validation path
constexpr int NT = 128;    // threads per CTA
constexpr int MAXTILE = 32 * NT;   // exposure times one CTA classifies per round, at most
constexpr int MAXCLUSTER = 8;

__constant__ double c_phi64[NQ64 / 2], c_om64[NQ64 / 2];

constexpr double kPi = 3.14159265358979323846;
constexpr double kTwoPi = 6.28318530717958647692;

// ------------------------------------------------------------------------------------------
// a0 + a2: everything that is constant for one walker.
// ------------------------------------------------------------------------------------------
struct Walker {
    // orbit (fp64: phases and Kepler's equation are always double)
    double t0, inv_P, aR, e, omega, cosi, Mc, Ec, sinEc, cosEc, sinw, cosw, sq1me2, half_win_phase,
        hard_phase, reach;
    // projected outline: semi-axes and the rotation into the kernel frame
    double a, b, cpsi, spsi;
    // limb darkening, already divided by the disc-integrated intensity
    double k0, k1, k2;
    // tidally locked planets (NEXT-2): the outline changes along the orbit, so the
    // squared semi-axes, the rows of R(zeta, eta, xi) and beta (sin(beta) = cos i) are kept, in both
    // precisions, for the per-sample shape of locked_axes()
    double S2[3], r[9], sinb, cosb;
    float S2f[3], rf[9], sinbf, cosbf;
    int locked;
    int valid;
};

// Walker::S2 / r / sinb / cosb in the compute type
template <typename T> struct LockedView;
template <> struct LockedView<double> {
    static __device__ __forceinline__ const double* S2(const Walker& w) { return w.S2; }
    static __device__ __forceinline__ const double* r(const Walker& w) { return w.r; }
    static __device__ __forceinline__ double sinb(const Walker& w) { return w.sinb; }
    static __device__ __forceinline__ double cosb(const Walker& w) { return w.cosb; }
};
template <> struct LockedView<float> {
    static __device__ __forceinline__ const float* S2(const Walker& w) { return w.S2f; }
    static __device__ __forceinline__ const float* r(const Walker& w) { return w.rf; }
    static __device__ __forceinline__ float sinb(const Walker& w) { return w.sinbf; }
    static __device__ __forceinline__ float cosb(const Walker& w) { return w.cosbf; }
};

// Semi-axes a >= b and the major-axis direction (cos psi >= 0, sin psi) of the ellipse with covariance
// [[Cxx, Cxy], [Cxy, Cyy]] and determinant det (passed separately: eq. 13 / B16 give it without the
// cancellation of Cxx Cyy - Cxy^2).  psi = atan2(Cxy, (Cxx - Cyy)/2) / 2 by half-angle formulas.
template <typename R>
__device__ __forceinline__ void axes_from_covariance(R Cxx, R Cxy, R Cyy, R det, R* a, R* b, R* cpsi,
                                                     R* spsi) {
    const R hd = R(0.5) * (Cxx - Cyy);
    const R rad = glc::gsqrt(hd * hd + Cxy * Cxy);
    *a = glc::gsqrt(R(0.5) * (Cxx + Cyy) + rad);
    *b = glc::gsqrt(det) / *a;
    if (!(rad > R(0))) {
        *cpsi = R(1);
        *spsi = R(0);
        return;
    }
    const R c2 = hd / rad, s2 = Cxy / rad;
    if (c2 >= R(0)) {
        *cpsi = glc::gsqrt(R(0.5) * (R(1) + c2));
        *spsi = s2 / (R(2) * *cpsi);
    } else {
        const R sa = glc::gsqrt(R(0.5) * (R(1) - c2));
        *spsi = s2 < R(0) ? -sa : sa;
        *cpsi = glc::gabs(s2) / (R(2) * sa);
    }
}

// Outline of a tidally locked ellipsoid at orbital angle alpha (sa = sin alpha, ca = cos alpha):
// eq. B13 maps observer coordinates x to body coordinates x' = R Rx(-alpha) Ry(beta) x + const, so
// the body seen by the observer has covariance (M^T S M) with M = R Rx(-alpha) Ry(beta), whose sky
// block is eqs. B14-B16:
//   p_k = sin(beta) (r_k3 cos(alpha) + r_k2 sin(alpha)) - r_k1 cos(beta),  q_k = r_k3 sin(alpha) - r_k2 cos(alpha)
//   Cxx = dx^2 = sum S_k p_k^2 (B14),  Cxy = dx dy1 = sum S_k p_k q_k (B15),  Cyy = sum S_k q_k^2,
//   det = (dx dy2)^2 = S_a S_b s_c^2 + S_a S_c s_b^2 + S_b S_c s_a^2 (B16),
//   s_k = r_k1 sin(beta) + cos(beta) (r_k3 cos(alpha) + r_k2 sin(alpha)).
template <typename T>
__device__ __forceinline__ void locked_axes(const Walker& w, T sa, T ca, T* a, T* b, T* cpsi, T* spsi) {
    const T* S2 = LockedView<T>::S2(w);
    const T* r = LockedView<T>::r(w);
    const T sb = LockedView<T>::sinb(w), cb = LockedView<T>::cosb(w);
    T Cxx = T(0), Cxy = T(0), Cyy = T(0), sk[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const T m = r[3 * k + 2] * ca + r[3 * k + 1] * sa;
        const T p = sb * m - r[3 * k] * cb;
        const T q = r[3 * k + 2] * sa - r[3 * k + 1] * ca;
        sk[k] = r[3 * k] * sb + cb * m;
        Cxx += S2[k] * p * p;
        Cxy += S2[k] * p * q;
        Cyy += S2[k] * q * q;
    }
    const T det = S2[0] * S2[1] * sk[2] * sk[2] + S2[0] * S2[2] * sk[1] * sk[1] +
                  S2[1] * S2[2] * sk[0] * sk[0];
    axes_from_covariance<T>(Cxx, Cxy, Cyy, det, a, b, cpsi, spsi);
}


// Semi-axes (a >= b) and major-axis angle psi of the sky-projected outline of an ellipsoid with
// semi-axes (sa, sb, sc) along x', y', z' rotated by R = Rx(zeta) Ry(eta) Rz(xi)
// (eqs. 3-6).  The outline x = dx cos th, y = dy1 cos th + dy2 sin th of
// PAPER.md:89-96 (eqs. 11-13) is the image of the unit circle under the lower-Cholesky factor of
//   C = [[Cxx, Cxy], [Cxy, Cyy]],  Cxx = dx^2 = sa^2 r1^2 + sb^2 r4^2 + sc^2 r7^2   (eq. 11)
//   Cxy = dx dy1 = sa^2 r1 r2 + sb^2 r4 r5 + sc^2 r7 r8                               (eq. 12)
//   det C = (dx dy2)^2 = sa^2 sb^2 r9^2 + sa^2 sc^2 r6^2 + sb^2 sc^2 r3^2             (eq. 13)
// so its principal axes are the eigenvectors of C: a^2 = larger eigenvalue, b = sqrt(det C)/a.
// R = double for the validation path; float for the production path, whose per-walker constants
// are narrowed to fp32 anyway (relative 1e-7 on a, b, psi: < 1e-8 in flux).
template <typename R>
__device__ void outline_axes(R sa, R sb, R sc, R zeta, R eta, R xi, R* a, R* b, R* cpsi, R* spsi,
                             R* rows) {
    R sz, cz, se, ce, sx, cx;
    glc::gsincos(zeta, &sz, &cz);
    glc::gsincos(eta, &se, &ce);
    glc::gsincos(xi, &sx, &cx);
    // rows of Rx(zeta) Ry(eta) Rz(xi)
    const R r1 = ce * cx, r2 = -ce * sx, r3 = se;
    const R r4 = cz * sx + sz * se * cx, r5 = cz * cx - sz * se * sx, r6 = -sz * ce;
    const R r7 = sz * sx - cz * se * cx, r8 = sz * cx + cz * se * sx, r9 = cz * ce;
    const R A2 = sa * sa, B2 = sb * sb, C2 = sc * sc;
    const R Cxx = A2 * r1 * r1 + B2 * r4 * r4 + C2 * r7 * r7;
    const R Cxy = A2 * r1 * r2 + B2 * r4 * r5 + C2 * r7 * r8;
    const R Cyy = A2 * r2 * r2 + B2 * r5 * r5 + C2 * r8 * r8;
    const R det = A2 * B2 * r9 * r9 + A2 * C2 * r6 * r6 + B2 * C2 * r3 * r3;
    axes_from_covariance<R>(Cxx, Cxy, Cyy, det, a, b, cpsi, spsi);
    if (rows) {
        rows[0] = r1; rows[1] = r2; rows[2] = r3;
        rows[3] = r4; rows[4] = r5; rows[5] = r6;
        rows[6] = r7; rows[7] = r8; rows[8] = r9;
    }
}

// nparams = GL_NPARAMS (oblate, free orientation) or GL_NPARAMS_EX (NEXT-2: + zeta, b-axis/Rp_eq,
// c-axis/Rp_eq, locked flag).
__device__ __forceinline__ bool walker_valid(const double* __restrict__ p, int nparams) {
    const double P = p[1], aR = p[2], b = p[3], e = p[4], om = p[5];
    const double Rp = p[6], f = p[7], u1 = p[10], u2 = p[11];
    bool ok = true;
    for (int k = 0; k < GL_NPARAMS; ++k) ok = ok && isfinite(p[k]);
    const double norm = 1.0 - u1 / 3.0 - u2 / 6.0;
    ok = ok && (P > 0.0) && (e >= 0.0) && (e < 1.0) && (Rp > 0.0) && (Rp < 0.5) && (f >= 0.0) &&
         (f < 1.0) && (aR * (1.0 - e) > 1.0) && (norm > 0.0);
    if (ok) ok = (e == 0.0) ? (fabs(b) <= aR) : (fabs(b) * (1.0 + e * sin(om)) <= aR * (1.0 - e * e));
    if (ok && nparams == GL_NPARAMS_EX) {
        const double rb = p[13], rc = p[14];
        ok = isfinite(p[12]) && isfinite(rb) && isfinite(rc) && (rb > 0.0) && (rc > 0.0) &&
             (Rp * rb < 0.5) && (Rp * rc < 0.5) && (p[15] == 0.0 || p[15] == 1.0);
    }
    return ok;
}

// The prelude is split in two independent halves so that two warps can run them side by side:
// ORBIT (validity, phase constants, cos i, transit window, Kepler constants) and SHAPE (projected
// outline, limb-darkening constants).  R as in outline_axes.
// Largest semi-axis of the ellipsoid = upper bound of the projected semi-major axis (equal to it
// for the oblate model, whose projected semi-major axis is the equatorial radius).
__device__ __forceinline__ double largest_axis(const double* __restrict__ p, int nparams) {
    double m = fmax(p[6] * (1.0 - p[7]), p[6]);
    if (nparams == GL_NPARAMS_EX) m = fmax(p[6] * (1.0 - p[7]), fmax(p[6] * p[13], p[6] * p[14]));
    return m;
}

// The ORBIT half comes in three parts that write disjoint fields of the Walker and read only the parameter
// row, so that three threads can run them side by side (generic_unit: a dozen fp64 libm calls in a row took
// 4 us on one thread); walker_prelude_orbit runs them one after the other.
//   basic  : validity, t0, 1/P, a/R*, e, omega, locked
//   kepler : Kepler constants of the conjunction (R7)
//   window : sin/cos omega, cos i, the transit window in phase, reach (+ what locked_axes needs)
__device__ void walker_prelude_basic(const double* __restrict__ p, int nparams, Walker* w) {
    w->valid = walker_valid(p, nparams) ? 1 : 0;
    w->locked = (nparams == GL_NPARAMS_EX && p[15] == 1.0) ? 1 : 0;
    w->t0 = p[0];
    w->inv_P = 1.0 / p[1];
    w->aR = p[2];
    w->e = p[4];
    w->omega = p[5];
}
__device__ void walker_prelude_kepler(const double* __restrict__ p, Walker* w) {
    const double e = p[4], om = p[5];
    if (e == 0.0) {
        w->Mc = w->Ec = w->sinEc = 0.0;
        w->cosEc = 1.0;
        w->sq1me2 = 1.0;
        return;
    }
    // R7: conjunction at true anomaly pi/2 - omega
    const double nuc = 0.5 * kPi - om;
    const double s1 = sqrt(1.0 + e), s2 = sqrt(1.0 - e);
    const double Ec = 2.0 * atan2(s2 * sin(0.5 * nuc), s1 * cos(0.5 * nuc));
    sincos(Ec, &w->sinEc, &w->cosEc);
    w->Ec = Ec;
    w->Mc = Ec - e * w->sinEc;
    w->sq1me2 = s1 * s2;
}
template <typename R>
__device__ void walker_prelude_window(const double* __restrict__ p, int nparams, double t_exp, Walker* w) {
    const double P = p[1], aR = p[2], b = p[3], e = p[4], om = p[5];
    const double inv_P = 1.0 / P;
    const double Rp = largest_axis(p, nparams);
    // the projected semi-major axis of an oblate spheroid is its equatorial radius: the window
    // does not have to wait for the SHAPE half
    const bool lowp = sizeof(R) == 4;
    const double reach = (1.0 + Rp) * (lowp ? 1.0 + 1e-5 : 1.0 + 1e-12);
    double hw = -1.0;   // < 0: never in transit
    double cosi;
    if (e == 0.0) {
        // PAPER.md:85-87 eqs. 9-10: the centre is within `reach` of the star centre iff
        //   sin^2(phi) < [(reach/aR)^2 - cos^2 i] / sin^2 i  and cos(phi) > 0;
        // stored as a half-width in orbital phase, widened by half an exposure.
        cosi = b / aR;
        w->sinw = 0.0;
        w->cosw = 1.0;
        const R ci2 = R(cosi) * R(cosi), q = R(reach) / R(aR);
        const R S2 = (q * q - ci2) / (R(1) - ci2);
        if (S2 > R(0))
            hw = (S2 >= R(1)) ? 0.25
                              : (double)(glc::gasin(glc::gsqrt(S2)) * R(0.15915494309189535)) *
                                    (lowp ? 1.0 + 1e-5 : 1.0);
        if (hw >= 0.0) hw += 0.5 * t_exp * inv_P + (lowp ? 1e-9 : 1e-13);
        // exposures wholly inside |phase| < hard_phase keep the outline at least 0.01 inside the
        // limb (the cheap tiers of gl_fast32.cuh); the others (ingress, egress, grazing) are
        // listed FIRST so that the expensive geometries start early (scheduling only)
        const R qh = R(0.99 - Rp) / R(aR);
        const R S2h = (qh * qh - ci2) / (R(1) - ci2);
        double hp = 0.0;
        if (S2h > R(0) && S2h < R(1))
            hp = (double)(glc::gasin(glc::gsqrt(S2h)) * R(0.15915494309189535)) - 0.5 * t_exp * inv_P;
        w->hard_phase = hp > 0.0 ? hp : 0.0;
    } else {
        // R7: cos i from the impact parameter
        const double nuc = 0.5 * kPi - om;
        const double s1 = sqrt(1.0 + e), s2 = sqrt(1.0 - e);
        sincos(om, &w->sinw, &w->cosw);
        cosi = (b / aR) * (1.0 + e * w->sinw) / (1.0 - e * e);
        // Transit window in phase, conservative.  With phi' = nu - nu_c the angle from conjunction,
        // the sky distance is >= r |sin phi'| >= aR (1-e) |sin phi'|, so in transit needs
        // |phi'| < phi_max = asin(reach / (aR (1-e))); the time to sweep phi_max is at most
        // phi_max / min(d nu/dt), d nu/dt = n (1 + e cos nu)^2 / (1-e^2)^{3/2}, minimum taken over
        // [nu_c - phi_max, nu_c + phi_max].  (Far from conjunction the planet is behind the star or
        // beyond reach: those exposures get flux = 1 without a Kepler solve.)
        const double smax = reach / (aR * (1.0 - e));
        if (smax >= 1.0) {
            hw = 0.5;
        } else {
            const double pmax = asin(smax);
            double cmin = fmin(cos(nuc - pmax), cos(nuc + pmax));
            double off = fmod(nuc - kPi, kTwoPi);   // does the interval contain nu = pi (apastron)?
            if (off > kPi) off -= kTwoPi;
            if (off < -kPi) off += kTwoPi;
            if (fabs(off) <= pmax) cmin = -1.0;
            const double slow = (1.0 + e * cmin) * (1.0 + e * cmin);
            hw = pmax / kTwoPi * (1.0 - e * e) * s1 * s2 / slow * (1.0 + 1e-6) + 0.5 * t_exp * inv_P + 1e-9;
            if (hw > 0.5) hw = 0.5;
        }
        w->hard_phase = 0.0;
    }
    w->cosi = cosi;
    w->half_win_phase = hw;
    w->reach = reach;
    if (nparams == GL_NPARAMS_EX && p[15] == 1.0) {
        // eq. 9: x0 = d cos(alpha) sin(beta)  =>  sin(beta) = cos i  (used by locked_axes)
        w->sinb = cosi;
        w->cosb = sqrt(fmax(1.0 - cosi * cosi, 0.0));
        w->sinbf = (float)w->sinb;
        w->cosbf = (float)w->cosb;
    }
}
template <typename R>
__device__ void walker_prelude_orbit(const double* __restrict__ p, int nparams, double t_exp, Walker* w) {
    walker_prelude_basic(p, nparams, w);
    if (!w->valid) return;
    walker_prelude_kepler(p, w);
    walker_prelude_window<R>(p, nparams, t_exp, w);
}

template <typename R>
__device__ void walker_prelude_shape(const double* __restrict__ p, int nparams, Walker* w) {
    const double Rp = p[6], f = p[7], xi = p[8], eta = p[9], u1 = p[10], u2 = p[11];
    // semi-axes along x', y', z': polar Rp (1-f) and, for the oblate model, equatorial Rp twice with
    // zeta = 0 (R4, R5); the extended row gives zeta and the two other axes in units of Rp
    const bool ex = nparams == GL_NPARAMS_EX;
    const double sa = Rp * (1.0 - f), sb = ex ? Rp * p[13] : Rp, sc = ex ? Rp * p[14] : Rp;
    const double zeta = ex ? p[12] : 0.0;
    R a, b, cpsi, spsi, rows[9];
    outline_axes<R>(R(sa), R(sb), R(sc), R(zeta), R(eta), R(xi), &a, &b, &cpsi, &spsi, rows);
    w->a = a;
    w->b = b;
    w->cpsi = cpsi;
    w->spsi = spsi;
    if (ex && p[15] == 1.0) {   // what locked_axes() needs
        w->S2[0] = sa * sa;
        w->S2[1] = sb * sb;
        w->S2[2] = sc * sc;
        for (int k = 0; k < 3; ++k) w->S2f[k] = (float)w->S2[k];
        for (int k = 0; k < 9; ++k) {
            w->r[k] = rows[k];
            w->rf[k] = (float)rows[k];
        }
    }
    const R pn = R(kPi * (1.0 - u1 / 3.0 - u2 / 6.0));
    w->k0 = R(1.0 - u1 - 2.0 * u2) / pn;
    w->k1 = R(u1 + 2.0 * u2) / pn;
    w->k2 = R(u2) / pn;
}

// ------------------------------------------------------------------------------------------
// a1: sky-plane position of the planet centre at time t, in the kernel frame.
//   e = 0: eqs. 9-10 with alpha = 2 pi (t - t0)/P, d = a/R*, sin(beta) = cos i.
//   e > 0: Kepler's equation in fp64 (R7).  Returns false when the planet is behind the star.
// The orbital phase is always formed and reduced in fp64.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double reduced_phase(const Walker& w, double t) {
    const double ph = (t - w.t0) * w.inv_P;
    return ph - rint(ph);
}

__device__ double kepler_E(double M, double e) {
    // Newton from E = M + e sin M, safeguarded by the bracket [M - e, M + e]
    double lo = M - e, hi = M + e;
    double E = fmin(fmax(M + e * sin(M), lo), hi);
    for (int it = 0; it < 64; ++it) {
        double s, c;
        sincos(E, &s, &c);
        const double f = E - e * s - M;
        if (f > 0.0) hi = E; else lo = E;
        double En = E - f / (1.0 - e * c);
        if (!(En > lo && En < hi)) En = 0.5 * (lo + hi);
        const double d = En - E;
        E = En;
        if (fabs(d) <= 2e-16 * fmax(1.0, fabs(E))) break;
    }
    return E;
}

// fp64 position in the SKY frame (x0 along the projected orbit normal, y0 along the chord).
__device__ bool sky_position_f64(const Walker& w, double ph, double* x0, double* y0, double* sphi,
                                 double* cphi) {
    if (w.e == 0.0) {
        double s, c;
        sincospi(2.0 * ph, &s, &c);
        *x0 = w.aR * c * w.cosi;
        *y0 = w.aR * s;
        *sphi = s;
        *cphi = c;
        return c > 0.0;
    }
    // Kepler's equation about the conjunction: E - e sin E = Mc + dM with Mc = Ec - e sin Ec, written
    // as (E - Ec) - e (sin E - sin Ec) = dM; Newton from the second-order expansion in dM (in-window
    // phases are close to conjunction: two or three steps), the bracketed solver as a fallback.
    const double dM = kTwoPi * ph;
    const double d1 = 1.0 / (1.0 - w.e * w.cosEc);
    double E = w.Ec + dM * d1 - 0.5 * w.e * w.sinEc * dM * dM * d1 * d1 * d1;
    double sE, cE;
    int it = 0;
    for (; it < 8; ++it) {
        sincos(E, &sE, &cE);
        const double dE = ((E - w.Ec) - w.e * (sE - w.sinEc) - dM) / (1.0 - w.e * cE);
        E -= dE;
        if (fabs(dE) < 1e-15) break;   // (sE, cE) then belong to E within 1e-15
    }
    if (it == 8) {
        E = kepler_E(w.Mc + dM, w.e);
        sincos(E, &sE, &cE);
    }
    // true anomaly and phi = nu + omega - pi/2 without inverse trigonometry:
    //   cos nu = (cos E - e)/(1 - e cos E), sin nu = sqrt(1-e^2) sin E/(1 - e cos E),
    //   cos phi = sin(nu + omega), sin phi = -cos(nu + omega)
    const double q = 1.0 - w.e * cE, iq = 1.0 / q;
    const double cnu = (cE - w.e) * iq, snu = w.sq1me2 * sE * iq;
    const double r = w.aR * q;
    const double cp = snu * w.cosw + cnu * w.sinw, sp = snu * w.sinw - cnu * w.cosw;
    *x0 = r * cp * w.cosi;
    *y0 = r * sp;
    *sphi = sp;
    *cphi = cp;
    return cp > 0.0;
}

// Per-walker constants narrowed to the compute type once per thread.
template <typename T> struct WalkerT {
    T aR, cosi, a, b, cpsi, spsi, k0, k1, k2;
    bool circular;
};
template <typename T> __device__ __forceinline__ WalkerT<T> narrow(const Walker& w) {
    WalkerT<T> v;
    v.aR = T(w.aR);
    v.cosi = T(w.cosi);
    v.a = T(w.a);
    v.b = T(w.b);
    v.cpsi = T(w.cpsi);
    v.spsi = T(w.spsi);
    v.k0 = T(w.k0);
    v.k1 = T(w.k1);
    v.k2 = T(w.k2);
    v.circular = (w.e == 0.0);
    return v;
}

// a3 + a4 for an outline centred at (xc, yc) in the kernel frame: fp64 = generic bracketed search +
// 48-point rule (validation), fp32 = gl_fast32.cuh (production).
template <typename T>
__device__ __forceinline__ T blocked_at(const glf::TrapNode* trap, T xc, T yc, T a, T b, T k0, T k1,
                                        T k2);
template <> __device__ __forceinline__ double blocked_at<double>(const glf::TrapNode*, double xc,
                                                                 double yc, double a, double b,
                                                                 double k0, double k1, double k2) {
    double A[3];
    if (!glc::overlap_areas<double, NQ64>(xc, yc, a, b, c_phi64, c_om64, A)) return 0.0;
    return k0 * A[0] + k1 * A[1] + k2 * A[2];
}
template <> __device__ __forceinline__ float blocked_at<float>(const glf::TrapNode* trap, float xc,
                                                               float yc, float a, float b, float k0,
                                                               float k1, float k2) {
    return glf::blocked_f32(trap, xc, yc, a, b, k0, k1, k2);
}

// Blocked fraction delta = 1 - F_inst at reduced phase ph (a1 + a3 + a4).
template <typename T, bool EX>
__device__ __forceinline__ T blocked_fraction(const glf::TrapNode* trap, const Walker& w,
                                              const WalkerT<T>& v, double ph) {
    T x0, y0, s, c;   // (s, c) = sine and cosine of the orbital angle from conjunction
    if (v.circular) {
        // phi = 2 pi ph, |ph| <= 1/2; narrowed AFTER the fp64 phase reduction
        glc::gsincos(T(kTwoPi * ph), &s, &c);
        if (!(c > T(0))) return T(0);
        x0 = v.aR * c * v.cosi;
        y0 = v.aR * s;
    } else {
        double X, Y, sphi, cphi;
        if (!sky_position_f64(w, ph, &X, &Y, &sphi, &cphi)) return T(0);
        x0 = T(X);
        y0 = T(Y);
        s = T(sphi);
        c = T(cphi);
    }
    T a = v.a, b = v.b, cpsi = v.cpsi, spsi = v.spsi;
    if (EX && w.locked) locked_axes<T>(w, s, c, &a, &b, &cpsi, &spsi);   // outline of THIS sub-exposure
    const T xc = cpsi * x0 + spsi * y0, yc = cpsi * y0 - spsi * x0;
    return blocked_at<T>(trap, xc, yc, a, b, v.k0, v.k1, v.k2);
}


}  // namespace

// hot_kernel's path for a walker off the common path (declared in gl_hot.cuh): the CTA -- or every CTA of
// the cluster, each on its share gtid, gtid + ntot, ... of the exposures -- runs the full-featured
// arithmetic: general prelude (validity incl. the eccentric rules, Kepler constants, conservative
// window), fp64 phase of every exposure (any order of the series, any number of transits), Kepler's
// equation per sub-exposure for e > 0, the generic crossing search where the evolute test asks for it.
// One exposure per lane and pass, sub-exposures in turn; chi^2 terms in hot_kernel's cancellation-free
// form.  Inlined into hot_kernel's second loop (behind the common path: fetched only when a walker needs it).
__device__ __forceinline__ int glh::generic_unit(const glh::HotArgs& A, bool pre, int wk, int t_lo, int nT,
                                                 int gtid, int ntot, const glf::TrapNode* trap, double* acc,
                                                 float* s_d, int* s_li, int* s_cnt) {
    __shared__ Walker gw;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double* p = A.params + (size_t)wk * GL_NPARAMS;
    // four threads of four warps, side by side (the parts write disjoint fields; on an invalid row the
    // three that do not judge validity compute garbage that nobody reads)
    if (tid == 0) walker_prelude_basic(p, GL_NPARAMS, &gw);
    if (tid == 32) walker_prelude_shape<float>(p, GL_NPARAMS, &gw);
    if (tid == 64) walker_prelude_kepler(p, &gw);
    if (tid == 96) walker_prelude_window<float>(p, GL_NPARAMS, A.t_exp, &gw);
    __syncthreads();
    GLH_TL(11);
    const double* __restrict__ seg = A.times + t_lo;
    float* frow = A.flux ? A.flux + (size_t)wk * A.T + t_lo : nullptr;
    if (!gw.valid) {
        if (frow)
            for (int i = gtid; i < nT; i += ntot) frow[i] = __int_as_float(0x7fc00000);
        return glh::CLS_INVALID;
    }
    const WalkerT<float> v = narrow<float>(gw);
    const int S = A.n_ss;
    const double hwin = gw.half_win_phase, inv_ss = 1.0 / (double)S;
    // mean over the exposure -> flux and this exposure's chi^2 term (hot_kernel's cancellation-free form)
    auto finish = [&](int i, float dbar) {
        if (frow) frow[i] = 1.f - dbar;
        if (A.chi2) {
            float ob, rs;
            if (pre) {
                const float2 o2 = A.ow[t_lo + i];
                ob = o2.x;
                rs = o2.y;
            } else {
                ob = (float)(A.obs[t_lo + i] - 1.0);
                const float sf = (float)A.sigma[t_lo + i];
                rs = glf::mufu_rcp(sf);
                rs = rs * fmaf(-sf, rs, 2.f);
            }
            const float d = dbar * rs;
            *acc += (double)(d * fmaf(2.f * ob, rs, d));
        }
    };
    auto sample = [&](double tc, int j) {
        const double t = tc + (((double)j + 0.5) * inv_ss - 0.5) * A.t_exp;
        return blocked_fraction<float, false>(trap, gw, v, reduced_phase(gw, t));
    };
    if (S > glh::CAP) {   // (more sub-exposures than the pair buffer holds: one exposure per lane, in turn)
        for (int i = gtid; i < nT; i += ntot) {
            const double tc = seg[i];
            if (!(fabs(reduced_phase(gw, tc)) < hwin)) {
                if (frow) frow[i] = 1.f;
                continue;
            }
            float sum = 0.f;
            for (int j = 0; j < S; ++j) sum += sample(tc, j);
            finish(i, sum * A.inv_ss);
        }
        return glh::CLS_SIMPLE;
    }
    // Passes of one exposure per thread: window test on the fp64 phase (any order of the series, any number
    // of transits), in-window indices compacted in thread order (ballot + counts of the 16 warps: the same
    // list in every run), then lane = (exposure, sub-exposure) pair in groups that fit the pair buffer,
    // exposure means in sub-exposure order (R18).  In-transit exposures are few and the generic geometry is
    // long: one exposure per lane with its sub-exposures in turn left most of the CTA idle.
    const int G = glh::CAP / S;   // exposures per group (>= 1)
    for (int base = 0; base < nT; base += ntot) {
        const int i = base + gtid;
        bool in = false;
        if (i < nT) {
            in = fabs(reduced_phase(gw, seg[i])) < hwin;
            if (!in && frow) frow[i] = 1.f;
        }
        const unsigned bal = __ballot_sync(0xffffffffu, in);
        // (the barrier also says that the previous pass is done with s_li / s_d / s_cnt; most passes of a
        // K2-shaped series hold no in-window exposure at all and end here)
        if (__syncthreads_count(in) == 0) continue;
        if (lane == 0) s_cnt[warp] = __popc(bal);
        __syncthreads();
        int before = 0, n_in = 0;
        for (int k = 0; k < glh::HOT_NW; ++k) {
            const int c = s_cnt[k];
            before += k < warp ? c : 0;
            n_in += c;
        }
        GLH_ASSERT(before + __popc(bal) <= n_in && n_in <= glh::HOT_NT && n_in <= glh::CAP);
        if (in) s_li[before + __popc(bal & ((1u << lane) - 1u))] = i;
        __syncthreads();
        GLH_TL(12);
        for (int g0 = 0; g0 < n_in; g0 += G) {   // (n_in is the CTA's: the barriers below are uniform)
            const int ng = min(G, n_in - g0);
            for (int q = tid; q < ng * S; q += glh::HOT_NT) {
                const int e = q / S, j = q - e * S;
                GLH_ASSERT(q < glh::CAP && g0 + e < n_in && s_li[g0 + e] >= 0 && s_li[g0 + e] < nT);
                s_d[q] = sample(seg[s_li[g0 + e]], j);
            }
            __syncthreads();
            GLH_TL(13);
            for (int e = tid; e < ng; e += glh::HOT_NT) {
                float sum = 0.f;
                GLH_ASSERT(e * S + S <= glh::CAP);
                for (int j = 0; j < S; ++j) sum += s_d[e * S + j];
                finish(s_li[g0 + e], sum * A.inv_ss);
            }
            __syncthreads();
            GLH_TL(14);
        }
    }
    return glh::CLS_SIMPLE;
}

namespace {

// ------------------------------------------------------------------------------------------
// Deterministic sum of one double per thread over the CTA (fixed shuffle tree, fixed warp order).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum(double v, double* warp_scratch) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) warp_scratch[warp] = v;
    __syncthreads();
    double tot = 0.0;
    if (threadIdx.x == 0)
        for (int k = 0; k < NT / 32; ++k) tot += warp_scratch[k];
    return tot;   // valid in thread 0
}

// ------------------------------------------------------------------------------------------
// The fused kernel.  grid = (cluster size C, walkers in flight); cluster = (C, 1, 1).
//   flux  : [B, T] of T-typed values or nullptr          chi2 : [B] or nullptr
//   obs, sigma : [T] fp64 or nullptr (only read when chi2 != nullptr)
// Per walker the exposure times are taken in rounds of C tiles (one round unless T > C * 4096):
// CTA r classifies tile r against the transit window -- out-of-window exposures are finished on
// the spot (flux = 1, baseline residual) -- and compacts the in-window indices into its own
// shared list; after ONE cluster barrier the cluster's warps take groups of in-window exposures
// in turn, reading the other CTAs' lists over DSMEM.  A K2-shaped series (1 % in transit, all of
// it inside one tile) is thereby spread over the whole cluster, and ingress/egress (the expensive
// geometries) over every warp.
// ------------------------------------------------------------------------------------------
// Residual^2 of one exposure against the data (R19), in the compute type; a bad sigma poisons the
// walker's chi^2.  fp64 path: IEEE division.  fp32 path: obs - 1 is formed in fp64 and narrowed (it
// is ~1e-4, so fp32 keeps 7 digits of it), 1/sigma is the MUFU reciprocal plus one Newton step;
// each term is good to ~2e-7 relative and the terms are summed in fp64 (chi^2 budget: 1e-4).
template <typename T> __device__ __forceinline__ T residual_sq(double obs_m1, T delta, double sg);
template <> __device__ __forceinline__ double residual_sq<double>(double obs_m1, double delta,
                                                                  double sg) {
    const double rr = (obs_m1 + delta) / sg;
    return (sg > 0.0 && isfinite(sg)) ? rr * rr : (double)INFINITY;
}
template <> __device__ __forceinline__ float residual_sq<float>(double obs_m1, float delta,
                                                                double sg) {
    const float sf = (float)sg;
    if (sf > 1e-30f && sf < 1e30f) {
        float r = glf::mufu_rcp(sf);
        r = r * fmaf(-sf, r, 2.f);
        const float rr = ((float)obs_m1 + delta) * r;
        return rr * rr;
    }
    return (float)residual_sq<double>(obs_m1, (double)delta, sg);   // out-of-range sigma
}

// chi^2 term of an in-window exposure.  shared_base: the launch-wide baseline
// S = sum_i ((obs_i - 1)/sigma_i)^2 (baseline_kernel) already counts this exposure as if it were out
// of transit, so the term is the DIFFERENCE model - baseline (0 when the baseline term is not finite:
// S is then +inf already).
template <typename T>
__device__ __forceinline__ double listed_residual(double obs_m1, T dbar, double sg, int shared_base) {
    const double term = (double)residual_sq<T>(obs_m1, dbar, sg);
    if (!shared_base) return term;
    const double base = (double)residual_sq<T>(obs_m1, T(0), sg);
    return isfinite(base) ? term - base : 0.0;
}

// fp32 path only: the walker-independent baseline S = sum_i ((obs_i - 1)/sigma_i)^2 over ALL
// exposures, once per launch instead of once per walker (every walker's chi^2 is S plus the
// model-minus-baseline differences of its in-window exposures).  One CTA, fp64, fixed summation
// order; S is left in chi2[0..B) (narrowed: 6e-8 relative, chi^2 budget 1e-4), where the transit
// kernel, launched right behind with programmatic dependent launch, picks it up at its very end.
__global__ void __launch_bounds__(1024)
baseline_kernel(const double* __restrict__ obs, const double* __restrict__ sigma, int nT,
                float* __restrict__ chi2, int B) {
    asm volatile("griddepcontrol.launch_dependents;");
    __shared__ double s_w[32];
    __shared__ double s_tot;
    double acc = 0.0;
    for (int i = threadIdx.x; i < nT; i += 1024) acc += residual_sq<double>(obs[i] - 1.0, 0.0, sigma[i]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < 32; ++k) tot += s_w[k];
        s_tot = tot;
    }
    __syncthreads();
    const float S = (float)s_tot;
    for (int b = threadIdx.x; b < B; b += 1024) chi2[b] = S;
}

// EX = extended parameter rows (NEXT-2); the 12-column instantiation carries none of that code.
// SEG = the series of a walker may be split into segments taken by separate clusters (flux-only calls).
template <typename T, bool EX, bool SEG>
__global__ void __launch_bounds__(NT, sizeof(T) == 4 ? 8 : 2)
transit_kernel(const double* __restrict__ params, int B,
               const double* __restrict__ times_all, int nT_all,
               int tile, double t_exp, int n_ss, const double* __restrict__ obs,
               const double* __restrict__ sigma, T* __restrict__ flux, T* chi2, int shared_base,
               int nseg_arg, int seglen_arg) {
    const int nseg = SEG ? nseg_arg : 1, seglen = SEG ? seglen_arg : nT_all;
    cg::cluster_group cluster = cg::this_cluster();
    const int crank = (int)cluster.block_rank(), csize = (int)cluster.num_blocks();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NT / 32;
    constexpr int nparams = EX ? GL_NPARAMS_EX : GL_NPARAMS;

    __shared__ Walker sw;
    __shared__ int s_list[MAXTILE];   // in-window time indices of this CTA's tile
    __shared__ int s_nlist[2];        // this CTA's list: [0] early (ingress/egress) entries, [1] the rest
    __shared__ int s_cnt[2][NW];      // in-window count per warp of the tile, early / rest
    __shared__ int s_pre[2][MAXCLUSTER + 1];   // prefix of the cluster's list lengths, early / rest
    __shared__ double s_red[NW];
    __shared__ double s_gather[2][MAXCLUSTER];   // rank 0's copy collects the CTAs' chi^2 partials
                                                 // (written over DSMEM; slot = walker parity)
    __shared__ glf::TrapNode s_trap[16];   // trapezoid nodes (per-lane strides: not constant memory)
    if (tid < 16) s_trap[tid] = glf::TrapNode{glf::c_trap_cos[tid], glf::c_trap_sin[tid]};

    const double inv_ss = 1.0 / (double)n_ss;
    const int nsub = tile / NT;   // exposures per thread and tile (<= 32: one mask bit each)
    const int round_span = csize * tile;
    const bool want_chi2 = (chi2 != nullptr);
    int wpar = 0;
    bool lists_live = false;   // uniform over the cluster

    // warm the L2 with this CTA's first tile while the prelude runs (one line = 16 doubles)
    for (int i = crank * tile + tid * 16; i < min(nT_all, (crank + 1) * tile); i += NT * 16) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(times_all + i));
        if (want_chi2) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(obs + i));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(sigma + i));
        }
    }
    // A cluster works on one (walker, segment of the series); nseg > 1 only for flux-only calls with
    // few walkers and a long series (one light curve of 1e5 exposures would otherwise use 8 CTAs of
    // the whole GPU); chi^2 calls keep nseg = 1 (the sum over a walker's series stays in one cluster).
    for (long long vw = blockIdx.y; vw < (long long)B * nseg; vw += gridDim.y) {
        const int wk = (int)(vw / nseg), t_lo = (int)(vw - (long long)wk * nseg) * seglen;
        const double* __restrict__ times = times_all + t_lo;
        const int nT = min(seglen, nT_all - t_lo);
        const int nrounds = (nT + round_span - 1) / round_span;
        __syncthreads();
        if (tid == 0) walker_prelude_orbit<T>(params + (size_t)wk * nparams, nparams, t_exp, &sw);
        if (tid == 32) walker_prelude_shape<T>(params + (size_t)wk * nparams, nparams, &sw);
        __syncthreads();
        const bool valid = sw.valid != 0;
        double acc = 0.0;   // this thread's chi^2 terms
        T* frow = flux ? flux + (size_t)wk * nT_all + t_lo : nullptr;

        if (!valid) {
            if (frow)
                for (int i = crank * NT + tid; i < nT; i += csize * NT) frow[i] = T(NAN);
            acc = (double)INFINITY;
        } else {
            const WalkerT<T> v = narrow<T>(sw);
            const double hwin = sw.half_win_phase, hard_ph = sw.hard_phase;
            for (int round = 0; round < nrounds; ++round) {
                const int i0 = (round * csize + crank) * tile;
                // ---- pass 1: classify this thread's exposures of the tile against the window;
                // out-of-window ones are finished here
                unsigned mask = 0;    // bit r: exposure i0 + r NT + tid is in the window
                unsigned early = 0;   // ... and near its edge (ingress / egress): listed first
                int wcount = 0, wearly = 0;
#pragma unroll 2
                for (int r = 0; r < nsub; ++r) {
                    const int i = i0 + r * NT + tid;
                    bool inwin = false, isearly = false;
                    if (i < nT) {
                        const double ph = reduced_phase(sw, times[i]);
                        inwin = fabs(ph) < hwin;
                        isearly = inwin && !(fabs(ph) < hard_ph);
                        if (want_chi2 && !shared_base) {
                            const T r2 = residual_sq<T>(obs[i] - 1.0, T(0), sigma[i]);
                            if (!inwin) acc += (double)r2;
                        }
                        if (!inwin && frow) frow[i] = T(1);
                    }
                    mask |= (inwin ? 1u : 0u) << r;
                    early |= (isearly ? 1u : 0u) << r;
                    wcount += __popc(__ballot_sync(0xffffffffu, inwin));
                    wearly += __popc(__ballot_sync(0xffffffffu, isearly));
                }
                if (lane == 0) {
                    s_cnt[0][warp] = wearly;
                    s_cnt[1][warp] = wcount - wearly;
                }
                // nobody may still be reading the lists of the previous round / walker
                GLH_DELAY(13);
                if (lists_live) cluster.sync(); else __syncthreads();
                // ---- pass 2: compact the in-window indices into this CTA's list: early entries
                // first, then the rest, each ordered by (warp, sub-chunk, lane) -- fixed for a given
                // launch, so chi^2 is reproducible
                {
                    int base0 = 0, tot0 = 0, base1 = 0, tot1 = 0;
#pragma unroll
                    for (int q = 0; q < NW; ++q) {
                        if (q == warp) {
                            base0 = tot0;
                            base1 = tot1;
                        }
                        tot0 += s_cnt[0][q];
                        tot1 += s_cnt[1][q];
                    }
                    base1 += tot0;
                    if (wcount) {
                        for (int r = 0; r < nsub; ++r) {
                            const bool b0 = (early >> r) & 1u, b1 = ((mask & ~early) >> r) & 1u;
                            const unsigned bal0 = __ballot_sync(0xffffffffu, b0);
                            const unsigned bal1 = __ballot_sync(0xffffffffu, b1);
                            const unsigned lt = (1u << lane) - 1u;
                            GLH_ASSERT(!b0 || base0 + __popc(bal0 & lt) < MAXTILE);
                            GLH_ASSERT(!b1 || base1 + __popc(bal1 & lt) < MAXTILE);
                            if (b0) s_list[base0 + __popc(bal0 & lt)] = i0 + r * NT + tid;
                            if (b1) s_list[base1 + __popc(bal1 & lt)] = i0 + r * NT + tid;
                            base0 += __popc(bal0);
                            base1 += __popc(bal1);
                        }
                    }
                    if (tid == 0) {
                        s_nlist[0] = tot0;
                        s_nlist[1] = tot1;
                    }
                }
                // ---- share the round's list over the cluster.  Cluster-wide order: the early
                // entries of CTA 0, 1, ..., then the remaining entries of CTA 0, 1, ...
                GLH_DELAY(14);
                cluster.sync();
                lists_live = true;
                GLH_DELAY(15);
                if (tid < 2) {
                    int run = 0;
                    for (int r = 0; r < csize; ++r) {
                        s_pre[tid][r] = run;
                        run += *cluster.map_shared_rank(&s_nlist[tid], r);
                    }
                    for (int r = csize; r <= MAXCLUSTER; ++r) s_pre[tid][r] = run;
                }
                __syncthreads();
                const int M0 = s_pre[0][MAXCLUSTER], M = M0 + s_pre[1][MAXCLUSTER];
                auto fetch = [&](int p) {   // p-th entry of the cluster-wide list
                    const int k = p >= M0 ? 1 : 0;
                    const int q = p - (k ? M0 : 0);
                    int r = 0;
#pragma unroll
                    for (int c = 1; c < MAXCLUSTER; ++c) r += (q >= s_pre[k][c] && c < csize) ? 1 : 0;
                    const int local = q - s_pre[k][r] + (k ? s_pre[0][r + 1] - s_pre[0][r] : 0);
                    GLH_ASSERT(r >= 0 && r < csize && local >= 0 && local < MAXTILE);
                    return *cluster.map_shared_rank(&s_list[local], r);
                };
                // ---- evaluate the round's list: the cluster's warps take groups of exposures in
                // turn (interleaved, so that ingress and egress are spread over every warp), each
                // warp on its own (no block barriers)
                const int gwarp = warp * csize + crank, gstride = csize * NW;   // CTAs first: the early (expensive)
                                                                            // groups land on different SMs
                if (n_ss <= 32) {
                    // a lane takes JS consecutive sub-exposures of one exposure, a warp G = 32 / JB
                    // whole exposures (JB = blocks of JS per exposure).  Sparse lists (K2-shaped:
                    // fewer pairs than the cluster has lanes) use JS = 1, one pair per lane; dense
                    // lists raise JS up to n_ss, which amortises the list fetch, the mean and the
                    // residual over more arithmetic and fills all 32 lanes.
                    const long long pairs = (long long)M * n_ss;
                    const int JS = (int)min((long long)n_ss, max(1LL, pairs / (4LL * 32 * gstride)));
                    const int JB = (n_ss + JS - 1) / JS, Gr = 32 / JB;
                    const int my_l = lane / JB, my_b = lane - my_l * JB;
                    // sweep k hands group k gstride + (warp order, reversed on odd sweeps): the warps
                    // that opened with the early (expensive) groups get the last groups, if any
                    const int nsweeps = (M + gstride * Gr - 1) / (gstride * Gr);
                    for (int k = 0; k < nsweeps; ++k) {
                        const int p0 = (k * gstride + ((k & 1) ? gstride - 1 - gwarp : gwarp)) * Gr;
                        if (p0 >= M) continue;   // warp-uniform
                        const int p = p0 + my_l;
                        const bool active = (my_l < Gr) && (p < M);
                        int i = 0;
                        T delta = T(0);
                        if (active) {
                            i = fetch(p);
                            const double tc = times[i];
                            for (int j = my_b * JS; j < min(n_ss, (my_b + 1) * JS); ++j) {
                                const double t = tc + (((double)j + 0.5) * inv_ss - 0.5) * t_exp;
                                delta += blocked_fraction<T, EX>(s_trap, sw, v, reduced_phase(sw, t));
                            }
                        }
                        T sum = T(0);   // exposure mean, blocks in sub-exposure order (R18)
                        for (int bb = 0; bb < JB; ++bb)
                            sum += __shfl_sync(0xffffffffu, delta, (lane + bb) & 31);
                        if (active && my_b == 0) {
                            const T dbar = sum * T(inv_ss);
                            GLH_ASSERT(i >= 0 && i < nT);
                            if (frow) frow[i] = T(1) - dbar;
                            if (want_chi2) acc += listed_residual<T>(obs[i] - 1.0, dbar, sigma[i], shared_base);
                        }
                    }
                } else {
                    // more sub-exposures than lanes: one exposure per warp, lanes stride over j
                    for (int p = gwarp; p < M; p += gstride) {
                        const int i = fetch(p);
                        const double tc = times[i];
                        T sum = T(0);
                        for (int j = lane; j < n_ss; j += 32) {
                            const double t = tc + (((double)j + 0.5) * inv_ss - 0.5) * t_exp;
                            sum += blocked_fraction<T, EX>(s_trap, sw, v, reduced_phase(sw, t));
                        }
#pragma unroll
                        for (int off = 16; off > 0; off >>= 1)
                            sum += __shfl_xor_sync(0xffffffffu, sum, off);
                        if (lane == 0) {
                            const T dbar = sum * T(inv_ss);
                            if (frow) frow[i] = T(1) - dbar;
                            if (want_chi2) acc += listed_residual<T>(obs[i] - 1.0, dbar, sigma[i], shared_base);
                        }
                    }
                }
            }
        }
        // ---- chi^2: CTA sum; every CTA PUSHES its partial into rank 0's shared memory over DSMEM,
        // one cluster barrier, then rank 0 adds them in rank order.  Nothing is read remotely after
        // that barrier, so the other CTAs may move on (or exit) at once.  The slots alternate with
        // the walker parity: a slot is rewritten two walkers later, i.e. after a barrier that rank 0
        // can only pass once it has read the slot.
        if (want_chi2) {
            const double tot = block_sum(acc, s_red);
            GLH_DELAY(16);
            if (tid == 0) *cluster.map_shared_rank(&s_gather[wpar][crank], 0) = tot;
            GLH_DELAY(17);
            cluster.sync();
            GLH_DELAY(18);
            lists_live = false;   // every CTA is past its evaluation
            if (crank == 0 && tid == 0) {
                double c2 = 0.0;
                for (int r = 0; r < csize; ++r) c2 += s_gather[wpar][r];
                if (shared_base) {
                    // baseline_kernel left sum_i ((obs_i - 1)/sigma_i)^2 in chi2[wk]; it was launched
                    // before this grid, which may have started early (programmatic dependent launch)
                    asm volatile("griddepcontrol.wait;" ::: "memory");
                    c2 += (double)*(volatile T*)&chi2[wk];
                }
                chi2[wk] = valid ? T(c2) : T(INFINITY);
            }
            wpar ^= 1;
        }
    }
    // no CTA may exit while a neighbour can still read its lists (flux-only calls: no barrier above)
    if (lists_live) cluster.sync();
}

// ------------------------------------------------------------------------------------------
// Steps a3 + a4 alone, one bare geometry per thread (config 5 of BASELINE.json).
// row = (d, Rp, f_proj, PA, u1, u2): planet centre at (d, 0), major axis at angle PA from +x, so
// in the kernel frame the centre is (d cos PA, -d sin PA).
// ------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(NT)
geometry_kernel(const double* __restrict__ geom, long long N, T* __restrict__ out) {
    __shared__ glf::TrapNode s_trap[16];
    if (threadIdx.x < 16)
        s_trap[threadIdx.x] = glf::TrapNode{glf::c_trap_cos[threadIdx.x], glf::c_trap_sin[threadIdx.x]};
    __syncthreads();
    const long long k = (long long)blockIdx.x * NT + threadIdx.x;
    if (k >= N) return;
    const double* g = geom + k * GL_NGEOM;
    const double d = g[0], Rp = g[1], fp = g[2], pa = g[3], u1 = g[4], u2 = g[5];
    const double norm = 1.0 - u1 / 3.0 - u2 / 6.0;
    bool ok = isfinite(d) && isfinite(Rp) && isfinite(fp) && isfinite(pa) && isfinite(u1) &&
              isfinite(u2) && (d >= 0.0) && (Rp > 0.0) && (Rp < 0.5) && (fp >= 0.0) && (fp < 1.0) &&
              (norm > 0.0);
    if (!ok) {
        out[k] = T(NAN);
        return;
    }
    T s, c;
    glc::gsincos(T(pa), &s, &c);
    const T a = T(Rp), b = T(Rp * (1.0 - fp));
    const double pn = kPi * norm;
    const T delta = blocked_at<T>(s_trap, T(d) * c, -T(d) * s, a, b, T((1.0 - u1 - 2.0 * u2) / pn),
                                  T((u1 + 2.0 * u2) / pn), T(u2 / pn));
    out[k] = T(1) - delta;
}

// fp32 production version of the above.  Bare geometries arrive in random order (config 5: 76 % inside
// the disc, 14 % crossing the limb, 10 % outside, plus forced tangent / grazing / four-crossing rows),
// and with one row per thread in input order a warp executed every code path for a few lanes each
// (7.8 of 32 lanes active per instruction; a three-bin ordering per CTA reached 16.8: round 1).  Here a
// CTA takes GEO_ROWS rows and SORTS them by the code path they will really take, in two stages:
//   stage 1  validity, kernel-frame centre, path_of() (gl_hot.cuh): no overlap -> done; 6 / 8 / 16 fixed
//            nodes -> three lists; near the limb -> a fourth list
//   stage 2  the three fixed-node lists, one after the other, full warps (glh::cheap_delta)
//   stage 3  near-limb rows: evolute test (only rows whose star centre may lie inside the outline's
//            evolute take the generic bracketed search) and the farthest point; what comes out -- inside
//            with 16 or 32 nodes, two crossings, evolute -- is listed again
//   stage 4  those three lists, full warps each (glh::near_rest, glc::overlap_areas)
// Outputs go to fixed slots, so the order inside a list (atomics) does not matter.
constexpr int GEO_NT = 256, GEO_PER = 4, GEO_ROWS = GEO_NT * GEO_PER;
constexpr uint32_t GEO_MARK = 0x7fc0deadu;   // "left to geometry_evolute_kernel": a quiet NaN no arithmetic here produces
__global__ void __launch_bounds__(GEO_NT)
geometry_sorted_kernel(const double* __restrict__ geom, long long N, float* __restrict__ out) {
    __shared__ glf::TrapNode s_trap[16];
    __shared__ float s_par[7][GEO_ROWS];        // xc, yc (folded), a, b, k0, k1, k2 of the CTA's rows
    __shared__ float s_far[2][GEO_ROWS];        // near-limb rows: farthest outline point (cos, sin)
    __shared__ unsigned short s_ord[GEO_ROWS];  // stage-1 lists: paths 4, 3, 2, 1 one after the other
    __shared__ unsigned short s_ord2[GEO_ROWS]; // stage-3 lists: crossing, inside near the limb, evolute
    __shared__ int s_count[4], s_start[5], s_count2[3], s_start2[4];
    const int tid = threadIdx.x;
    asm volatile("griddepcontrol.launch_dependents;");   // geometry_evolute_kernel may become resident
    // node table of the fixed-angle rules (constant memory): the loads are issued now by the last 16 threads, the
    // values stored behind stage 1 -- nobody waits for the constant cache in front of the kernel's first barrier
    float2 trap_mine = make_float2(0.f, 0.f);
    if (tid >= GEO_NT - 16) trap_mine = glh::c_trap16[tid - (GEO_NT - 16)];
    if (tid < 4) s_count[tid] = 0;
    if (tid < 3) s_count2[tid] = 0;
    __syncthreads();
    // rows are dealt to the CTAs in blocks of 32 (one coalesced 1.5 KB read per warp), ROUND-ROBIN: local
    // row loc sits in block (loc / 32) gridDim.x + blockIdx.x.  A stretch of the input full of one
    // expensive kind of geometry (config 5 ends with 100 000 forced rows) is thereby spread over the
    // whole grid instead of landing on a few CTAs that finish long after the others.
    auto row_of = [&](int loc) {
        return ((long long)(loc >> 5) * gridDim.x + blockIdx.x) * 32 + (loc & 31);
    };
    int path[GEO_PER], slot[GEO_PER];
#pragma unroll
    for (int q = 0; q < GEO_PER; ++q) {
        const int loc = q * GEO_NT + tid;
        const long long k = row_of(loc);
        path[q] = 0;
        slot[q] = 0;
        if (k >= N) continue;
        const double* g = geom + k * GL_NGEOM;
        const double d = g[0], Rp = g[1], fp = g[2], pa = g[3], u1 = g[4], u2 = g[5];
        const double norm = 1.0 - u1 / 3.0 - u2 / 6.0;
        const bool ok = isfinite(d) && isfinite(Rp) && isfinite(fp) && isfinite(pa) && isfinite(u1) &&
                        isfinite(u2) && (d >= 0.0) && (Rp > 0.0) && (Rp < 0.5) && (fp >= 0.0) &&
                        (fp < 1.0) && (norm > 0.0);
        if (!ok) {
            out[k] = NAN;
            continue;
        }
        float s, c;
        glh::angle_sincos(pa, &s, &c);
        const float a = (float)Rp, b = (float)(Rp * (1.0 - fp)), r0 = (float)d;
        const float xc = fabsf(r0 * c), yc = fabsf(r0 * s);
        float r0r;
        path[q] = glh::path_of(fmaf(xc, xc, yc * yc), a, &r0r);
        if (path[q] == 0) {   // no overlap
            out[k] = 1.f;
            continue;
        }
        const float ipn = glh::rcp_nr((float)(kPi * norm));
        s_par[0][loc] = xc;
        s_par[1][loc] = yc;
        s_par[2][loc] = a;
        s_par[3][loc] = b;
        s_par[4][loc] = (float)(1.0 - u1 - 2.0 * u2) * ipn;
        s_par[5][loc] = (float)(u1 + 2.0 * u2) * ipn;
        s_par[6][loc] = (float)u2 * ipn;
        slot[q] = atomicAdd(&s_count[4 - path[q]], 1);   // list 0 = path 4 (the long one first)
    }
    if (tid >= GEO_NT - 16) s_trap[tid - (GEO_NT - 16)] = glf::TrapNode{trap_mine.x, trap_mine.y};
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        for (int l = 0; l < 4; ++l) {
            s_start[l] = run;
            run += s_count[l];
        }
        s_start[4] = run;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < GEO_PER; ++q)
        if (path[q] > 0) s_ord[s_start[4 - path[q]] + slot[q]] = (unsigned short)(q * GEO_NT + tid);
    __syncthreads();
    const int n_near = s_start[1], n_all = s_start[4];
    // ---- stage 2: fixed-node rules (lists 1..3 = paths 3, 2, 1)
    for (int j = n_near + tid; j < n_all; j += GEO_NT) {
        const int loc = s_ord[j];
        const int pth = j < s_start[2] ? 3 : (j < s_start[3] ? 2 : 1);
        const float xc = s_par[0][loc], yc = s_par[1][loc], a = s_par[2][loc], b = s_par[3][loc];
        const float delta = glh::cheap_delta(s_trap, pth, xc, yc, fmaf(xc, xc, yc * yc), a, b, a * b, s_par[4][loc],
                                             s_par[5][loc], s_par[6][loc]);
        out[row_of(loc)] = 1.f - delta;
    }
    // ---- stage 3: near-limb rows: which of them need the generic search, farthest point of the others
    for (int j = tid; j < n_near; j += GEO_NT) {
        const int loc = s_ord[j];
        const float xc = s_par[0][loc], yc = s_par[1][loc], a = s_par[2][loc], b = s_par[3][loc];
        const float e2 = (a - b) * (a + b), Aa = a * xc, Bb = b * yc;
        int lst;
        if (Aa < e2 && Bb < e2 && glf::evolute_inside(Aa, Bb, e2)) {
            // the generic bracketed search is ~10x longer than anything else here: left to
            // geometry_evolute_kernel, which gathers these rows from the whole grid into full warps
            out[row_of(loc)] = __uint_as_float(GEO_MARK);
            s_ord2[j] = 0xffffu;
            continue;
        } else {
            const float rn = glf::mufu_rsqrt(fmaf(Aa, Aa, Bb * Bb));
            float cf = Aa * rn, sf = Bb * rn;
            glh::critical_point_rt(xc, yc, a, b, 1.f, &cf, &sf);
            s_far[0][loc] = cf;
            s_far[1][loc] = sf;
            const float xf = fmaf(a, cf, xc), yf = fmaf(b, sf, yc);
            lst = fmaf(xf, xf, fmaf(yf, yf, -1.f)) <= 0.f ? 1 : 0;
        }
        const int sl = atomicAdd(&s_count2[lst], 1);
        // (positions inside a list are final only after the counts are: keep (list, slot) in s_ord2 for now)
        s_ord2[j] = (unsigned short)((lst << 12) | sl);
    }
    __syncthreads();
    if (tid == 0) {
        s_start2[0] = 0;
        s_start2[1] = s_count2[0];
        s_start2[2] = s_count2[0] + s_count2[1];
        s_start2[3] = s_count2[0] + s_count2[1] + s_count2[2];
    }
    __syncthreads();
    // scatter the row numbers to their final positions (through registers: s_ord2 is rewritten in place)
    {
        int locs[GEO_PER], poss[GEO_PER];
#pragma unroll
        for (int q = 0; q < GEO_PER; ++q) {
            const int j = q * GEO_NT + tid;
            poss[q] = -1;
            locs[q] = 0;
            if (j < n_near && s_ord2[j] != 0xffffu) {
                const int code = s_ord2[j];
                poss[q] = s_start2[code >> 12] + (code & 0xfff);
                locs[q] = s_ord[j];
            }
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < GEO_PER; ++q)
            if (poss[q] >= 0) s_ord2[poss[q]] = (unsigned short)locs[q];
    }
    __syncthreads();
    // ---- stage 4: two crossings / inside near the limb (evolute rows: geometry_evolute_kernel)
    const int n_stage4 = s_start2[2];
    for (int j = tid; j < n_stage4; j += GEO_NT) {
        const int loc = s_ord2[j];
        const float xc = s_par[0][loc], yc = s_par[1][loc], a = s_par[2][loc], b = s_par[3][loc];
        const float Aa = a * xc, Bb = b * yc;
        const float rn = glf::mufu_rsqrt(fmaf(Aa, Aa, Bb * Bb));
        const float delta = glh::near_rest<false>(s_trap, xc, yc, fmaf(xc, xc, yc * yc), a, b, a * b,
                                                  (a - b) * (a + b), s_par[4][loc], s_par[5][loc], s_par[6][loc],
                                                  s_far[0][loc], s_far[1][loc], -(Aa * rn), -(Bb * rn), 0,
                                                  0xffffffffu);
        out[row_of(loc)] = 1.f - delta;
    }
}

// Second launch of the fp32 bare-geometry call (programmatic dependent launch behind
// geometry_sorted_kernel): the rows that kernel marked -- star centre possibly inside the outline's
// evolute: up to four crossings, generic bracketed search (gl_core.cuh).  They are few (config 5: a few per
// cent) and ~10x longer than any other row.  A CTA walks its share of the output in rounds of EVO_ROWS rows,
// keeps appending the marked ones to one list (ballot + one shared counter update per warp) and evaluates the
// list when the next round might overflow it or at the end.  Grid: EVO_CTAS_PER_SM CTAs per SM (what fits at
// 55 registers and 40 KB of shared memory): one evaluation is a long dependent chain, so warps in flight count
// for more than full lists -- config 5 (1e6 rows), the whole call: 2 per SM 72.9 us, 3 70.1, 4 68.1, 5 (a
// second wave) 86.3.
constexpr int EVO_NT = 256, EVO_ROWS = 256, EVO_CAP = 512;   // rows looked at per round; list capacity
constexpr int EVO_CTAS_PER_SM = 4;
// The evaluation itself is glc::overlap_areas cut at its stage boundaries (gl_core.cuh), with the rows
// RE-LISTED between the stages, so that a warp runs one stage for 32 rows that all need it:
//   E1  every listed row: critical points of g (3 root searches); outline wholly inside the disc -> its arcs
//       are known; else the row goes on the crossing list
//   E2  crossing list: nearest point, exit and entry crossings (2-5 root searches) -> arcs, or no overlap
//   E3  arc list, one lane per ARC (a row has one or two): the three boundary integrals of the arc
//   E4  every row with arcs: the arcs' sums in arc order, the limb arcs that close the contour, the flux
// Every result lands in a slot fixed by its row (and arc number): the order in which rows enter a list
// (atomics) changes nothing.  Measured on config 5: one lane per row through all of overlap_areas ran at 9.5 of
// 32 lanes, 13.6 M warp instructions, 54 us; staged 16.5 lanes, 9.5 M, 34.6 us (the call: 89.9 -> 68.1 us).
struct EvoRow {
    glc::Outline<float> o;
    float k0, k1, k2;
};
__device__ __forceinline__ EvoRow evo_row(const double* __restrict__ geom, long long k) {
    const double* g = geom + k * GL_NGEOM;
    const double d = g[0], Rp = g[1], fp = g[2], pa = g[3], u1 = g[4], u2 = g[5];
    float s, c;
    glh::angle_sincos(pa, &s, &c);   // (the same preparation as geometry_sorted_kernel)
    const float a = (float)Rp, b = (float)(Rp * (1.0 - fp)), r0 = (float)d;
    const float ipn = glh::rcp_nr((float)(kPi * (1.0 - u1 / 3.0 - u2 / 6.0)));
    EvoRow r;
    r.o = glc::make_outline(fabsf(r0 * c), fabsf(r0 * s), a, b);
    r.k0 = (float)(1.0 - u1 - 2.0 * u2) * ipn;
    r.k1 = (float)(u1 + 2.0 * u2) * ipn;
    r.k2 = (float)u2 * ipn;
    return r;
}
__global__ void __launch_bounds__(EVO_NT)
geometry_evolute_kernel(const double* __restrict__ geom, long long N, float* out) {
    __shared__ long long s_rows[EVO_CAP];
    __shared__ float s_cp[6][EVO_CAP];            // tfar, gfar, ta, tb, ga, gb of a row
    __shared__ unsigned char s_flag[EVO_CAP];     // bit 0: the pair (ta, tb) exists; bits 1-2: arcs; bit 3: limb
    __shared__ unsigned short s_cross[EVO_CAP];   // E2's list (positions in s_rows)
    __shared__ unsigned short s_arcs[2 * EVO_CAP];   // E3's list (arc slots: 2 * position + arc number)
    __shared__ float s_as[2 * EVO_CAP], s_ae[2 * EVO_CAP], s_A[3][2 * EVO_CAP];   // per arc slot
    __shared__ int s_n, s_ncross, s_narcs;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_n = 0;
    // the quadrature table (constant memory) is copied while this grid still waits for the first kernel: E3
    // finds it in shared memory instead of missing the constant cache on its critical path
    __shared__ float s_gl[16];
    if (tid < 8) {
        s_gl[tid] = glf::c_gl_phi[tid];
        s_gl[8 + tid] = glf::c_gl_om[tid];
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");
    __syncthreads();
    // warp-aggregated append to a shared list (the ballot is taken by all 32 lanes)
    auto append = [&](bool mine, int* counter, unsigned short* list, int capacity, int value) {
        const unsigned bal = __ballot_sync(0xffffffffu, mine);
        if (!bal) return;
        int base = 0;
        if (lane == 0) base = atomicAdd(counter, __popc(bal));
        base = __shfl_sync(0xffffffffu, base, 0);
        GLH_ASSERT(base >= 0 && base + __popc(bal) <= capacity);
        (void)capacity;
        if (mine) list[base + __popc(bal & ((1u << lane) - 1u))] = (unsigned short)value;
    };
    auto push_arcs = [&](int j, const glc::ArcPlan<float>& pl) {   // (narc > 0)
        s_flag[j] = (unsigned char)((s_flag[j] & 1u) | (pl.narc << 1) | (pl.limb ? 8u : 0u));
        for (int i = 0; i < pl.narc; ++i) {
            s_as[2 * j + i] = pl.as[i];
            s_ae[2 * j + i] = pl.ae[i];
        }
    };
    auto evaluate = [&](int n) {
        if (tid == 0) s_ncross = s_narcs = 0;
        __syncthreads();
        // ---- E1
        for (int j0 = 0; j0 < n; j0 += EVO_NT) {   // (whole warps stay in the loop: the appends vote)
            const int j = j0 + tid;
            bool cross = false;
            int narc = 0;
            if (j < n) {
                const EvoRow r = evo_row(geom, s_rows[j]);
                glc::CritPoints<float> cp;
                s_flag[j] = 0;
                if (!glc::critical_points<float, true>(r.o, &cp)) {
                    out[s_rows[j]] = 1.f;
                } else {
                    s_cp[0][j] = cp.tfar;
                    s_cp[1][j] = cp.gfar;
                    s_cp[2][j] = cp.ta;
                    s_cp[3][j] = cp.tb;
                    s_cp[4][j] = cp.ga;
                    s_cp[5][j] = cp.gb;
                    s_flag[j] = cp.evol ? 1 : 0;
                    if (cp.gfar <= 0.f) {
                        glc::ArcPlan<float> pl;
                        glc::plan_inside(cp, &pl);
                        push_arcs(j, pl);
                        narc = pl.narc;
                    } else {
                        cross = true;
                    }
                }
            }
            append(cross, &s_ncross, s_cross, EVO_CAP, j);
            append(narc >= 1, &s_narcs, s_arcs, 2 * EVO_CAP, 2 * j);
            append(narc == 2, &s_narcs, s_arcs, 2 * EVO_CAP, 2 * j + 1);
        }
        __syncthreads();
        // ---- E2
        const int ncross = s_ncross;
        for (int q0 = 0; q0 < ncross; q0 += EVO_NT) {
            const int q = q0 + tid;
            int narc = 0, j = 0;
            if (q < ncross) {
                j = s_cross[q];
                const EvoRow r = evo_row(geom, s_rows[j]);
                glc::CritPoints<float> cp;
                cp.tfar = s_cp[0][j];
                cp.gfar = s_cp[1][j];
                cp.ta = s_cp[2][j];
                cp.tb = s_cp[3][j];
                cp.ga = s_cp[4][j];
                cp.gb = s_cp[5][j];
                cp.evol = (s_flag[j] & 1u) != 0;
                glc::ArcPlan<float> pl;
                glc::plan_crossing<float, true>(r.o, cp, &pl);
                if (pl.narc == 0) out[s_rows[j]] = 1.f;
                else push_arcs(j, pl);
                narc = pl.narc;
            }
            append(narc >= 1, &s_narcs, s_arcs, 2 * EVO_CAP, 2 * j);
            append(narc == 2, &s_narcs, s_arcs, 2 * EVO_CAP, 2 * j + 1);
        }
        __syncthreads();
        // ---- E3
        const int narcs = s_narcs;
        for (int q = tid; q < narcs; q += EVO_NT) {
            const int slot = s_arcs[q];
            const EvoRow r = evo_row(geom, s_rows[slot >> 1]);
            const glc::ArcCoef<float> kc = glc::arc_coefficients(r.o);
            const float t1 = s_as[slot], t2 = s_ae[slot];
            float s1, c1, s2, c2, A[3] = {0.f, 0.f, 0.f};
            glc::gtrig<true>(t1, &s1, &c1);
            glc::gtrig<true>(t2, &s2, &c2);
            glc::add_outline_arc<float, 16, true>(r.o, kc, t1, s1, c1, t2, s2, c2, s_gl, s_gl + 8, A);
            s_A[0][slot] = A[0];
            s_A[1][slot] = A[1];
            s_A[2][slot] = A[2];
        }
        __syncthreads();
        // ---- E4
        for (int j = tid; j < n; j += EVO_NT) {
            const int narc = (s_flag[j] >> 1) & 3;
            if (narc == 0) continue;
            const EvoRow r = evo_row(geom, s_rows[j]);
            float A[3] = {0.f, 0.f, 0.f};
            for (int i = 0; i < narc; ++i) {
                A[0] += s_A[0][2 * j + i];
                A[1] += s_A[1][2 * j + i];
                A[2] += s_A[2][2 * j + i];
            }
            if (s_flag[j] & 8u) {
                float ss[2], cs[2], se[2], ce[2];
                for (int i = 0; i < narc; ++i) {
                    glc::gtrig<true>(s_as[2 * j + i], &ss[i], &cs[i]);
                    glc::gtrig<true>(s_ae[2 * j + i], &se[i], &ce[i]);
                }
                for (int i = 0; i < narc; ++i) {
                    const int i2 = (i + 1 == narc) ? 0 : i + 1;
                    glc::add_limb_arc(r.o.xc + r.o.a * ce[i], r.o.yc + r.o.b * se[i], r.o.xc + r.o.a * cs[i2],
                                      r.o.yc + r.o.b * ss[i2], A);
                }
            }
            out[s_rows[j]] = 1.f - fmaf(r.k0, A[0], fmaf(r.k1, A[1], r.k2 * A[2]));
        }
    };
    // blocks of 32 rows, round-robin over the CTAs (see geometry_sorted_kernel); warp w of the CTA takes
    // the CTA's blocks w, w + 8, ... of a round
    const long long nblocks = (N + 31) / 32;
    for (long long b0 = blockIdx.x; b0 < nblocks; b0 += (long long)gridDim.x * (EVO_ROWS / 32)) {
        for (int r = warp; r < EVO_ROWS / 32; r += EVO_NT / 32) {
            const long long blk = b0 + (long long)r * gridDim.x;
            const long long k = blk * 32 + lane;
            const bool marked = blk < nblocks && k < N &&
                                *reinterpret_cast<const volatile uint32_t*>(out + k) == GEO_MARK;
            const unsigned bal = __ballot_sync(0xffffffffu, marked);
            if (bal) {   // (warp-uniform)
                int base = 0;
                if (lane == 0) base = atomicAdd(&s_n, __popc(bal));
                base = __shfl_sync(0xffffffffu, base, 0);
                GLH_ASSERT(base >= 0 && base + __popc(bal) <= EVO_CAP);
                if (marked) s_rows[base + __popc(bal & ((1u << lane) - 1u))] = k;
            }
        }
        __syncthreads();
        const int n = s_n;
        if (n > EVO_CAP - EVO_ROWS) {   // the next round might not fit: evaluate what is listed (CTA-uniform)
            evaluate(n);
            __syncthreads();
            if (tid == 0) s_n = 0;
            __syncthreads();
        }
    }
    evaluate(s_n);
}

// ------------------------------------------------------------------------------------------
// Ceiling probes (gl_probe_peaks): 8 independent register-only chains per thread.
// ------------------------------------------------------------------------------------------
__global__ void empty_kernel(int dependent) {
    if (dependent) asm volatile("griddepcontrol.wait;" ::: "memory");
    else asm volatile("griddepcontrol.launch_dependents;");
}
template <typename T> __global__ void probe_fma(T* out, int iters, T a, T b) {
    T x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = T(threadIdx.x + i);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) x[i] = x[i] * a + b;
    }
    T s = T(0);
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void probe_mufu(float* out, int iters) {
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = 1.5f + threadIdx.x + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

// ==========================================================================================
// Host side: table upload, launch configuration, C ABI.
// ==========================================================================================
namespace {

thread_local long long tl_launches = 0;
thread_local char tl_cuda_err[256] = "";

int cuda_fail(cudaError_t e, const char* where) {
    snprintf(tl_cuda_err, sizeof(tl_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return GL_ECUDA;
}

// Quadrature tables go to constant memory once per device (immutable afterwards).
int ensure_tables() {
    static std::mutex mu;
    static unsigned long long done_mask = 0;   // devices 0..63
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    std::lock_guard<std::mutex> lock(mu);
    if (dev < 64 && (done_mask >> dev) & 1ull) return GL_OK;
    float p32[NQ32 / 2], o32[NQ32 / 2];
    double p64[NQ64 / 2], o64[NQ64 / 2];
    glt::smoothed_gauss_legendre<float>(NQ32, p32, o32);
    glt::smoothed_gauss_legendre<double>(NQ64, p64, o64);
    float tc[16], ts[16];
    for (int k = 0; k < 16; ++k) {
        tc[k] = (float)cosl(3.141592653589793238462643383279502884L * k / 16.0L);
        ts[k] = (float)sinl(3.141592653589793238462643383279502884L * k / 16.0L);
    }
    tc[8] = 0.f;   // exact zeros at the axes
    ts[0] = 0.f;
    if ((e = cudaMemcpyToSymbol(glf::c_gl_phi, p32, sizeof(p32))) != cudaSuccess ||
        (e = cudaMemcpyToSymbol(glf::c_gl_om, o32, sizeof(o32))) != cudaSuccess ||
        (e = cudaMemcpyToSymbol(glf::c_trap_cos, tc, sizeof(tc))) != cudaSuccess ||
        (e = cudaMemcpyToSymbol(glf::c_trap_sin, ts, sizeof(ts))) != cudaSuccess ||
        (e = cudaMemcpyToSymbol(c_phi64, p64, sizeof(p64))) != cudaSuccess ||
        (e = cudaMemcpyToSymbol(c_om64, o64, sizeof(o64))) != cudaSuccess)
        return cuda_fail(e, "cudaMemcpyToSymbol");
    if (dev < 64) done_mask |= 1ull << dev;
    return GL_OK;
}

// Number of SMs of the current device (cached per device).
int sm_count() {
    static int cached[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    if (!cached[dev]) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cached[dev] = n;
    }
    return cached[dev];
}

// transit_kernel: cluster size C and tile length -- as many CTAs per walker as keep the whole batch
// resident in one wave (8 CTAs of 128 threads x 64 registers per SM), each with at least NT
// exposures; the tile is the CTA's share of the series, so that one round covers it unless
// T > C * MAXTILE.
void pick_shape(long long rows, int nT, int* C, int* tile) {
    const long long slots = (long long)sm_count() * 8;
    int c = 1;
    while (c < MAXCLUSTER && (long long)c * 2 * NT <= nT && rows * c * 2 <= slots) c *= 2;
    int t = ((nT + c - 1) / c + NT - 1) / NT * NT;
    t = t < NT ? NT : (t > MAXTILE ? MAXTILE : t);
    *C = c;
    *tile = t;
}

// One launch of transit_kernel<T, EX, SEG>.
template <typename T>
int launch_full(const double* params, int nparams, int B, const double* times, int nT, double t_exp,
                int n_ss, const double* obs, const double* sigma, void* flux, void* chi2,
                int shared_base, int nseg, int seglen, bool pdl, cudaStream_t st) {
    const long long units = (long long)B * nseg;
    const long long rows = units < 65535 ? units : 65535;
    int C, tile;
    pick_shape(rows, seglen, &C, &tile);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)C, (unsigned)rows, 1);
    cfg.blockDim = dim3(NT, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)C;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 2 : 1;
    auto launch = [&]() {
        if (nseg > 1)   // flux-only, 12-column rows or extended ones
            return (nparams == GL_NPARAMS_EX)
                       ? cudaLaunchKernelEx(&cfg, transit_kernel<T, true, true>, params, B, times, nT, tile,
                                            t_exp, n_ss, obs, sigma, (T*)flux, (T*)chi2, shared_base, nseg,
                                            seglen)
                       : cudaLaunchKernelEx(&cfg, transit_kernel<T, false, true>, params, B, times, nT, tile,
                                            t_exp, n_ss, obs, sigma, (T*)flux, (T*)chi2, shared_base, nseg,
                                            seglen);
        return (nparams == GL_NPARAMS_EX)
                   ? cudaLaunchKernelEx(&cfg, transit_kernel<T, true, false>, params, B, times, nT, tile,
                                        t_exp, n_ss, obs, sigma, (T*)flux, (T*)chi2, shared_base, 1, nT)
                   : cudaLaunchKernelEx(&cfg, transit_kernel<T, false, false>, params, B, times, nT, tile,
                                        t_exp, n_ss, obs, sigma, (T*)flux, (T*)chi2, shared_base, 1, nT);
    };
    cudaError_t e = launch();
    if (e != cudaSuccess && pdl) {
        // no early start then: plain stream order is just as correct
        (void)cudaGetLastError();
        cfg.numAttrs = 1;
        e = launch();
    }
    if (e != cudaSuccess) return cuda_fail(e, "transit_kernel launch");
    ++tl_launches;
    return GL_OK;
}

// Launch shape of hot_kernel (gl_hot.cuh).  chi^2 calls: one cluster of C CTAs per walker, C > 1 only
// when the batch alone does not fill the GPU (two CTAs of 512 threads per SM) and every CTA still
// gets >= 2048 exposures.  Flux-only calls: single-CTA units, a long series cut into segments
// (>= 512 exposures each) until the GPU is full.
struct HotShape {
    int C, nseg, seglen;
};
HotShape pick_hot_shape(int B, int nT, bool want_chi2) {
    const long long slots = (long long)sm_count() * 2;
    HotShape h = {1, 1, nT};
    if (want_chi2) {
        while (h.C < glh::MAXC && (long long)B * h.C * 2 <= slots && nT / (h.C * 2) >= 2048) h.C *= 2;
    } else {
        long long n = slots / B;
        const long long most = (nT + 511) / 512;
        if (n > most) n = most;
        if ((long long)B * n >= (1LL << 31)) n = 1;
        if (n > 1) {
            int len = (int)((nT + n - 1) / n);
            len = (len + 3) & ~3;
            h.seglen = len;
            h.nseg = (nT + len - 1) / len;
        }
    }
    return h;
}

struct SeriesView {          // what gl_series keeps resident (all nullptr / 0 for a plain call)
    const float2* ow = nullptr;
    double S = 0.0;
    int sorted_known = 0;
    int* done_count = nullptr;   // see glh::HotArgs
    int* done_flag = nullptr;
};

// fp32, 12-column rows, nT > 0: [baseline_kernel ->] hot_kernel.
int launch_hot(const double* params, int B, const double* times, int nT, double t_exp, int n_ss,
               const double* obs, const double* sigma, float* flux, float* chi2, const SeriesView& sv,
               cudaStream_t st) {
    const bool pre = sv.ow != nullptr, want_chi2 = chi2 != nullptr;
    const HotShape h = pick_hot_shape(B, nT, want_chi2);
    {   // (a walker off the common path runs the generic code, which reads the constant-memory tables)
        const int rc = ensure_tables();
        if (rc != GL_OK) return rc;
    }
    if (want_chi2 && !pre) {
        baseline_kernel<<<1, 1024, 0, st>>>(obs, sigma, nT, chi2, B);
        cudaError_t e0 = cudaGetLastError();
        if (e0 != cudaSuccess) return cuda_fail(e0, "baseline_kernel launch");
        ++tl_launches;
    }
    glh::HotArgs a;
    a.params = params;
    a.times = times;
    a.obs = obs;
    a.sigma = sigma;
    a.ow = sv.ow;
    a.flux = flux;
    a.chi2 = chi2;
    a.S = sv.S;
    a.t_exp = t_exp;
    a.inv_ss = 1.f / (float)n_ss;
    a.doff = (float)(t_exp / (double)n_ss);
    a.off0 = (float)((0.5 / (double)n_ss - 0.5) * t_exp);
    a.ss_magic = n_ss > 1 ? (unsigned)((0x100000000ULL + (unsigned long long)n_ss - 1) / (unsigned long long)n_ss) : 0u;
    a.B = B;
    a.T = nT;
    a.n_ss = n_ss;
    a.nseg = h.nseg;
    a.seglen = h.seglen;
    a.sorted_known = sv.sorted_known;
    a.done_count = sv.done_count;
    a.done_flag = sv.done_flag;
    const long long units = (long long)B * h.nseg;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)h.C, (unsigned)(units < 65535 ? units : 65535), 1);
    cfg.blockDim = dim3(glh::HOT_NT, 1, 1);
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (h.C > 1) {
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = (unsigned)h.C;
        attr[na].val.clusterDim.y = 1;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    const int na_plain = na;
    if (want_chi2 && !pre) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    auto launch = [&]() {
        return pre ? cudaLaunchKernelEx(&cfg, glh::hot_kernel<true>, a)
                   : cudaLaunchKernelEx(&cfg, glh::hot_kernel<false>, a);
    };
    cudaError_t e = launch();
    if (e != cudaSuccess && na != na_plain) {
        (void)cudaGetLastError();
        cfg.numAttrs = na_plain;
        e = launch();
    }
    if (e != cudaSuccess) return cuda_fail(e, "hot_kernel launch");
    ++tl_launches;
    return GL_OK;
}

template <typename T>
int launch_transit(const double* params, int nparams, int B, const double* times, int nT,
                   double t_exp, int n_ss,
                   const double* obs, const double* sigma, void* flux, void* chi2,
                   cudaStream_t st) {
    if (sizeof(T) == 4 && nparams == GL_NPARAMS && nT > 0)
        return launch_hot(params, B, times, nT, t_exp, n_ss, obs, sigma, (float*)flux, (float*)chi2,
                          SeriesView(), st);
    // flux-only calls with few walkers and a series longer than one round: split the series into
    // segments that separate clusters take (no reduction is needed between them)
    int C, tile;
    pick_shape(B, nT, &C, &tile);
    int nseg = 1, seglen = nT;
    if (chi2 == nullptr && nT > 0) {
        const long long span = (long long)C * tile;
        const long long rounds = (nT + span - 1) / span;
        const long long room = ((long long)sm_count() * 8) / ((long long)B * C);
        if (rounds > 1 && room > 1) {
            nseg = (int)(rounds < room ? rounds : room);
            const long long per = (rounds + nseg - 1) / nseg;   // rounds per segment
            seglen = (int)(per * span);
            nseg = (int)((nT + (long long)seglen - 1) / seglen);
        }
    }
    // fp32 chi^2: launch-wide baseline first, the transit kernel right behind it (see baseline_kernel)
    const int shared_base = (sizeof(T) == 4 && chi2 != nullptr && nT > 0) ? 1 : 0;
    if (shared_base) {
        baseline_kernel<<<1, 1024, 0, st>>>(obs, sigma, nT, (float*)chi2, B);
        cudaError_t e0 = cudaGetLastError();
        if (e0 != cudaSuccess) return cuda_fail(e0, "baseline_kernel launch");
        ++tl_launches;
    }
    return launch_full<T>(params, nparams, B, times, nT, t_exp, n_ss, obs, sigma, flux, chi2, shared_base,
                          nseg, seglen, shared_base != 0, st);
}

int run_transit(const double* params, int nparams, int B, const double* times, int nT, double t_exp,
                int n_ss,
                const double* obs, const double* sigma, void* flux, void* chi2, gl_dtype dtype,
                void* stream, bool need_flux, bool need_chi2) {
    if (B < 0 || nT < 0 || n_ss < 1 || !(t_exp >= 0.0) || !isfinite(t_exp)) return GL_EINVAL;
    if (dtype != GL_F32 && dtype != GL_F64) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if (nT == 0 && !need_chi2) return GL_OK;
    if (!params || (nT > 0 && !times)) return GL_EINVAL;
    if (need_flux && nT > 0 && !flux) return GL_EINVAL;
    if (need_chi2 && (!chi2 || (nT > 0 && (!obs || !sigma)))) return GL_EINVAL;
    if ((long long)B * (long long)nT >= (1LL << 40)) return GL_EUNSUPPORTED;
    int rc = ensure_tables();
    if (rc != GL_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    return dtype == GL_F32
               ? launch_transit<float>(params, nparams, B, times, nT, t_exp, n_ss, obs, sigma, flux,
                                       chi2, st)
               : launch_transit<double>(params, nparams, B, times, nT, t_exp, n_ss, obs, sigma, flux,
                                        chi2, st);
}

}  // namespace

extern "C" {

int gl_lightcurve(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                  void* flux_out, gl_dtype dtype, void* stream) {
    return run_transit(params, GL_NPARAMS, B, times, T, t_exp, n_ss, nullptr, nullptr, flux_out,
                       nullptr, dtype, stream, true, false);
}

int gl_lightcurve_ex(const double* params_ex, int B, const double* times, int T, double t_exp,
                     int n_ss, void* flux_out, gl_dtype dtype, void* stream) {
    return run_transit(params_ex, GL_NPARAMS_EX, B, times, T, t_exp, n_ss, nullptr, nullptr, flux_out,
                       nullptr, dtype, stream, true, false);
}

int gl_loglike_ex(const double* params_ex, int B, const double* times, int T, double t_exp, int n_ss,
                  const double* obs, const double* sigma, void* chi2_out, void* flux_out_or_null,
                  gl_dtype dtype, void* stream) {
    return run_transit(params_ex, GL_NPARAMS_EX, B, times, T, t_exp, n_ss, obs, sigma,
                       flux_out_or_null, chi2_out, dtype, stream, false, true);
}

int gl_loglike(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
               const double* obs, const double* sigma, void* chi2_out, void* flux_out_or_null,
               gl_dtype dtype, void* stream) {
    return run_transit(params, GL_NPARAMS, B, times, T, t_exp, n_ss, obs, sigma, flux_out_or_null,
                       chi2_out, dtype, stream, false, true);
}

int gl_flux_geometry(const double* geom, long long N, void* flux_out, gl_dtype dtype,
                     void* stream) {
    if (N < 0 || (dtype != GL_F32 && dtype != GL_F64)) return GL_EINVAL;
    if (N == 0) return GL_OK;
    if (!geom || !flux_out) return GL_EINVAL;
    if (N >= (1LL << 40)) return GL_EUNSUPPORTED;
    int rc = ensure_tables();
    if (rc != GL_OK) return rc;
    const unsigned blocks = (unsigned)((N + NT - 1) / NT);
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == GL_F32) {
        geometry_sorted_kernel<<<(unsigned)((N + GEO_ROWS - 1) / GEO_ROWS), GEO_NT, 0, st>>>(
            geom, N, (float*)flux_out);
        cudaError_t e1 = cudaGetLastError();
        if (e1 != cudaSuccess) return cuda_fail(e1, "geometry_sorted_kernel launch");
        ++tl_launches;
        cudaLaunchConfig_t cfg = {};
        {   // EVO_CTAS_PER_SM CTAs per SM, but no more than there are rounds of EVO_ROWS rows
            const long long want = (N + EVO_ROWS - 1) / EVO_ROWS, room = (long long)sm_count() * EVO_CTAS_PER_SM;
            cfg.gridDim = dim3((unsigned)(want < room ? want : room), 1, 1);
        }
        cfg.blockDim = dim3(EVO_NT, 1, 1);
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        e1 = cudaLaunchKernelEx(&cfg, geometry_evolute_kernel, geom, N, (float*)flux_out);
        if (e1 != cudaSuccess) return cuda_fail(e1, "geometry_evolute_kernel launch");
    } else
        geometry_kernel<double><<<blocks, NT, 0, st>>>(geom, N, (double*)flux_out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "geometry_kernel launch");
    ++tl_launches;
    return GL_OK;
}

int gl_flux_geometry_simpson(const double* geom, long long N, int n_intervals, void* flux_out,
                             gl_dtype dtype, void* stream) {
    if (N < 0 || (dtype != GL_F32 && dtype != GL_F64)) return GL_EINVAL;
    if (n_intervals < 2 || (n_intervals & 1) || n_intervals > (1 << 24)) return GL_EINVAL;
    if (N == 0) return GL_OK;
    if (!geom || !flux_out) return GL_EINVAL;
    if (N >= (1LL << 40)) return GL_EUNSUPPORTED;
    const long long threads = N * 32;   // one warp per geometry
    const long long blocks = (threads + 127) / 128;
    if (blocks > 0x7fffffffLL) return GL_EUNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == GL_F32)
        gls::simpson_kernel<float><<<(unsigned)blocks, 128, 0, st>>>(geom, N, n_intervals, (float*)flux_out);
    else
        gls::simpson_kernel<double><<<(unsigned)blocks, 128, 0, st>>>(geom, N, n_intervals, (double*)flux_out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "simpson_kernel launch");
    ++tl_launches;
    return GL_OK;
}

int gl_params_from_munu(const double* sampling, int B, double* params_out,
                        double* logprior_out_or_null, void* stream) {
    if (B < 0) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if (!sampling || !params_out) return GL_EINVAL;
    glm::params_from_munu_kernel<<<(unsigned)((B + 127) / 128), 128, 0, (cudaStream_t)stream>>>(
        sampling, B, params_out, logprior_out_or_null);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "params_from_munu_kernel launch");
    ++tl_launches;
    return GL_OK;
}

int gl_munu_from_uniform(const double* uw, int B, double* munu_out, void* stream) {
    if (B < 0) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if (!uw || !munu_out) return GL_EINVAL;
    glm::munu_from_uniform_kernel<<<(unsigned)((B + 127) / 128), 128, 0, (cudaStream_t)stream>>>(
        uw, B, munu_out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "munu_from_uniform_kernel launch");
    ++tl_launches;
    return GL_OK;
}

int gl_gp_loglike(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                  const double* obs, const double* sigma, const double* gp, double* loglike_out,
                  void* flux_work, gl_dtype dtype, void* stream) {
    if (B < 0 || T < 0 || (dtype != GL_F32 && dtype != GL_F64)) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if (!gp || !loglike_out || (T > 0 && (!obs || !sigma || !flux_work))) return GL_EINVAL;
    int rc = gl_lightcurve(params, B, times, T, t_exp, n_ss, flux_work, dtype, stream);
    if (rc != GL_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // one CTA per walker, parallel in time (gl_gp_scan.cuh)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)B, 1, 1);
    cfg.blockDim = dim3(glg::GP_NT, 1, 1);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t el = (dtype == GL_F32)
        ? cudaLaunchKernelEx(&cfg, glg::gp_scan_kernel<float>, (const float*)flux_work, B, times, T,
                             obs, sigma, gp, loglike_out)
        : cudaLaunchKernelEx(&cfg, glg::gp_scan_kernel<double>, (const double*)flux_work, B, times, T,
                             obs, sigma, gp, loglike_out);
    if (el != cudaSuccess) return cuda_fail(el, "gp_scan_kernel launch");
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "gp_scan_kernel launch");
    ++tl_launches;
    return GL_OK;
}

int gl_probe_peaks(double* out3) {
    if (!out3) return GL_EINVAL;
    void* scratch = nullptr;
    const int blocks = sm_count() * 8, thr = 256, iters = 8192;
    cudaError_t e = cudaMalloc(&scratch, (size_t)blocks * thr * sizeof(double));
    if (e != cudaSuccess) return cuda_fail(e, "gl_probe_peaks cudaMalloc");
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    for (int which = 0; which < 3; ++which) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {   // rep 0 warms up
            cudaEventRecord(a);
            if (which == 0) probe_fma<float><<<blocks, thr>>>((float*)scratch, iters, 1.0001f, 0.5f);
            if (which == 1) probe_fma<double><<<blocks, thr>>>((double*)scratch, iters / 2, 1.0001, 0.5);
            if (which == 2) probe_mufu<<<blocks, thr>>>((float*)scratch, iters / 4);
            cudaEventRecord(b);
            cudaEventSynchronize(b);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, a, b);
            if (rep > 0 && ms < best) best = ms;
        }
        const double n = (double)blocks * thr * 8.0;
        const double ops = which == 0 ? 2.0 * n * iters : which == 1 ? 2.0 * n * (iters / 2)
                                                                     : n * (iters / 4);
        out3[which] = ops / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    e = cudaGetLastError();
    cudaFree(scratch);
    if (e != cudaSuccess) return cuda_fail(e, "gl_probe_peaks");
    return GL_OK;
}

// Launch floor: an EMPTY kernel with a given grid/cluster/block shape, optionally followed by a
// second empty grid chained by programmatic dependent launch (the shape of a flux kernel + dependent kernel pair, e.g. the GP likelihood).
// bench.py times it exactly as it times a step; what it measures is what any launch of that shape
// costs on this box before a single useful instruction runs.
int gl_probe_empty_launch(int cluster, int rows, int threads, int dep_cluster, int dep_rows,
                          void* stream) {
    if (cluster < 1 || cluster > 8 || rows < 1 || threads < 32 || threads > 1024) return GL_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[2];
    cfg.gridDim = dim3((unsigned)cluster, (unsigned)rows, 1);
    cfg.blockDim = dim3((unsigned)threads, 1, 1);
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, empty_kernel, 0);
    if (e != cudaSuccess) return cuda_fail(e, "empty_kernel launch");
    if (dep_rows > 0) {
        cfg.gridDim = dim3((unsigned)dep_cluster, (unsigned)dep_rows, 1);
        cfg.blockDim = dim3(NT, 1, 1);
        attr[0].val.clusterDim.x = (unsigned)dep_cluster;
        attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.numAttrs = 2;
        e = cudaLaunchKernelEx(&cfg, empty_kernel, 1);
        if (e != cudaSuccess) return cuda_fail(e, "empty_kernel (dependent) launch");
    }
    return GL_OK;
}

// The same empty kernel replayed as a CUDA graph (captured once per shape and calling thread), the way
// gl_series_loglike_dev launches a step.
int gl_probe_empty_graph(int cluster, int rows, int threads, void* stream) {
    if (cluster < 1 || cluster > 8 || rows < 1 || threads < 32 || threads > 1024) return GL_EINVAL;
    thread_local cudaGraphExec_t exec = nullptr;
    thread_local int shape[3] = {0, 0, 0};
    if (!exec || shape[0] != cluster || shape[1] != rows || shape[2] != threads) {
        if (exec) cudaGraphExecDestroy(exec);
        exec = nullptr;
        cudaStream_t cs = nullptr;
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
        if (e == cudaSuccess) {
            const int rc = gl_probe_empty_launch(cluster, rows, threads, 1, 0, cs);
            e = cudaStreamEndCapture(cs, &graph);
            if (rc != GL_OK && e == cudaSuccess) e = cudaErrorUnknown;
        }
        if (e == cudaSuccess) e = cudaGraphInstantiate(&exec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        if (cs) cudaStreamDestroy(cs);
        if (e != cudaSuccess) {
            exec = nullptr;
            return cuda_fail(e, "gl_probe_empty_graph capture");
        }
        shape[0] = cluster;
        shape[1] = rows;
        shape[2] = threads;
    }
    const cudaError_t e = cudaGraphLaunch(exec, (cudaStream_t)stream);
    return e == cudaSuccess ? GL_OK : cuda_fail(e, "gl_probe_empty_graph launch");
}

long long gl_launch_count(void) { return tl_launches; }
const char* gl_last_cuda_error(void) { return tl_cuda_err; }
int gl_version(void) { return 100; }

}  // extern "C"

// ------------------------------------------------------------------------------------------
// gl_gp_loglike_static: the GP likelihood with its flux scratch in a file-scope device array, for
// callers that may not allocate (stream capture, serving loops).  Nothing here calls an allocator.
// ------------------------------------------------------------------------------------------
namespace {

// [B, T] fp32 model flux between the transit kernel and gp_scan_kernel.  4 MiB of every GPU that loads the
// library, until the process exits.  In host code this NAME is a host-side stand-in, not a device address:
// the address the kernels get comes from cudaGetSymbolAddress below.
static __device__ __align__(256) float g_gp_static_flux[GL_GP_STATIC_MAX_ELEMS];

// Device address of g_gp_static_flux on the CURRENT device, resolved once per device.
int gp_static_scratch(float** out) {
    static std::mutex mu;
    static float* ptrs[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && ptrs[dev]) {
        *out = ptrs[dev];
        return GL_OK;
    }
    float* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_gp_static_flux);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_gp_static_flux)");
    if (!p) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_gp_static_flux)");
    if (dev >= 0 && dev < 64) ptrs[dev] = p;
    *out = p;
    return GL_OK;
}

}  // namespace

extern "C" {

long long gl_gp_static_capacity(void) { return (long long)GL_GP_STATIC_MAX_ELEMS; }

int gl_gp_loglike_static(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                         const double* obs, const double* sigma, const double* gp, double* loglike_out,
                         void* stream) {
    if (B < 0 || T < 0) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if ((long long)B * (long long)T > (long long)GL_GP_STATIC_MAX_ELEMS) return GL_ECAPACITY;
    float* scratch = nullptr;
    const int rc = gp_static_scratch(&scratch);
    if (rc != GL_OK) return rc;
    // every one of the B*T elements is rewritten by the transit kernel before gp_scan_kernel reads it
    // (in-transit flux, 1 out of transit, NaN rows for invalid walkers): nothing has to start at zero
    return gl_gp_loglike(params, B, times, T, t_exp, n_ss, obs, sigma, gp, loglike_out, scratch, GL_F32, stream);
}

const char* gl_strerror(int code) {
    switch (code) {
        case GL_OK: return "ok";
        case GL_EINVAL: return "invalid argument";
        case GL_ECUDA: return "CUDA error (see gl_last_cuda_error)";
        case GL_EUNSUPPORTED: return "size not supported";
        case GL_ECAPACITY: return "size beyond the fixed capacity of a static-scratch entry point";
        default: return "unknown status";
    }
}

}  // extern "C"

// ------------------------------------------------------------------------------------------
// HOST-buffer wrappers: stream-ordered scratch from the device's default memory pool, copies in,
// the kernel above, copies out, one synchronise.
// ------------------------------------------------------------------------------------------
namespace {

// One non-blocking stream and one PRIVATE memory pool per calling thread and device, created on first
// use and kept for the life of the thread (include/greenlantern_b200.h says so).  The pool keeps its
// memory between calls (release threshold = max), otherwise every synchronise hands the scratch back
// to the driver and the next call pays milliseconds to get it again; the device's default pool is
// not touched.
struct HostCtx {
    cudaStream_t st = nullptr;
    cudaMemPool_t pool = nullptr;
};
HostCtx* host_ctx(cudaError_t* err) {
    thread_local HostCtx ctx[64];
    int dev = 0;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= 64) dev = 63;
    HostCtx* c = &ctx[dev];
    if (!c->st) {
        *err = cudaStreamCreateWithFlags(&c->st, cudaStreamNonBlocking);
        if (*err != cudaSuccess) return nullptr;
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        *err = cudaMemPoolCreate(&c->pool, &props);
        if (*err != cudaSuccess) {
            cudaStreamDestroy(c->st);
            c->st = nullptr;
            return nullptr;
        }
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(c->pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    return c;
}

struct HostCall {
    cudaStream_t st = nullptr;
    cudaMemPool_t pool = nullptr;
    void* bufs[8];
    int nbufs = 0;
    cudaError_t err = cudaSuccess;
    HostCall() {
        if (HostCtx* c = host_ctx(&err)) {
            st = c->st;
            pool = c->pool;
        }
    }
    void* alloc(size_t bytes) {
        void* p = nullptr;
        if (err != cudaSuccess) return nullptr;
        err = cudaMallocFromPoolAsync(&p, bytes ? bytes : 1, pool, st);
        if (err == cudaSuccess) bufs[nbufs++] = p;
        return p;
    }
    void* upload(const void* host, size_t bytes) {
        void* p = alloc(bytes);
        if (p && bytes) err = cudaMemcpyAsync(p, host, bytes, cudaMemcpyHostToDevice, st);
        return p;
    }
    void download(void* host, const void* dev, size_t bytes) {
        if (err == cudaSuccess && bytes)
            err = cudaMemcpyAsync(host, dev, bytes, cudaMemcpyDeviceToHost, st);
    }
    int finish(int rc) {
        for (int i = 0; i < nbufs; ++i) cudaFreeAsync(bufs[i], st);
        cudaError_t e2 = st ? cudaStreamSynchronize(st) : cudaSuccess;
        if (rc != GL_OK) return rc;
        if (err != cudaSuccess) return cuda_fail(err, "host wrapper");
        if (e2 != cudaSuccess) return cuda_fail(e2, "host wrapper sync");
        return GL_OK;
    }
};

size_t elem(gl_dtype d) { return d == GL_F64 ? 8 : 4; }

}  // namespace

extern "C" {

int gl_loglike_host(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                    const double* obs, const double* sigma, void* chi2_out, void* flux_out_or_null,
                    gl_dtype dtype) {
    if (B < 0 || T < 0 || (dtype != GL_F32 && dtype != GL_F64)) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if (!params || !chi2_out || (T > 0 && (!times || !obs || !sigma))) return GL_EINVAL;
    HostCall h;
    void* dp = h.upload(params, sizeof(double) * GL_NPARAMS * (size_t)B);
    void* dt = h.upload(times, sizeof(double) * (size_t)T);
    void* dob = h.upload(obs, sizeof(double) * (size_t)T);
    void* dsg = h.upload(sigma, sizeof(double) * (size_t)T);
    void* dc = h.alloc(elem(dtype) * (size_t)B);
    void* df = flux_out_or_null ? h.alloc(elem(dtype) * (size_t)B * (size_t)T) : nullptr;
    int rc = GL_OK;
    if (h.err == cudaSuccess)
        rc = gl_loglike((const double*)dp, B, (const double*)dt, T, t_exp, n_ss, (const double*)dob,
                        (const double*)dsg, dc, df, dtype, h.st);
    if (rc == GL_OK) {
        h.download(chi2_out, dc, elem(dtype) * (size_t)B);
        if (df) h.download(flux_out_or_null, df, elem(dtype) * (size_t)B * (size_t)T);
    }
    return h.finish(rc);
}

int gl_lightcurve_host(const double* params, int B, const double* times, int T, double t_exp,
                       int n_ss, void* flux_out, gl_dtype dtype) {
    if (B < 0 || T < 0 || (dtype != GL_F32 && dtype != GL_F64)) return GL_EINVAL;
    if (B == 0 || T == 0) return GL_OK;
    if (!params || !times || !flux_out) return GL_EINVAL;
    HostCall h;
    void* dp = h.upload(params, sizeof(double) * GL_NPARAMS * (size_t)B);
    void* dt = h.upload(times, sizeof(double) * (size_t)T);
    void* df = h.alloc(elem(dtype) * (size_t)B * (size_t)T);
    int rc = GL_OK;
    if (h.err == cudaSuccess)
        rc = gl_lightcurve((const double*)dp, B, (const double*)dt, T, t_exp, n_ss, df, dtype, h.st);
    if (rc == GL_OK) h.download(flux_out, df, elem(dtype) * (size_t)B * (size_t)T);
    return h.finish(rc);
}

int gl_flux_geometry_host(const double* geom, long long N, void* flux_out, gl_dtype dtype) {
    if (N < 0 || (dtype != GL_F32 && dtype != GL_F64)) return GL_EINVAL;
    if (N == 0) return GL_OK;
    if (!geom || !flux_out) return GL_EINVAL;
    HostCall h;
    void* dg = h.upload(geom, sizeof(double) * GL_NGEOM * (size_t)N);
    void* df = h.alloc(elem(dtype) * (size_t)N);
    int rc = GL_OK;
    if (h.err == cudaSuccess) rc = gl_flux_geometry((const double*)dg, N, df, dtype, h.st);
    if (rc == GL_OK) h.download(flux_out, df, elem(dtype) * (size_t)N);
    return h.finish(rc);
}

}  // extern "C"

// ------------------------------------------------------------------------------------------
// gl_series: a RESIDENT series.  An MCMC run evaluates thousands of parameter batches against one
// fixed (times, obs, sigma); everything that depends on the series alone is done
// once here: upload, order check, baseline S = sum_i ((obs_i - 1)/sigma_i)^2 in fp64, the fp32 pairs
// (obs_i - 1, 1/sigma_i) the in-window residuals use, device and pinned staging buffers.
// ------------------------------------------------------------------------------------------
namespace {

// One CTA: ow[i] = (obs_i - 1, 1/sigma_i) in fp32, S in fp64 (fixed summation order, as
// baseline_kernel), sorted = times non-decreasing.
__global__ void __launch_bounds__(1024)
series_prepare_kernel(const double* __restrict__ times, const double* __restrict__ obs,
                      const double* __restrict__ sigma, int nT, float2* __restrict__ ow,
                      double* __restrict__ S_out, int* __restrict__ sorted_out) {
    __shared__ double s_w[32];
    __shared__ int s_bad;
    if (threadIdx.x == 0) s_bad = 0;
    __syncthreads();
    double acc = 0.0;
    int bad = 0;
    for (int i = threadIdx.x; i < nT; i += 1024) {
        const double o = obs[i] - 1.0, sg = sigma[i];
        acc += residual_sq<double>(o, 0.0, sg);
        ow[i] = make_float2((float)o, (float)(1.0 / sg));
        if (i + 1 < nT) bad |= !(times[i] <= times[i + 1]);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = acc;
    if (bad) atomicOr(&s_bad, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < 32; ++k) tot += s_w[k];
        *S_out = tot;
        *sorted_out = s_bad ? 0 : 1;
    }
}

}  // namespace

struct gl_series {
    int dev = 0, T = 0, n_ss = 1, B_max = 0;
    double t_exp = 0.0, S = 0.0;
    int sorted = 0;
    cudaStream_t st = nullptr;       // host calls run here
    double *d_times = nullptr, *d_obs = nullptr, *d_sigma = nullptr;
    float2* d_ow = nullptr;
    float* d_flux = nullptr;         // [B_max, T], allocated by the first host call that asks for flux
    // pinned, device-mapped staging: the kernel reads params and writes chi^2 over PCIe
    double* h_params = nullptr;
    float* h_chi2 = nullptr;
    double* m_params = nullptr;      // device aliases
    float* m_chi2 = nullptr;
    int* h_done = nullptr;           // completion flag of the host call (pinned, mapped) ...
    int* m_done = nullptr;
    int* d_done_count = nullptr;     // ... and the device counter behind it
    // gl_series_loglike_dev: the launch captured once per (params, B, chi2, flux) and replayed as a
    // CUDA graph (callers reuse their buffers from step to step; a graph launch costs the GPU ~1 us
    // less than the stream launch it replaces)
    struct DevGraph {
        const double* params = nullptr;
        float *chi2 = nullptr, *flux = nullptr;
        int B = 0;
        bool signal = false;
        cudaGraphExec_t exec = nullptr;
        unsigned long long used = 0;
    } graphs[4];
    unsigned long long graph_clock = 0;
    std::mutex graph_mu;
};

extern "C" {

int gl_series_create(const double* times, const double* obs, const double* sigma, int T, double t_exp,
                     int n_ss, int B_max, gl_series** out) {
    if (!out) return GL_EINVAL;
    *out = nullptr;
    if (T < 1 || B_max < 1 || n_ss < 1 || !(t_exp >= 0.0) || !isfinite(t_exp) || !times || !obs || !sigma)
        return GL_EINVAL;
    {   // generic_unit (walkers off the common path) reads the constant-memory tables
        const int rc = ensure_tables();
        if (rc != GL_OK) return rc;
    }
    gl_series* s = new (std::nothrow) gl_series;
    if (!s) return GL_ECUDA;
    s->T = T;
    s->n_ss = n_ss;
    s->B_max = B_max;
    s->t_exp = t_exp;
    cudaError_t e = cudaGetDevice(&s->dev);
    const size_t tb = sizeof(double) * (size_t)T;
    double* d_S = nullptr;
    int* d_sorted = nullptr;
    auto ok = [&]() { return e == cudaSuccess; };
    if (ok()) e = cudaStreamCreateWithFlags(&s->st, cudaStreamNonBlocking);
    if (ok()) e = cudaMalloc(&s->d_times, tb);
    if (ok()) e = cudaMalloc(&s->d_obs, tb);
    if (ok()) e = cudaMalloc(&s->d_sigma, tb);
    if (ok()) e = cudaMalloc(&s->d_ow, sizeof(float2) * (size_t)T);
    if (ok()) e = cudaMalloc(&d_S, sizeof(double));
    if (ok()) e = cudaMalloc(&d_sorted, sizeof(int));
    if (ok()) e = cudaHostAlloc(&s->h_params, sizeof(double) * GL_NPARAMS * (size_t)B_max, cudaHostAllocMapped);
    if (ok()) e = cudaHostAlloc(&s->h_chi2, sizeof(float) * (size_t)B_max, cudaHostAllocMapped);
    if (ok()) e = cudaHostAlloc(&s->h_done, sizeof(int), cudaHostAllocMapped);
    if (ok()) e = cudaHostGetDevicePointer(&s->m_done, s->h_done, 0);
    if (ok()) e = cudaMalloc(&s->d_done_count, sizeof(int));
    if (ok()) e = cudaMemsetAsync(s->d_done_count, 0, sizeof(int), s->st);
    if (ok()) e = cudaHostGetDevicePointer(&s->m_params, s->h_params, 0);
    if (ok()) e = cudaHostGetDevicePointer(&s->m_chi2, s->h_chi2, 0);
    if (ok()) e = cudaMemcpyAsync(s->d_times, times, tb, cudaMemcpyHostToDevice, s->st);
    if (ok()) e = cudaMemcpyAsync(s->d_obs, obs, tb, cudaMemcpyHostToDevice, s->st);
    if (ok()) e = cudaMemcpyAsync(s->d_sigma, sigma, tb, cudaMemcpyHostToDevice, s->st);
    if (ok()) {
        series_prepare_kernel<<<1, 1024, 0, s->st>>>(s->d_times, s->d_obs, s->d_sigma, T, s->d_ow, d_S, d_sorted);
        e = cudaGetLastError();
    }
    if (ok()) e = cudaMemcpyAsync(&s->S, d_S, sizeof(double), cudaMemcpyDeviceToHost, s->st);
    if (ok()) e = cudaMemcpyAsync(&s->sorted, d_sorted, sizeof(int), cudaMemcpyDeviceToHost, s->st);
    if (ok()) e = cudaStreamSynchronize(s->st);
    cudaFree(d_S);
    cudaFree(d_sorted);
    if (!ok()) {
        const int rc = cuda_fail(e, "gl_series_create");
        gl_series_destroy(s);
        return rc;
    }
    ++tl_launches;
    *out = s;
    return GL_OK;
}

int gl_series_destroy(gl_series* s) {
    if (!s) return GL_OK;
    if (s->st) cudaStreamSynchronize(s->st);
    for (auto& g : s->graphs)
        if (g.exec) cudaGraphExecDestroy(g.exec);
    cudaFree(s->d_times);
    cudaFree(s->d_obs);
    cudaFree(s->d_sigma);
    cudaFree(s->d_ow);
    cudaFree(s->d_flux);
    if (s->h_params) cudaFreeHost(s->h_params);
    if (s->h_chi2) cudaFreeHost(s->h_chi2);
    if (s->h_done) cudaFreeHost(s->h_done);
    cudaFree(s->d_done_count);
    if (s->st) cudaStreamDestroy(s->st);
    delete s;
    return GL_OK;
}

int gl_series_info(const gl_series* s, int* T, int* n_ss, int* B_max, int* sorted, double* baseline) {
    if (!s) return GL_EINVAL;
    if (T) *T = s->T;
    if (n_ss) *n_ss = s->n_ss;
    if (B_max) *B_max = s->B_max;
    if (sorted) *sorted = s->sorted;
    if (baseline) *baseline = s->S;
    return GL_OK;
}

}  // extern "C"

// One likelihood launch against the resident series on `stream`: replay of the captured graph if this
// (params, B, chi2, flux) was seen before, else capture + launch; plain stream launch if capture fails.
static int series_launch(gl_series* s, const double* params, int B, float* chi2_out, float* flux_out_or_null,
                         void* stream, bool signal = false) {
    {
        std::lock_guard<std::mutex> lock(s->graph_mu);
        gl_series::DevGraph* slot = &s->graphs[0];
        for (auto& g : s->graphs) {
            if (g.exec && g.params == params && g.B == B && g.chi2 == chi2_out && g.flux == flux_out_or_null &&
                g.signal == signal) {
                g.used = ++s->graph_clock;
                const cudaError_t e = cudaGraphLaunch(g.exec, (cudaStream_t)stream);
                if (e != cudaSuccess) return cuda_fail(e, "gl_series_loglike_dev graph launch");
                tl_launches += 1;
                return GL_OK;
            }
            if (g.used < slot->used) slot = &g;   // least recently used (empty slots have used = 0)
        }
        // not seen before: capture the launch on the handle's own stream, keep it, launch it
        SeriesView svc;
        svc.ow = s->d_ow;
        svc.S = s->S;
        svc.sorted_known = s->sorted;
        if (signal) {
            svc.done_count = s->d_done_count;
            svc.done_flag = s->m_done;
        }
        cudaGraph_t graph = nullptr;
        cudaGraphExec_t exec = nullptr;
        const long long before = tl_launches;
        cudaError_t e = cudaStreamBeginCapture(s->st, cudaStreamCaptureModeThreadLocal);
        if (e == cudaSuccess) {
            const int rc = launch_hot(params, B, s->d_times, s->T, s->t_exp, s->n_ss, s->d_obs, s->d_sigma,
                                      flux_out_or_null, chi2_out, svc, s->st);
            e = cudaStreamEndCapture(s->st, &graph);
            if (rc != GL_OK && e == cudaSuccess) e = cudaErrorUnknown;
        }
        tl_launches = before;
        if (e == cudaSuccess) e = cudaGraphInstantiate(&exec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        if (e == cudaSuccess) {
            if (slot->exec) cudaGraphExecDestroy(slot->exec);
            slot->params = params;
            slot->B = B;
            slot->chi2 = chi2_out;
            slot->flux = flux_out_or_null;
            slot->signal = signal;
            slot->exec = exec;
            slot->used = ++s->graph_clock;
            e = cudaGraphLaunch(exec, (cudaStream_t)stream);
            if (e != cudaSuccess) return cuda_fail(e, "gl_series_loglike_dev graph launch");
            tl_launches += 1;
            return GL_OK;
        }
        (void)cudaGetLastError();   // no graph then: plain stream launches below
    }
    SeriesView sv;
    sv.ow = s->d_ow;
    sv.S = s->S;
    sv.sorted_known = s->sorted;
    if (signal) {
        sv.done_count = s->d_done_count;
        sv.done_flag = s->m_done;
    }
    return launch_hot(params, B, s->d_times, s->T, s->t_exp, s->n_ss, s->d_obs, s->d_sigma,
                      flux_out_or_null, chi2_out, sv, (cudaStream_t)stream);
}

extern "C" {

int gl_series_loglike_dev(gl_series* s, const double* params, int B, float* chi2_out,
                          float* flux_out_or_null, void* stream) {
    if (!s || B < 0) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if (!params || !chi2_out) return GL_EINVAL;
    return series_launch(s, params, B, chi2_out, flux_out_or_null, stream);
}

int gl_series_loglike(gl_series* s, const double* params, int B, float* chi2_out, float* flux_out_or_null) {
    if (!s || B < 0 || B > s->B_max) return GL_EINVAL;
    if (B == 0) return GL_OK;
    if (!params || !chi2_out) return GL_EINVAL;
    cudaError_t e = cudaSuccess;
    if (flux_out_or_null && !s->d_flux) {
        e = cudaMalloc(&s->d_flux, sizeof(float) * (size_t)s->B_max * (size_t)s->T);
        if (e != cudaSuccess) return cuda_fail(e, "gl_series_loglike flux buffer");
    }
    memcpy(s->h_params, params, sizeof(double) * GL_NPARAMS * (size_t)B);
    float* flux = flux_out_or_null ? s->d_flux : nullptr;
    *(volatile int*)s->h_done = 0;
    const int rc = series_launch(s, s->m_params, B, s->m_chi2, flux, s->st, /*signal=*/!flux);   // (graph replay)
    if (rc != GL_OK) return rc;
    if (flux) {
        e = cudaMemcpyAsync(flux_out_or_null, flux, sizeof(float) * (size_t)B * (size_t)s->T,
                            cudaMemcpyDeviceToHost, s->st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->st);
    } else {
        // chi^2 only: the kernel's last CTA raises a flag in pinned host memory once every chi^2 is written;
        // spinning on it returns sooner than a stream synchronise.  No flag within 2 s: let the stream say why.
        const auto t_start = std::chrono::steady_clock::now();
        unsigned spins = 0;
        while (*(volatile int*)s->h_done == 0) {
            if ((++spins & 0x3ffu) == 0 &&
                std::chrono::steady_clock::now() - t_start > std::chrono::seconds(2)) {
                e = cudaStreamSynchronize(s->st);
                if (e == cudaSuccess && *(volatile int*)s->h_done == 0) {
                    cudaMemsetAsync(s->d_done_count, 0, sizeof(int), s->st);   // re-arm for the next call
                    e = cudaErrorUnknown;
                }
                break;
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
    }
    if (e != cudaSuccess) return cuda_fail(e, "gl_series_loglike");
    memcpy(chi2_out, s->h_chi2, sizeof(float) * (size_t)B);
    return GL_OK;
}

}  // extern "C"
