// gl_core.cuh -- device arithmetic of the oblate-transit hot path (steps a3 + a4 of DESIGN.md):
// outline/limb crossings and the Green's-theorem boundary integrals, templated on the arithmetic
// type (float = production, double = validation).  Shares nothing with oracle/.
//
// Frame used here: origin at the star centre, axes along the principal
// axes of the projected outline, so the outline of PAPER.md:79-82 (eqs. 7-8) reads
//     x(t) = xc + a cos t,   y(t) = yc + b sin t,   a >= b > 0
// (eqs. 7-8 with dy1 = 0; the Cholesky parameter theta of eqs. 11-13 differs from t by a constant
// shift).  A, the three area integrals, are invariant under the rotation and under the mirror
// images x -> -x, y -> -y, so the caller's centre is first folded into xc >= 0, yc >= 0.
#pragma once
#include <math.h>

#ifdef __CUDACC__
#define GL_DEV __device__ __forceinline__
#else
#define GL_DEV inline
#endif

namespace glc {

template <typename T> struct num;
template <> struct num<float> {
    static constexpr float pi = 3.14159265358979323846f;
    // angle tolerance of the bracketed solves: an angle error eps moves the areas by O(eps^2) only
    // (gl_fast32.cuh header), so fp32 does not chase the last ulp
    static constexpr float tol = 2e-5f;
    // ... and the CRITICAL POINTS of g need far less: they serve as brackets for the crossings, as places to
    // open or split a contour (any point will do) and as the arguments of g(t_far), g(t_a), g(t_b), g(t_near),
    // which are stationary there (an angle error eps moves them by O(eps^2) = 1e-6 of an O(a) quantity).
    // Measured on config 5 (host build, 4e5 rows): iterations of a critical-point search 3.9 -> 2.4 on average,
    // 95th percentile 12 -> 4 (the tail was bisection inside the tiny brackets of nearly symmetric outlines),
    // max |flux error| per class unchanged (1.3e-7).
    static constexpr float tol_h = 1e-3f;
    static constexpr float nudge = 2.5e-7f; // quadrant brackets are pulled strictly inside by this
    static constexpr int maxit = 40;
};
template <> struct num<double> {
    static constexpr double pi = 3.14159265358979323846;
    static constexpr double tol = 4e-16;
    static constexpr double tol_h = 4e-16;
    static constexpr double nudge = 5e-16;
    static constexpr int maxit = 80;
};

GL_DEV float gsqrt(float x) { return sqrtf(x); }
GL_DEV double gsqrt(double x) { return sqrt(x); }
GL_DEV float gabs(float x) { return fabsf(x); }
GL_DEV double gabs(double x) { return fabs(x); }
GL_DEV float gatan2(float y, float x) { return atan2f(y, x); }
GL_DEV double gatan2(double y, double x) { return atan2(y, x); }
GL_DEV float gasin(float x) { return asinf(x); }
GL_DEV double gasin(double x) { return asin(x); }
GL_DEV float gacos(float x) { return acosf(x); }
GL_DEV double gacos(double x) { return acos(x); }
GL_DEV float gcbrt(float x) { return cbrtf(x); }
GL_DEV double gcbrt(double x) { return cbrt(x); }
GL_DEV float gmax(float a, float b) { return fmaxf(a, b); }
GL_DEV double gmax(double a, double b) { return fmax(a, b); }
GL_DEV float gmin(float a, float b) { return fminf(a, b); }
GL_DEV double gmin(double a, double b) { return fmin(a, b); }
GL_DEV void gsincos(float t, float* s, float* c) { sincosf(t, s, c); }
// Sine and cosine of an OUTLINE angle in [0, 3 pi] (the geometry routines below; never the orbital
// phase, whose sine is multiplied by a/R*).  FT = false: libm.  FT = true (fp32 on the device only):
// MUFU, angle folded into [-pi, pi] -- absolute error 2^-21, inside the fp32 budget (gl_fast32.cuh
// header).  A template flag and not a global choice because MUFU sine/cosine in this code, which is
// inlined into the fused transit kernel but rarely executed there, made that kernel's register
// allocation spill three times as much (cfg3 +2 us, cfg4 +6 us); the bare-geometry kernel, where the
// evolute regime is common (config 5), instantiates FT = true.
template <bool FT> GL_DEV void gtrig(float t, float* s, float* c) {
#ifdef __CUDACC__
    if (FT) {
        const float tr = t > 3.14159265358979323846f ? t - 6.28318530717958647692f : t;
        *s = __sinf(tr);
        *c = __cosf(tr);
        return;
    }
#endif
    sincosf(t, s, c);
}
template <bool FT> GL_DEV void gtrig(double t, double* s, double* c) { sincos(t, s, c); }
GL_DEV void gsincos(double t, double* s, double* c) { sincos(t, s, c); }

// The outline in the kernel frame and everything derived from it once per sub-sample.
template <typename T> struct Outline {
    T xc, yc, a, b, e2;   // e2 = a^2 - b^2 >= 0
};

// g(t) = x^2 + y^2 - 1 and h(t) = g'(t)/2 = x x' + y y'  (x' = -a sin t, y' = b cos t;
// PAPER.md:102-104 eqs. 14-15 in the kernel frame).
template <typename T, bool FT = false> GL_DEV void eval_g(const Outline<T>& o, T t, T* g, T* h) {
    T s, c;
    gtrig<FT>(t, &s, &c);
    const T x = o.xc + o.a * c, y = o.yc + o.b * s;
    *g = x * x + (y * y - T(1));
    *h = o.b * c * y - o.a * s * x;
}
// h(t) and h'(t) for the critical points of g.
template <typename T, bool FT = false> GL_DEV void eval_h(const Outline<T>& o, T t, T* h, T* hp) {
    T s, c;
    gtrig<FT>(t, &s, &c);
    const T x = o.xc + o.a * c, y = o.yc + o.b * s;
    *h = o.b * c * y - o.a * s * x;
    const T bc = o.b * c, as = o.a * s;
    *hp = bc * bc + as * as - o.b * s * y - o.a * c * x;
}

// Root of a function that changes sign exactly once on [lo, hi]: Newton, with bisection whenever
// the Newton step leaves the bracket.  rising = the function is <= 0 at lo and >= 0 at hi.
// WHICH = 0: root of g, WHICH = 1: root of h.
template <typename T, int WHICH, bool FT = false>
GL_DEV T solve_in(const Outline<T>& o, T lo, T hi, T t, bool rising) {
    t = gmin(gmax(t, lo), hi);
    for (int it = 0; it < num<T>::maxit; ++it) {
        T f, df;
        if (WHICH == 0) {
            eval_g<T, FT>(o, t, &f, &df);
            df = df + df;
        } else {
            eval_h<T, FT>(o, t, &f, &df);
        }
        if ((f > T(0)) == rising) hi = t; else lo = t;
        T tn = t - f / df;
        if (!(tn > lo && tn < hi)) tn = T(0.5) * (lo + hi);
        const T d = tn - t;
        t = tn;
        if (gabs(d) <= (WHICH == 1 ? num<T>::tol_h : num<T>::tol) * gmax(T(1), gabs(t))) break;
    }
    return t;
}

// First guess for the root of g on a monotone arc [ta, tb] with end values ga, gb of opposite
// sign: between two consecutive critical points g looks like half a cosine period.
template <typename T> GL_DEV T cosine_guess(T ta, T tb, T ga, T gb) {
    const T mid = T(0.5) * (ga + gb), amp = T(0.5) * (ga - gb);   // g ~ mid + amp cos(pi u)
    T r = -mid / amp;
    r = gmin(gmax(r, T(-1)), T(1));
    return ta + (tb - ta) * gacos(r) * (T(1) / num<T>::pi);
}

// ---------------------------------------------------------------------------------------------
// Boundary integrals (step a4).  All three 1-forms are weights of f_flat (eq. 21):
//   f_flat = (x y' - y x')/2,  f_lin = (2/3) W(r^2) f_flat (eq. 22),
//   f_quad = (r^2/2) f_flat  -- a 1-form with the same curl r^2 as PAPER.md:135 eq. 23 (they
//   differ by an exact differential, so every closed-contour integral agrees; D3).
//   W(s) = [1 - (1-s)^{3/2}]/s = 1 + m^2/(1+m), m = sqrt(1-s): no cancellation at s -> 0 (R9),
//   1-s clamped at 0 (R11).
// On the outline 2 f_flat = ab + u cos t + v sin t with u = b xc, v = a yc, so the flat and quad
// integrals over an arc are elementary; only f_lin is summed numerically (NQ-point Gauss-Legendre
// in z after t = tm + hw (3z - z^3)/2, which removes the (1-r^2)^{3/2} end-point singularity).
// ---------------------------------------------------------------------------------------------
template <typename T> struct ArcCoef {
    T ab, u, v;                       // 2 f_flat = ab + u c + v s
    T k0, kc, ks, kc2, ks2, kc3, ks3; // r^2 * 2 f_flat as a trigonometric polynomial
};

template <typename T> GL_DEV ArcCoef<T> arc_coefficients(const Outline<T>& o) {
    ArcCoef<T> k;
    k.ab = o.a * o.b;
    k.u = o.b * o.xc;
    k.v = o.a * o.yc;
    const T R1 = o.xc * o.xc + o.yc * o.yc + T(0.5) * (o.a * o.a + o.b * o.b);
    const T p = T(2) * o.a * o.xc, q = T(2) * o.b * o.yc, w = T(0.5) * o.e2;
    k.k0 = R1 * k.ab + T(0.5) * (p * k.u + q * k.v);
    k.kc = R1 * k.u + p * k.ab + T(0.5) * w * k.u;
    k.ks = R1 * k.v + q * k.ab - T(0.5) * w * k.v;
    k.kc2 = T(0.5) * (p * k.u - q * k.v) + w * k.ab;
    k.ks2 = T(0.5) * (p * k.v + q * k.u);
    k.kc3 = T(0.5) * w * k.u;
    k.ks3 = T(0.5) * w * k.v;
    return k;
}

// Antiderivative pieces at one end point (sine/cosine given): returns the non-secular parts.
template <typename T> GL_DEV void arc_primitive(const ArcCoef<T>& k, T s, T c, T* pflat, T* pquad) {
    *pflat = k.u * s - k.v * c;
    const T s2 = T(2) * s * c, c2 = (c - s) * (c + s);
    const T s3 = s * (T(3) - T(4) * s * s), c3 = c * (T(4) * c * c - T(3));
    *pquad = k.kc * s - k.ks * c + T(0.5) * (k.kc2 * s2 - k.ks2 * c2) +
             (T(1) / T(3)) * (k.kc3 * s3 - k.ks3 * c3);
}

// Adds the integrals of f_flat, f_lin, f_quad along the outline from t1 to t2 (t2 >= t1) to A[0..2].
// qphi[k] = (3 z_k - z_k^3)/2 and qom[k] = w_k * 1.5 (1 - z_k^2) for the NQ/2 positive nodes z_k.
template <typename T, int NQ, bool FT = false>
GL_DEV void add_outline_arc(const Outline<T>& o, const ArcCoef<T>& k, T t1, T s1, T c1, T t2, T s2,
                            T c2, const T* qphi, const T* qom, T* A) {
    const T dt = t2 - t1;
    T f1, q1, f2, q2;
    arc_primitive(k, s1, c1, &f1, &q1);
    arc_primitive(k, s2, c2, &f2, &q2);
    A[0] += T(0.5) * (k.ab * dt + (f2 - f1));
    A[2] += T(0.25) * (k.k0 * dt + (q2 - q1));
    const T hw = T(0.5) * dt, tm = t1 + hw;
    T sm, cm;
    gtrig<FT>(tm, &sm, &cm);
    T acc = T(0);
#pragma unroll
    for (int i = 0; i < NQ / 2; ++i) {
        T sd, cd;
        gtrig<FT>(hw * qphi[i], &sd, &cd);
        const T cp = cm * cd - sm * sd, sp = sm * cd + cm * sd;   // t = tm + delta
        const T cq = cm * cd + sm * sd, sq = sm * cd - cm * sd;   // t = tm - delta
        const T xp = o.xc + o.a * cp, yp = o.yc + o.b * sp;
        const T xq = o.xc + o.a * cq, yq = o.yc + o.b * sq;
        const T mp2 = gmax(T(1) - (xp * xp + yp * yp), T(0));
        const T mq2 = gmax(T(1) - (xq * xq + yq * yq), T(0));
        const T mp = gsqrt(mp2), mq = gsqrt(mq2);
        const T Wp = T(1) + mp2 / (T(1) + mp), Wq = T(1) + mq2 / (T(1) + mq);
        const T fp = k.ab + k.u * cp + k.v * sp, fq = k.ab + k.u * cq + k.v * sq;
        acc += qom[i] * (Wp * fp + Wq * fq);
    }
    A[1] += (T(1) / T(3)) * hw * acc;
}

// Limb arc from outline point (xa, ya) counter-clockwise to (xb, yb): on r = 1 the three forms are
// lambda'/2, lambda'/3 (W(1) = 1) and lambda'/4; the arc is shorter than pi because a < 1/2 (R13).
template <typename T> GL_DEV void add_limb_arc(T xa, T ya, T xb, T yb, T* A) {
    const T dl = gatan2(xa * yb - ya * xb, xa * xb + ya * yb);
    A[0] += T(0.5) * dl;
    A[1] += (T(1) / T(3)) * dl;
    A[2] += T(0.25) * dl;
}

// ---------------------------------------------------------------------------------------------
// Step a3 + a4 together: A = {A_flat, A_lin, A_quad} of (outline) n (unit disc).  Returns false
// (A untouched) when the overlap is empty.
//
// Crossing search (R3).  With xc, yc >= 0, A = a xc, B = b yc:
//   h = g'/2 has exactly one zero in [0, pi/2] (the outline point farthest from the star centre,
//   t_far), exactly one in [pi, 3pi/2] (the nearest, t_near), none in (3pi/2, 2pi), and either
//   none or two in (pi/2, pi): two exactly when the star centre lies inside the outline's evolute,
//   A^{2/3} + B^{2/3} < (a^2-b^2)^{2/3}; they straddle t* = pi - atan((B/A)^{1/3}) (a local minimum
//   t_a < t* and a local maximum t_b > t* of g).  Between consecutive critical points g is
//   monotone, so each crossing is the single root of g in a known bracket: no quartic algebra.
// ---------------------------------------------------------------------------------------------
// The search is written in three stages so that a kernel can run each stage over a list of its own (the
// bare-geometry kernel sorts its rows between them); overlap_areas() below runs them back to back.
template <typename T> struct CritPoints {   // stage 1: the critical points of g and g there
    T tfar, gfar, ta, tb, ga, gb;
    bool evol;                              // the pair (ta, tb) exists
};
template <typename T> struct ArcPlan {      // stage 2: the arcs of the outline that lie inside the disc
    T as[2], ae[2];
    int narc;                               // 0: no overlap
    bool limb;                              // the contour is closed along the limb
};
template <typename T> GL_DEV Outline<T> make_outline(T xc_in, T yc_in, T a, T b) {
    Outline<T> o;
    o.xc = gabs(xc_in);
    o.yc = gabs(yc_in);
    o.a = a;
    o.b = b;
    o.e2 = (a - b) * (a + b);
    return o;
}
// Stage 1.  false: the outline cannot reach the disc.
template <typename T, bool FT>
GL_DEV bool critical_points(const Outline<T>& o, CritPoints<T>* cp) {
    const T pi = num<T>::pi, half = T(0.5) * pi;
    // quadrant boundaries pulled strictly inside their quadrant, so that a rounded boundary can
    // never sit on the far side of a neighbouring critical point
    const T q1hi = half * (T(1) - num<T>::nudge), q2lo = half * (T(1) + num<T>::nudge);
    const T q2hi = pi * (T(1) - num<T>::nudge);
    const T r0sq = o.xc * o.xc + o.yc * o.yc;
    if (r0sq >= (T(1) + o.a) * (T(1) + o.a)) return false;
    const T Aa = o.a * o.xc, Bb = o.b * o.yc;
    T hd;
    cp->tfar = T(0);
    if (Aa > T(0) || Bb > T(0)) cp->tfar = solve_in<T, 1, FT>(o, T(0), q1hi, gatan2(Bb, Aa), false);
    eval_g<T, FT>(o, cp->tfar, &cp->gfar, &hd);
    cp->evol = false;
    cp->ta = cp->tb = cp->ga = cp->gb = T(0);
    if (Aa < o.e2 && Bb < o.e2) {
        const T cA = gcbrt(Aa), cB = gcbrt(Bb), cE = gcbrt(o.e2);
        if (cA * cA + cB * cB < cE * cE) {
            cp->evol = true;
            const T tstar = gmin(gmax(pi - gatan2(cB, cA), q2lo), q2hi);
            cp->ta = solve_in<T, 1, FT>(o, q2lo, tstar, T(0.5) * (q2lo + tstar), true);
            cp->tb = solve_in<T, 1, FT>(o, tstar, q2hi, T(0.5) * (tstar + q2hi), false);
            eval_g<T, FT>(o, cp->ta, &cp->ga, &hd);
            eval_g<T, FT>(o, cp->tb, &cp->gb, &hd);
        }
    }
    return true;
}
// Stage 2a: the whole outline is inside the disc (gfar <= 0): open the contour at the point nearest the limb.
template <typename T> GL_DEV void plan_inside(const CritPoints<T>& cp, ArcPlan<T>* pl) {
    const T pi = num<T>::pi;
    pl->limb = false;
    pl->narc = 1;
    pl->as[0] = cp.tfar;
    pl->ae[0] = cp.tfar + T(2) * pi;
    if (cp.evol) {
        pl->narc = 2;
        pl->ae[0] = cp.tb;
        pl->as[1] = cp.tb;
        pl->ae[1] = cp.tfar + T(2) * pi;
    }
}
// Stage 2b: gfar > 0: the nearest point and the crossings.  narc = 0: the outline misses the disc.
template <typename T, bool FT>
GL_DEV void plan_crossing(const Outline<T>& o, const CritPoints<T>& cp, ArcPlan<T>* pl) {
    const T pi = num<T>::pi, half = T(0.5) * pi;
    const T q3lo = pi * (T(1) + num<T>::nudge), q3hi = T(3) * half * (T(1) - num<T>::nudge);
    const T Aa = o.a * o.xc, Bb = o.b * o.yc;
    const T tfar = cp.tfar, gfar = cp.gfar, ta = cp.ta, tb = cp.tb, ga = cp.ga, gb = cp.gb;
    T* as = pl->as;
    T* ae = pl->ae;
    pl->limb = true;
    pl->narc = 0;
    const T tnear = solve_in<T, 1, FT>(o, q3lo, q3hi, pi + gatan2(Bb, Aa), true);
    T gnear, hd;
    eval_g<T, FT>(o, tnear, &gnear, &hd);
    if (gnear >= T(0)) return;
    pl->narc = 1;
    const T tend = tfar + T(2) * pi;
    const T rexit = solve_in<T, 0, FT>(o, tnear, tend, cosine_guess(tnear, tend, gnear, gfar), true);
    if (!cp.evol) {
        as[0] = solve_in<T, 0, FT>(o, tfar, tnear, cosine_guess(tfar, tnear, gfar, gnear), false);
        ae[0] = rexit;
    } else if (ga < T(0) && gb > T(0)) {
        pl->narc = 2;
        as[0] = solve_in<T, 0, FT>(o, tfar, ta, cosine_guess(tfar, ta, gfar, ga), false);
        ae[0] = solve_in<T, 0, FT>(o, ta, tb, cosine_guess(ta, tb, ga, gb), true);
        as[1] = solve_in<T, 0, FT>(o, tb, tnear, cosine_guess(tb, tnear, gb, gnear), false);
        ae[1] = rexit;
    } else if (ga >= T(0)) {
        as[0] = solve_in<T, 0, FT>(o, tb, tnear, cosine_guess(tb, tnear, gb, gnear), false);
        ae[0] = rexit;
    } else {
        // local maximum at t_b stays inside the disc: split there (near-singular integrand)
        pl->narc = 2;
        as[0] = solve_in<T, 0, FT>(o, tfar, ta, cosine_guess(tfar, ta, gfar, ga), false);
        ae[0] = tb;
        as[1] = tb;
        ae[1] = rexit;
    }
}
// Stage 3: the boundary integrals along the planned arcs (and the limb arcs that close the contour).
template <typename T, int NQ, bool FT>
GL_DEV void integrate_plan(const Outline<T>& o, const ArcPlan<T>& pl, const T* qphi, const T* qom, T* A) {
    const ArcCoef<T> k = arc_coefficients(o);
    A[0] = A[1] = A[2] = T(0);
    T ss[2], cs[2], se[2], ce[2];
    for (int i = 0; i < pl.narc; ++i) {
        gtrig<FT>(pl.as[i], &ss[i], &cs[i]);
        gtrig<FT>(pl.ae[i], &se[i], &ce[i]);
        add_outline_arc<T, NQ, FT>(o, k, pl.as[i], ss[i], cs[i], pl.ae[i], se[i], ce[i], qphi, qom, A);
    }
    if (pl.limb) {
        for (int i = 0; i < pl.narc; ++i) {
            const int j = (i + 1 == pl.narc) ? 0 : i + 1;
            add_limb_arc(o.xc + o.a * ce[i], o.yc + o.b * se[i], o.xc + o.a * cs[j], o.yc + o.b * ss[j], A);
        }
    }
}

template <typename T, int NQ, bool FT = false>
GL_DEV bool overlap_areas(T xc_in, T yc_in, T a, T b, const T* qphi, const T* qom, T* A) {
    const Outline<T> o = make_outline(xc_in, yc_in, a, b);
    CritPoints<T> cp;
    if (!critical_points<T, FT>(o, &cp)) return false;
    ArcPlan<T> pl;
    if (cp.gfar <= T(0)) {
        plan_inside(cp, &pl);
    } else {
        plan_crossing<T, FT>(o, cp, &pl);
        if (pl.narc == 0) return false;
    }
    integrate_plan<T, NQ, FT>(o, pl, qphi, qom, A);
    return true;
}

}  // namespace glc
