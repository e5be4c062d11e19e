// gl_fast32.cuh -- fp32 PRODUCTION arithmetic of steps a3 + a4: the same three area
// integrals as gl_core.cuh, arranged for throughput on the sm_100a FP32 and MUFU pipes.
//
// What is different from the generic (validation) code in gl_core.cuh, and why it is allowed:
//  * The result wanted is the BLOCKED FRACTION delta = 1 - F <= ~0.06, to 5e-7 absolute, i.e. to
//    1e-5 relative at best: MUFU approximations (sin/cos/rcp/sqrt .approx, ~2^-21 absolute) are far
//    inside the budget as long as no step cancels (every term below is O(a) or smaller).
//  * A crossing angle that is wrong by eps moves the three areas by O(eps^2): all three 1-forms
//    (eqs. 21-23, D3) are multiples of x dy - y dx, which vanishes on the radial
//    segment that joins a slightly-off crossing point to the limb, so only the sliver between the
//    two curves (width ~ |g'| eps, length eps) is mis-counted (R12).  Crossings are therefore
//    solved to 5e-5 rad, not to an ulp.
//  * An outline that lies wholly inside the disc is a closed, periodic contour: the N-point
//    trapezoid rule at FIXED angles 2 pi k/N converges geometrically and needs no trigonometry at
//    run time (cos/sin of the nodes are constants).  Measured on 4e5 config-5 geometries in fp64
//    (DESIGN.md 5.6): N = 16 is good to 2e-8 in flux once the gap to the limb is >= 0.01, N = 32 to
//    1.7e-8 for every gap down to tangency.
//  * Only the rare geometries whose star centre may lie inside the outline's evolute (a second
//    pair of critical points, up to four crossings) go through gl_core.cuh's bracketed search.
#pragma once
#include "gl_core.cuh"

namespace glf {

#ifdef __CUDACC__
#define GLF_DEV __device__ __forceinline__
#define GLF_CONST __constant__
#else   // host build: only for checking the arithmetic on a CPU (exact math in place of MUFU)
#define GLF_DEV inline
#define GLF_CONST static
#endif

// cos, sin of 2 pi k / 32, k = 0..15 (the other half is the mirror image); filled at library load.
GLF_CONST float c_trap_cos[16], c_trap_sin[16];
// smoothed Gauss-Legendre table of the generic path (gl_tables.h), fp32 copy: 8 positive nodes.
GLF_CONST float c_gl_phi[8], c_gl_om[8];

constexpr float kPiF = 3.14159265358979323846f;
constexpr float kTwoPiF = 6.28318530717958647692f;

#ifdef __CUDACC__
GLF_DEV float mufu_rcp(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
GLF_DEV float mufu_sqrt(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
GLF_DEV float mufu_rsqrt(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
GLF_DEV float mufu_sin(float x) {
    float r;
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
GLF_DEV float mufu_cos(float x) {
    float r;
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
GLF_DEV float fast_div(float x, float y) { return __fdividef(x, y); }
#else
GLF_DEV float mufu_rcp(float x) { return 1.f / x; }
GLF_DEV float mufu_sqrt(float x) { return sqrtf(x); }
GLF_DEV float mufu_rsqrt(float x) { return 1.f / sqrtf(x); }
#ifdef GLF_HOST_NOISE   // the harness models the 2^-21 absolute error of MUFU.SIN/COS
GLF_DEV float mufu_sin(float x) { return sinf(x) + nz(); }
GLF_DEV float mufu_cos(float x) { return cosf(x) + nz(); }
#else
GLF_DEV float mufu_sin(float x) { return sinf(x); }
GLF_DEV float mufu_cos(float x) { return cosf(x); }
#endif
GLF_DEV float fast_div(float x, float y) { return x / y; }
#endif
// pi / nh for nh = 4, 8 or 16 half-nodes of a fixed-angle rule.  A division by a power of two is exact, so
// the selected constants ARE what the IEEE division gives -- without its slow-path call in the inner code.
GLF_DEV float pi_over_nodes(int nh) {
    return nh == 4 ? 0.25f * kPiF : (nh == 8 ? 0.125f * kPiF : (nh == 16 ? 0.0625f * kPiF : kPiF * 0.5f));
}
// sin, cos of an angle in [-pi, 3 pi]: folded into [-pi, pi], where the MUFU error is 2^-21.
GLF_DEV void mufu_sincos(float t, float* s, float* c) {
    const float tr = (t > kPiF) ? t - kTwoPiF : t;
    *s = mufu_sin(tr);
    *c = mufu_cos(tr);
}

// W(s) f for the two mirror nodes of a pair, sharing ONE reciprocal:
//   W = 1 + m^2/(1+m), m = sqrt(max(1 - r^2, 0))   (eq. 22 in the form of R9, R11)
// CLAMP = false where every node is known to lie strictly inside the disc.
template <bool CLAMP> GLF_DEV float pair_term(float m2p, float fp, float m2q, float fq) {
    if (CLAMP) {
        m2p = fmaxf(m2p, 0.f);
        m2q = fmaxf(m2q, 0.f);
    }
    const float dp = 1.f + mufu_sqrt(m2p), dq = 1.f + mufu_sqrt(m2q);
    const float r = mufu_rcp(dp * dq);             // 1/dp = dq r, 1/dq = dp r
    const float Wp = fmaf(m2p, dq * r, 1.f), Wq = fmaf(m2q, dp * r, 1.f);
    return fmaf(Wp, fp, Wq * fq);
}

// Integral over the WHOLE outline of W(r^2) (2 f_flat) dt by the N-point trapezoid rule, N = 2 nh,
// nh = 4, 8 or 16 chosen PER LANE: one loop serves every tier, so a warp whose lanes need
// different orders runs the longest one once instead of one code copy per tier.
// 2 f_flat = ab + u cos t + v sin t with u = b xc, v = a yc (gl_core.cuh).  Nodes k and k + N/2 are
// mirror images, so each table entry serves two nodes.  trap[k] = (cos, sin)(2 pi k / 32), k < 16:
// a copy of c_trap_cos/sin that the caller keeps in SHARED memory (per-lane strides would
// serialise in the constant cache).
struct TrapNode {
    float c, s;
};
GLF_DEV float whole_outline_lin(const TrapNode* trap, int nh, float xc, float yc, float a, float b,
                                float ab, float u, float v) {
    const int stride = 16 / nh;
    float acc = 0.f;
    for (int k0 = 0; k0 < nh; k0 += 4) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            const TrapNode nd = trap[(k0 + kk) * stride];
            const float p = a * nd.c, q = b * nd.s;
            const float xp = xc + p, yp = yc + q, xq = xc - p, yq = yc - q;
            const float m2p = fmaf(-xp, xp, fmaf(-yp, yp, 1.f));
            const float m2q = fmaf(-xq, xq, fmaf(-yq, yq, 1.f));
            const float w = fmaf(u, nd.c, v * nd.s);
            acc += pair_term<true>(m2p, ab + w, m2q, ab - w);
        }
    }
    return acc * pi_over_nodes(nh);
}

// The same integral with SIX nodes (0, 60, ..., 300 degrees), for outlines deep inside the disc: the
// node cosines and sines are immediates, and the pair on the major axis needs no y offset.  fp64
// experiment (as above, 5e5 geometries): flux error <= 6.2e-9 once gap >= 3 a, <= 1.4e-8 for gap >= 0.5.
GLF_DEV float whole_outline_lin6(float xc, float yc, float a, float b, float ab, float u, float v) {
    constexpr float S60 = 0.86602540378443864676f;
    const float yy = fmaf(-yc, yc, 1.f);
    const float x0p = xc + a, x0q = xc - a;
    float acc = pair_term<false>(fmaf(-x0p, x0p, yy), ab + u, fmaf(-x0q, x0q, yy), ab - u);
    const float p = 0.5f * a, q = S60 * b, hu = 0.5f * u, sv = S60 * v;
    {
        const float xp = xc + p, yp = yc + q, xq = xc - p, yq = yc - q;
        const float w = hu + sv;
        acc += pair_term<false>(fmaf(-xp, xp, fmaf(-yp, yp, 1.f)), ab + w,
                                fmaf(-xq, xq, fmaf(-yq, yq, 1.f)), ab - w);
    }
    {
        const float xp = xc - p, yp = yc + q, xq = xc + p, yq = yc - q;
        const float w = sv - hu;
        acc += pair_term<false>(fmaf(-xp, xp, fmaf(-yp, yp, 1.f)), ab + w,
                                fmaf(-xq, xq, fmaf(-yq, yq, 1.f)), ab - w);
    }
    return acc * (kPiF / 3.f);
}

// The outline in the kernel frame, re-parametrised by tau = t - t_far (t_far = the outline point
// farthest from the star centre, given by its cosine/sine cf, sf).
struct Arc {
    float xc, yc, a, b, cf, sf;
};
GLF_DEV void abs_trig(const Arc& o, float tau, float* s, float* c) {
    float st, ct;
    mufu_sincos(tau, &st, &ct);
    *c = o.cf * ct - o.sf * st;
    *s = o.sf * ct + o.cf * st;
}
// g = x^2 + y^2 - 1 and g'/2 at tau; also returns the absolute sine/cosine.
GLF_DEV void eval_g(const Arc& o, float tau, float* g, float* h, float* s,
                                       float* c) {
    abs_trig(o, tau, s, c);
    const float x = fmaf(o.a, *c, o.xc), y = fmaf(o.b, *s, o.yc);
    *g = fmaf(x, x, fmaf(y, y, -1.f));
    *h = o.b * *c * y - o.a * *s * x;
}

// Crossing of g on [lo, hi] (one sign change): Newton from `t`, bisection whenever the step leaves
// the bracket.  Stops BEFORE applying a step shorter than 5e-5 rad, or when |g| is at the fp32
// rounding level of x^2 + y^2 - 1 (near-tangent crossings, where Newton would only chase noise),
// or at the iteration cap -- always WITHOUT moving, so that (s, c) belong to the angle returned
// (a mismatch would open a gap between the outline arc and the limb arc).
GLF_DEV float crossing(const Arc& o, float lo, float hi, float t, bool rising, float* s, float* c) {
    t = fminf(fmaxf(t, lo), hi);
    for (int it = 0;; ++it) {
        float g, h;
        eval_g(o, t, &g, &h, s, c);
        if ((g > 0.f) == rising) hi = t; else lo = t;
        float tn = t - fast_div(g, h + h);
        if (!(tn > lo && tn < hi)) tn = 0.5f * (lo + hi);
        if (fabsf(tn - t) < 5e-5f || fabsf(g) < 1.5e-7f || it == 23) break;
        t = tn;
    }
    return t;
}

// acos for a FIRST GUESS only (error < 0.02 rad): sqrt(2(1-r)) series, mirrored for r < 0.
GLF_DEV float rough_acos(float r) {
    const float q = 1.f - fabsf(r);
    const float u = mufu_sqrt(q + q) * fmaf(q, fmaf(q, 0.01875f, 0.0833333f), 1.f);
    return r < 0.f ? kPiF - u : u;
}

// Critical point of g near the unit vector (c, s): Newton on h = g'/2 by small rotations, kept
// inside the quadrant with sign pattern (sx, sy).  SGN = +1: the maximum (h' < 0 there; where the
// curvature has the wrong sign the step is a fixed 0.5 rad uphill), SGN = -1: the minimum.
// Stops after a step shorter than 1e-3 rad (the error left is ~ that step squared).
template <int SGN>
GLF_DEV void critical_point(float xc, float yc, float a, float b, float* c,
                                               float* s, float sx, float sy) {
    for (int it = 0; it < 12; ++it) {
        const float x = fmaf(a, *c, xc), y = fmaf(b, *s, yc);
        const float bc = b * *c, as = a * *s;
        const float h = bc * y - as * x;
        const float hp = fmaf(bc, bc, as * as) - fmaf(b * *s, y, a * *c * x);
        float d = (float(SGN) * hp < 0.f) ? -fast_div(h, hp) : copysignf(0.5f, float(SGN) * h);
        d = fminf(fmaxf(d, -0.5f), 0.5f);
        // rotate (c, s) by d: sin d, cos d to O(d^7), then renormalise
        const float d2 = d * d;
        const float sd = d * fmaf(d2, fmaf(d2, 1.f / 120.f, -1.f / 6.f), 1.f);
        const float cd = fmaf(d2, fmaf(d2, fmaf(d2, -1.f / 720.f, 1.f / 24.f), -0.5f), 1.f);
        float cn = *c * cd - *s * sd, sn = *s * cd + *c * sd;
        cn = sx * fmaxf(sx * cn, 0.f);
        sn = sy * fmaxf(sy * sn, 0.f);
        const float rn = mufu_rsqrt(fmaf(cn, cn, sn * sn));
        *c = cn * rn;
        *s = sn * rn;
        if (fabsf(d) < 1e-3f) break;
    }
}

// Is the star centre inside the outline's evolute, A^(2/3) + B^(2/3) < (a^2 - b^2)^(2/3) (a second
// pair of critical points of g)?  Decided with a 30 % safety margin towards "yes": just outside the evolute the maximum of g is nearly
// degenerate and the unbracketed Newton of critical_point converges slowly (the generic path
// is always correct, only slower); A, B < e2 is the cheap necessary condition tested first.
GLF_DEV bool evolute_inside(float A, float B, float e2) {
    const float ie = mufu_rcp(e2);
    const float ca = cbrtf(A * ie), cb = cbrtf(B * ie);
    return fmaf(ca, ca, cb * cb) < 1.3f;
}

// Blocked fraction delta = k0 A_flat + k1 A_lin + k2 A_quad for an outline with centre (xc, yc) in
// the kernel frame (any signs), semi-axes a >= b > 0, a < 1/2.  k0, k1, k2 = c0, c1, c2 of R8 divided
// by pi (1 - u1/3 - u2/6).  Returns 0 when the overlap is empty.
// EVOL_EXACT (the bare-geometry kernel, where very flat outlines near the limb are common: config 5):
// decide the evolute regime with evolute_inside() instead of its cheap necessary condition alone, and
// run the bracketed search with MUFU sine/cosine (glc::gtrig<true>).
template <bool EVOL_EXACT = false>
GLF_DEV float blocked_f32(const TrapNode* trap, float xc_in, float yc_in, float a, float b, float k0,
                          float k1, float k2) {
    const float xc = fabsf(xc_in), yc = fabsf(yc_in);   // mirror images have the same areas
    const float r0sq = fmaf(xc, xc, yc * yc);
    const float reach = 1.f + a;
    if (r0sq >= reach * reach) return 0.f;
    const float ab = a * b, u = b * xc, v = a * yc;
    const float e2 = (a - b) * (a + b);
    const float r0 = r0sq * mufu_rsqrt(fmaxf(r0sq, 1e-30f));
    const float Aa = a * xc, Bb = b * yc;
    // nh = half the trapezoid order for an outline wholly inside the disc, 0 = not (yet) known to be
    int nh = 0;
    float cf = 1.f, sf = 0.f, gfar = 0.f;
    if (r0 + a <= 0.99f) {
        // well inside the limb (gap >= 0.01): 16 fixed nodes; 8 once the gap exceeds the semi-major
        // axis or 0.3 (error <= 6e-9 in flux on the config-5 sample)
        nh = (r0 + a + a <= 1.f || r0 + a <= 0.7f) ? 4 : 8;
        if (fmaf(4.f, a, r0) <= 1.f || r0 + a <= 0.5f) nh = 3;   // deep inside: six immediate nodes
    } else if (Aa < e2 && Bb < e2 && (!EVOL_EXACT || evolute_inside(Aa, Bb, e2))) {
        // the star centre lies inside the evolute (up to four crossings): bracketed search
        float A[3];
        if (!glc::overlap_areas<float, 16, EVOL_EXACT>(xc, yc, a, b, c_gl_phi, c_gl_om, A)) return 0.f;
        return fmaf(k0, A[0], fmaf(k1, A[1], k2 * A[2]));
    } else {
        // farthest outline point from the star centre: the only maximum of g (first quadrant)
        const float rn = mufu_rsqrt(fmaf(Aa, Aa, Bb * Bb));   // Aa, Bb not both 0 here (r0 > 0.49)
        cf = Aa * rn;
        sf = Bb * rn;
        critical_point<1>(xc, yc, a, b, &cf, &sf, 1.f, 1.f);
        const float xf = fmaf(a, cf, xc), yf = fmaf(b, sf, yc);
        gfar = fmaf(xf, xf, fmaf(yf, yf, -1.f));
        if (gfar <= 0.f) nh = (gfar < -0.04f) ? 8 : 16;   // wholly inside, close to the limb
    }
    if (nh) {
        // whole-outline closed forms: A_flat = pi a b, A_quad = pi a b (r0^2 + (a^2 + b^2)/4)
        const float in_flat = kPiF * ab;
        const float in_quad = in_flat * fmaf(0.25f, fmaf(a, a, b * b), r0sq);
        const float lin = (nh == 3) ? whole_outline_lin6(xc, yc, a, b, ab, u, v)
                                    : whole_outline_lin(trap, nh, xc, yc, a, b, ab, u, v);
        return fmaf(k0, in_flat, fmaf(k1 * (1.f / 3.f), lin, k2 * in_quad));
    }
    // the outline crosses the limb twice (or misses the disc).  tau = t - t_far in [0, 2 pi).
    Arc o = {xc, yc, a, b, cf, sf};
    float tsplit = kPiF;
    const float xo = fmaf(-a, cf, xc), yo = fmaf(-b, sf, yc);   // the point opposite t_far
    float gsplit = fmaf(xo, xo, fmaf(yo, yo, -1.f));
    if (gsplit >= 0.f) {
        // mostly outside: find the nearest outline point (third quadrant) and its tau
        float cn = -cf, sn = -sf;
        critical_point<-1>(xc, yc, a, b, &cn, &sn, -1.f, -1.f);
        const float xn = fmaf(a, cn, xc), yn = fmaf(b, sn, yc);
        gsplit = fmaf(xn, xn, fmaf(yn, yn, -1.f));
        if (gsplit >= 0.f) return 0.f;
        float dtau = atan2f(cf * sn - sf * cn, cf * cn + sf * sn);   // in (-pi, pi]
        tsplit = dtau < 0.f ? dtau + kTwoPiF : dtau;
    }
    // half-cosine model of g between its maximum and the split point (exact for a circle)
    const float mid = 0.5f * (gfar + gsplit), amp = 0.5f * (gfar - gsplit);
    const float uu = rough_acos(fminf(fmaxf(-fast_div(mid, amp), -1.f), 1.f)) * (1.f / kPiF);
    float s1, c1, s2, c2;
    const float t1 = crossing(o, 0.f, tsplit, uu * tsplit, false, &s1, &c1);
    const float t2 = crossing(o, tsplit, kTwoPiF, kTwoPiF - uu * (kTwoPiF - tsplit), true, &s2, &c2);
    // ---- outline arc [t1, t2] (inside the disc): flat and quad in closed form
    glc::Outline<float> oo = {xc, yc, a, b, e2};
    const glc::ArcCoef<float> k = glc::arc_coefficients(oo);
    const float dt = t2 - t1;
    float f1, q1, f2, q2;
    glc::arc_primitive(k, s1, c1, &f1, &q1);
    glc::arc_primitive(k, s2, c2, &f2, &q2);
    float Aflat = 0.5f * fmaf(k.ab, dt, f2 - f1);
    float Aquad = 0.25f * fmaf(k.k0, dt, q2 - q1);
    // ---- f_lin: 16-point Gauss-Legendre in z, t = tm + hw (3z - z^3)/2
    const float hw = 0.5f * dt;
    float sm, cm;
    abs_trig(o, t1 + hw, &sm, &cm);
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float sd, cd;
        const float dd = hw * c_gl_phi[i];   // in [0, pi]
        sd = mufu_sin(dd);
        cd = mufu_cos(dd);
        const float cp = cm * cd - sm * sd, sp = sm * cd + cm * sd;
        const float cq = cm * cd + sm * sd, sq = sm * cd - cm * sd;
        const float xp = fmaf(a, cp, xc), yp = fmaf(b, sp, yc);
        const float xq = fmaf(a, cq, xc), yq = fmaf(b, sq, yc);
        const float m2p = fmaf(-xp, xp, fmaf(-yp, yp, 1.f));
        const float m2q = fmaf(-xq, xq, fmaf(-yq, yq, 1.f));
        const float fp = fmaf(u, cp, fmaf(v, sp, ab)), fq = fmaf(u, cq, fmaf(v, sq, ab));
        acc = fmaf(c_gl_om[i], pair_term<true>(m2p, fp, m2q, fq), acc);
    }
    float Alin = (1.f / 3.f) * hw * acc;
    // ---- limb arc from the exit point (t2) counter-clockwise back to the entry point (t1)
    const float xa = fmaf(a, c2, xc), ya = fmaf(b, s2, yc);
    const float xb = fmaf(a, c1, xc), yb = fmaf(b, s1, yc);
    const float dl = atan2f(xa * yb - ya * xb, xa * xb + ya * yb);
    Aflat = fmaf(0.5f, dl, Aflat);
    Alin = fmaf(1.f / 3.f, dl, Alin);
    Aquad = fmaf(0.25f, dl, Aquad);
    return fmaf(k0, Aflat, fmaf(k1, Alin, k2 * Aquad));
}

}  // namespace glf
