// gl_hot.cuh -- hot_kernel: the COMMON path of the fused fp32 transit kernel and nothing else
// (DESIGN.md 5.4).  A walker is "simple" when its orbit is circular (eqs. 9-10 as
// printed), n_ss <= 32, its transit window is short (|phi| <= 0.8 rad), at most MAXEP transits fall
// inside the series, the star centre can never lie inside the outline's evolute while the outline
// is near the limb (so the outline crosses the limb at most twice), and the series is sorted.
// Simple walkers are finished here; every other walker is DEFERRED: the kernel leaves a marker (a
// NaN with a payload) in the walker's output slot and the full-featured transit_kernel, launched
// right behind with programmatic dependent launch, redoes exactly the marked walkers.  Invalid
// walkers (NaN row, chi^2 = +inf) are finished here too.
//
// Why a separate kernel: the full-featured kernel is ~340 KB of SASS (fp64 Kepler, the
// four-crossing search, libm slow paths); on a K2-shaped batch (config 3) it spent its time in
// instruction fetch and barriers, not arithmetic (profiles/r01_v5.md).  This one has no fp64
// arithmetic beyond the time difference t_i - t_c and the chi^2 sum, no libm call, no list, and
// one CTA (or one cluster, for long in-window ranges) per walker:
//   1. at entry every thread loads one COARSE sample of the series (every stride-th time) into
//      shared memory and, unless the caller vouches for the order, checks its share of adjacent
//      pairs; three threads of three warps run the walker prelude (orbit+window / outline / limb
//      darkening) side by side;
//   2. for a sorted series the in-window exposures of transit epoch n are ONE index range
//      [lo_n, hi_n): a warp per epoch finds it by binary search in the coarse table + one round of
//      global loads -- no scan of the series, no ballots, no compaction, no list;
//   3. out-of-window flux = 1 is plain 16-byte stores;
//   4. lane = (exposure, sub-exposure): position from dt = (float)(t_i - t_c) (the fp64 phase
//      reduction is gone: the epoch is known from the range), a3 + a4 by blocked_hot(), exposure
//      mean by shuffles, chi^2 term in the cancellation-free form d (2 o r + d), d = dbar/sigma;
//   5. chi^2 = S + sum of the terms, S = sum_i ((obs_i-1)/sigma_i)^2 once per series.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "gl_fast32.cuh"

// Development aid: a debug build (a translation unit outside the product tree) may define GLH_TL(k)
// to stamp the phases of a CTA; in the product it is nothing.
#ifndef GLH_TL
#define GLH_TL(k) do { } while (0)
#endif

namespace glh {

namespace cg = cooperative_groups;

constexpr int HOT_NT = 512;           // threads per CTA
constexpr int HOT_NW = HOT_NT / 32;
constexpr int MAXEP = 8;              // transit epochs of one walker inside one series segment
constexpr int MAXC = 8;               // CTAs per cluster (portable limit)
constexpr uint32_t MARK_BITS = 0x7fc0deadu;   // "deferred": a quiet NaN no arithmetic here produces

// cos, sin of pi k / 16, k = 0..15 (glf::whole_outline_lin's table), statically initialised.
__constant__ float2 c_trap16[16] = {
    {1.f, 0.f}, {0.980785251f, 0.195090324f}, {0.923879504f, 0.382683426f},
    {0.831469595f, 0.555570245f}, {0.707106769f, 0.707106769f}, {0.555570245f, 0.831469595f},
    {0.382683426f, 0.923879504f}, {0.195090324f, 0.980785251f}, {0.f, 1.f},
    {-0.195090324f, 0.980785251f}, {-0.382683426f, 0.923879504f}, {-0.555570245f, 0.831469595f},
    {-0.707106769f, 0.707106769f}, {-0.831469595f, 0.555570245f}, {-0.923879504f, 0.382683426f},
    {-0.980785251f, 0.195090324f}};

// Smoothed 16-point Gauss-Legendre rule (gl_tables.h: phi(z_k), w_k phi'(z_k), positive nodes),
// as literals so that the unrolled loop carries them as immediates (no constant-cache miss on the
// critical path of a cold launch).  tests/test_fast32_host.py checks them against the generator.
#define GLH_GL_PHI {0.142089903f, 0.411239654f, 0.638983905f, 0.808870733f, 0.917576194f, 0.974130571f, 0.995477259f, 0.999832094f}
#define GLH_GL_OM {0.281610548f, 0.252184302f, 0.200506464f, 0.13872686f, 0.0802668259f, 0.035781879f, 0.010064343f, 0.000858796586f}

// sin, cos of x for |x| <= 0.8 rad (the orbital angle of an in-window sub-exposure): Taylor
// polynomials to x^9 / x^10, truncation error < 3e-9 relative.  The sine keeps full RELATIVE
// precision at small x, which y0 = (a/R*) sin(phi) needs (a/R* ~ 230).
__device__ __forceinline__ void small_sincos(float x, float* s, float* c) {
    const float x2 = x * x;
    float ps = fmaf(x2, 2.7557319e-6f, -1.9841270e-4f);
    ps = fmaf(x2, ps, 8.3333333e-3f);
    ps = fmaf(x2, ps, -1.6666667e-1f);
    *s = fmaf(x * x2, ps, x);
    float pc = fmaf(x2, -2.7557319e-7f, 2.4801587e-5f);
    pc = fmaf(x2, pc, -1.3888889e-3f);
    pc = fmaf(x2, pc, 4.1666667e-2f);
    pc = fmaf(x2, pc, -0.5f);
    *c = fmaf(x2, pc, 1.f);
}

// sin, cos of an arbitrary angle given in fp64 (prelude only: xi, eta): reduced to [-pi, pi] in
// fp64, to [-pi/4, pi/4] in fp32, then the polynomials above (|x| <= 0.786).  No libm, no slow path.
__device__ __forceinline__ void angle_sincos(double ang, float* s, float* c) {
    const double k = rint(ang * 0.15915494309189535);
    const float r = (float)fma(-k, 6.283185307179586, ang);   // |r| <= pi (+ rounding)
    const float j = rintf(r * 0.636619772f);                  // quadrant, -2..2
    float y = fmaf(-j, 1.57079625f, r);                       // pi/2 = 1.57079625 + 7.54978942e-8
    y = fmaf(-j, 7.54978942e-8f, y);
    float sy, cy;
    small_sincos(y, &sy, &cy);
    const int q = ((int)j) & 3;
    const float ss = (q & 1) ? cy : sy, cc = (q & 1) ? sy : cy;
    *s = (q & 2) ? -ss : ss;
    *c = ((q + 1) & 2) ? -cc : cc;
}

// 1/x to ~1 ulp: MUFU reciprocal + one Newton step (no IEEE-division slow path in the code).
__device__ __forceinline__ float rcp_nr(float x) {
    const float r = glf::mufu_rcp(x);
    return fmaf(r, fmaf(-x, r, 1.f), r);
}

// atan2(y, x) in (-pi, pi], relative error 2e-7 (octant reduction + the Cephes atanf polynomial on
// [-tan(pi/8), tan(pi/8)]); divisions by rcp_nr.  atan2(0, 0) = 0.
__device__ __forceinline__ float atan2_fast(float y, float x) {
    const float ax = fabsf(x), ay = fabsf(y);
    const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
    float t = mx > 0.f ? mn * rcp_nr(mx) : 0.f;
    float base = 0.f;
    if (t > 0.41421356f) {
        t = (t - 1.f) * rcp_nr(t + 1.f);
        base = 0.78539816339744830962f;
    }
    const float z = t * t;
    float pz = fmaf(8.05374449538e-2f, z, -1.38776856032e-1f);
    pz = fmaf(pz, z, 1.99777106478e-1f);
    pz = fmaf(pz, z, -3.33329491539e-1f);
    float r = base + fmaf(pz * z, t, t);
    if (ay > ax) r = 1.57079632679489661923f - r;
    if (x < 0.f) r = 3.14159265358979323846f - r;
    return y < 0.f ? -r : r;
}

// asin(x) for 0 <= x <= 0.5 from below (series to x^13: short by at most 1.1e-6 relative; the
// window it sizes is widened by 1e-5).
__device__ __forceinline__ float asin_small(float x) {
    const float x2 = x * x;
    float q = fmaf(x2, 1.7352764e-2f, 2.2372159e-2f);
    q = fmaf(x2, q, 3.0381944e-2f);
    q = fmaf(x2, q, 4.4642857e-2f);
    q = fmaf(x2, q, 7.5e-2f);
    q = fmaf(x2, q, 1.6666667e-1f);
    return fmaf(x * x2, q, x);
}

// Blocked fraction delta = k0 A_flat + k1 A_lin + k2 A_quad (R8; eqs. 21-23) for an
// outline that crosses the limb AT MOST TWICE (the caller has excluded the evolute regime for the
// whole walker): glf::blocked_f32 (gl_fast32.cuh) without its generic branch, with
// the Gauss-Legendre table as immediates.  trap = shared-memory copy of c_trap16.
__device__ __forceinline__ float blocked_hot(const glf::TrapNode* trap, float xc_in, float yc_in, float a,
                                             float b, float ab, float e2, float k0, float k1, float k2) {
    using namespace glf;
    const float xc = fabsf(xc_in), yc = fabsf(yc_in);   // mirror images have the same areas
    const float r0sq = fmaf(xc, xc, yc * yc);
    const float reach = 1.f + a;
    if (r0sq >= reach * reach) return 0.f;
    const float u = b * xc, v = a * yc;
    const float r0 = r0sq * mufu_rsqrt(fmaxf(r0sq, 1e-30f));
    int nh = 0;
    float cf = 1.f, sf = 0.f, gfar = 0.f;
    if (r0 + a <= 0.99f) {
        nh = (r0 + a + a <= 1.f || r0 + a <= 0.7f) ? 4 : 8;
        if (fmaf(4.f, a, r0) <= 1.f || r0 + a <= 0.5f) nh = 3;
    } else {
        const float Aa = a * xc, Bb = b * yc;
        const float rn = mufu_rsqrt(fmaf(Aa, Aa, Bb * Bb));
        cf = Aa * rn;
        sf = Bb * rn;
        critical_point<1>(xc, yc, a, b, &cf, &sf, 1.f, 1.f);
        const float xf = fmaf(a, cf, xc), yf = fmaf(b, sf, yc);
        gfar = fmaf(xf, xf, fmaf(yf, yf, -1.f));
        if (gfar <= 0.f) nh = (gfar < -0.04f) ? 8 : 16;
    }
    if (nh) {
        const float in_flat = kPiF * ab;
        const float in_quad = in_flat * fmaf(0.25f, fmaf(a, a, b * b), r0sq);
        const float lin = (nh == 3) ? whole_outline_lin6(xc, yc, a, b, ab, u, v)
                                    : whole_outline_lin(trap, nh, xc, yc, a, b, ab, u, v);
        return fmaf(k0, in_flat, fmaf(k1 * (1.f / 3.f), lin, k2 * in_quad));
    }
    Arc o = {xc, yc, a, b, cf, sf};
    float tsplit = kPiF;
    const float xo = fmaf(-a, cf, xc), yo = fmaf(-b, sf, yc);
    float gsplit = fmaf(xo, xo, fmaf(yo, yo, -1.f));
    if (gsplit >= 0.f) {
        float cn = -cf, sn = -sf;
        critical_point<-1>(xc, yc, a, b, &cn, &sn, -1.f, -1.f);
        const float xn = fmaf(a, cn, xc), yn = fmaf(b, sn, yc);
        gsplit = fmaf(xn, xn, fmaf(yn, yn, -1.f));
        if (gsplit >= 0.f) return 0.f;
        const float dtau = atan2_fast(cf * sn - sf * cn, cf * cn + sf * sn);
        tsplit = dtau < 0.f ? dtau + kTwoPiF : dtau;
    }
    const float mid = 0.5f * (gfar + gsplit), amp = 0.5f * (gfar - gsplit);
    const float uu = rough_acos(fminf(fmaxf(-fast_div(mid, amp), -1.f), 1.f)) * (1.f / kPiF);
    float s1, c1, s2, c2;
    const float t1 = crossing(o, 0.f, tsplit, uu * tsplit, false, &s1, &c1);
    const float t2 = crossing(o, tsplit, kTwoPiF, kTwoPiF - uu * (kTwoPiF - tsplit), true, &s2, &c2);
    glc::Outline<float> oo = {xc, yc, a, b, e2};
    const glc::ArcCoef<float> k = glc::arc_coefficients(oo);
    const float dt = t2 - t1;
    float f1, q1, f2, q2;
    glc::arc_primitive(k, s1, c1, &f1, &q1);
    glc::arc_primitive(k, s2, c2, &f2, &q2);
    float Aflat = 0.5f * fmaf(k.ab, dt, f2 - f1);
    float Aquad = 0.25f * fmaf(k.k0, dt, q2 - q1);
    const float hw = 0.5f * dt;
    float sm, cm;
    abs_trig(o, t1 + hw, &sm, &cm);
    constexpr float gl_phi[8] = GLH_GL_PHI, gl_om[8] = GLH_GL_OM;
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float dd = hw * gl_phi[i];   // in [0, pi]
        const float sd = mufu_sin(dd), cd = mufu_cos(dd);
        const float cp = cm * cd - sm * sd, sp = sm * cd + cm * sd;
        const float cq = cm * cd + sm * sd, sq = sm * cd - cm * sd;
        const float xp = fmaf(a, cp, xc), yp = fmaf(b, sp, yc);
        const float xq = fmaf(a, cq, xc), yq = fmaf(b, sq, yc);
        const float m2p = fmaf(-xp, xp, fmaf(-yp, yp, 1.f));
        const float m2q = fmaf(-xq, xq, fmaf(-yq, yq, 1.f));
        const float fp = fmaf(u, cp, fmaf(v, sp, ab)), fq = fmaf(u, cq, fmaf(v, sq, ab));
        acc = fmaf(gl_om[i], pair_term<true>(m2p, fp, m2q, fq), acc);
    }
    float Alin = (1.f / 3.f) * hw * acc;
    const float xa = fmaf(a, c2, xc), ya = fmaf(b, s2, yc);
    const float xb = fmaf(a, c1, xc), yb = fmaf(b, s1, yc);
    const float dl = atan2_fast(xa * yb - ya * xb, xa * xb + ya * yb);
    Aflat = fmaf(0.5f, dl, Aflat);
    Alin = fmaf(1.f / 3.f, dl, Alin);
    Aquad = fmaf(0.25f, dl, Aquad);
    return fmaf(k0, Aflat, fmaf(k1, Alin, k2 * Aquad));
}

// ------------------------------------------------------------------------------------------
// Kernel arguments.  Unit of work = (walker, series segment): one cluster of gridDim.x CTAs.
// chi^2 calls use nseg = 1 (the sum over a walker's series stays in one cluster); flux-only calls
// may split a long series into nseg segments of seglen exposures, one single-CTA unit each.
// ------------------------------------------------------------------------------------------
struct HotArgs {
    const double* params;   // [B, 12]
    const double* times;    // [T]
    const double* obs;      // [T]  raw series (PRE = false)
    const double* sigma;    // [T]
    const float2* ow;       // [T]  (obs - 1, 1/sigma) in fp32 (PRE = true: gl_series)
    float* flux;            // [B, T] or nullptr
    float* chi2;            // [B] or nullptr
    int* status;            // nullptr, or a word that is set to 1 when any unit is deferred
    double S;               // PRE: baseline sum_i ((obs_i - 1)/sigma_i)^2
    double t_exp;
    float inv_ss, doff, off0;   // 1/n_ss, t_exp/n_ss, (0.5/n_ss - 0.5) t_exp: sub-exposure j sits at off0 + j doff (R18)
    int B, T, n_ss, nseg, seglen;   // B * nseg < 2^31
    int sorted_known;       // the caller vouches that times is non-decreasing (gl_series checked it)
};

enum { CLS_SIMPLE = 0, CLS_INVALID = 1, CLS_DEFER = 2 };

struct Unit {
    double tc[MAXEP];             // conjunction time of each listed transit epoch
    double qlo[MAXEP], qhi[MAXEP];   // its window [qlo, qhi) in time
    int lo[MAXEP], hi[MAXEP];     // ... and in index (relative to the segment)
    int nep;
    int cls_orbit, defer_shape;
    float w, aR, bimp, a, b, cpsi, spsi, k0, k1, k2;
};

// Orbit half of the prelude (one thread): validity, window, transit epochs inside [tfirst, tlast].
// e != 0 (or NaN) is deferred without looking further: the full kernel owns those rules.
__device__ __forceinline__ void hot_prelude_orbit(const double* p, double t_exp, int n_ss,
                                                  double tfirst, double tlast, Unit* u) {
    const double t0 = p[0], P = p[1], aR = p[2], b = p[3], e = p[4];
    const double Rp = p[6], f = p[7], u1 = p[10], u2 = p[11];
    u->nep = 0;
    if (!(e == 0.0) || n_ss > 32) {
        u->cls_orbit = CLS_DEFER;
        return;
    }
    bool ok = true;
#pragma unroll
    for (int k = 0; k < 12; ++k) ok = ok && (fabs(p[k]) <= 1.79769313486231570e308);   // finite
    ok = ok && (P > 0.0) && (Rp > 0.0) && (Rp < 0.5) && (f >= 0.0) && (f < 1.0) && (aR > 1.0) &&
         (1.0 - u1 / 3.0 - u2 / 6.0 > 0.0) && (fabs(b) <= aR);
    if (!ok) {
        u->cls_orbit = CLS_INVALID;
        return;
    }
    // PAPER.md:85-87 eqs. 9-10: the centre is within `reach` of the star centre iff
    // sin^2(phi) < [(reach/aR)^2 - cos^2 i] / sin^2 i (and cos(phi) > 0)
    const float aRf = (float)aR, bf = (float)b;
    const float iaR = rcp_nr(aRf);
    const float cosi = bf * iaR, ci2 = cosi * cosi;
    const float reach = (1.f + (float)Rp) * (1.f + 1e-5f);
    const float q = reach * iaR;
    const float S2 = glf::fast_div(q * q - ci2, 1.f - ci2);
    // 1/P in fp64 by Newton from the MUFU reciprocal (P must be in fp32's range for that)
    if (!(P > 1e-30 && P < 1e30)) {
        u->cls_orbit = CLS_DEFER;
        return;
    }
    double inv_P = (double)glf::mufu_rcp((float)P);
    inv_P = inv_P * fma(-P, inv_P, 2.0);
    inv_P = inv_P * fma(-P, inv_P, 2.0);
    const float w = (float)(6.28318530717958647692 * inv_P);
    u->w = w;
    u->aR = aRf;
    u->bimp = bf;
    u->cls_orbit = CLS_SIMPLE;
    if (S2 <= 0.f) return;   // never transits: nep = 0, flux = 1 everywhere
    if (!(S2 <= 0.25f)) {    // long window (or NaN: face-on orbit): not the common path
        u->cls_orbit = CLS_DEFER;
        return;
    }
    const float phimax = asin_small(glf::mufu_sqrt(S2) * (1.f + 1e-6f)) * (1.f + 1e-5f);
    if (!(phimax + w * (float)t_exp <= 0.8f)) {   // small_sincos's range
        u->cls_orbit = CLS_DEFER;
        return;
    }
    const double hw = (double)phimax * P * 0.15915494309189535 + 0.5 * t_exp + 1e-9 * P;
    const double nlo = ceil((tfirst - hw - t0) * inv_P - 1e-9);
    const double nhi = floor((tlast + hw - t0) * inv_P + 1e-9);
    const double cnt = nhi - nlo + 1.0;
    if (!(cnt <= (double)MAXEP)) {   // also NaN / infinite time stamps
        u->cls_orbit = CLS_DEFER;
        return;
    }
    const int nep = cnt > 0.0 ? (int)cnt : 0;
    for (int k = 0; k < nep; ++k) {
        const double tc = fma(nlo + (double)k, P, t0);
        u->tc[k] = tc;
        u->qlo[k] = tc - hw;
        u->qhi[k] = tc + hw;
    }
    u->nep = nep;
}

// Outline half (one thread): the oblate spheroid's projected outline in closed form -- semi-major
// axis Rp along (sin xi, cos xi), semi-minor Rp sqrt(1 - f(2-f) cos^2 eta) (eqs. 6, 11-13 with
// a = Rp(1-f), b = c = Rp, zeta = 0: SURVEY.md 8(c) "equation checks"; tests compare with the
// general eigen-axes of the full kernel) -- and the evolute exclusion: a second pair of critical
// points of g needs a xc < e2 and b yc < e2 (gl_core.cuh), i.e. r0 < e2 sqrt(1/a^2 + 1/b^2); if
// that is below 0.99 - a, blocked_hot's near-limb branch (r0 + a > 0.99) can never see one.
__device__ __forceinline__ void hot_prelude_shape(const double* p, Unit* u) {
    const float Rp = (float)p[6], f = (float)p[7];
    float sx, cx, se, ce;
    angle_sincos(p[8], &sx, &cx);
    angle_sincos(p[9], &se, &ce);
    const float a = Rp;
    const float b = Rp * glf::mufu_sqrt(fmaxf(1.f - f * (2.f - f) * ce * ce, 0.f));
    u->a = a;
    u->b = b;
    u->cpsi = sx;
    u->spsi = cx;
    const float e2 = (a - b) * (a + b);
    const float ia = glf::mufu_rcp(a), ib = glf::mufu_rcp(b);
    const float rmax = e2 * glf::mufu_sqrt(fmaf(ia, ia, ib * ib));
    u->defer_shape = !(rmax <= (0.99f - a) * 0.98f);   // NaN (b = 0) defers too
}

__device__ __forceinline__ void hot_prelude_ld(const double* p, Unit* u) {
    const double u1 = p[10], u2 = p[11];
    const float pn = (float)(3.14159265358979323846 * (1.0 - u1 / 3.0 - u2 / 6.0));
    const float ipn = rcp_nr(pn);
    u->k0 = (float)(1.0 - u1 - 2.0 * u2) * ipn;
    u->k1 = (float)(u1 + 2.0 * u2) * ipn;
    u->k2 = (float)u2 * ipn;
}

// #{i in [0, n) : seg[i] < q} for a non-decreasing segment, by the 16 lanes of a half-warp (all 32
// lanes of the warp call this; `hl` = lane & 15).  coarse[k] = seg[k stride], k < nc.
__device__ __forceinline__ int lower_bound_half(const double* __restrict__ seg, int n,
                                                const double* coarse, int nc, int stride, double q,
                                                int hl) {
    int lo = 0, hi = nc;
    while (lo < hi) {   // identical in every lane
        const int mid = (lo + hi) >> 1;
        if (coarse[mid] < q) lo = mid + 1; else hi = mid;
    }
    // (no early exit: the two halves of the warp meet again at the shuffles below)
    const bool none = (lo == 0);
    const int base = none ? 0 : (lo - 1) * stride, end = none ? 0 : min(lo * stride, n);
    int cnt = 0;
    for (int m = base + 1 + hl; m < end; m += 16) cnt += (seg[m] < q) ? 1 : 0;
#pragma unroll
    for (int off = 8; off > 0; off >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, off);
    return none ? 0 : base + 1 + cnt;
}

template <bool PRE>
__global__ void __launch_bounds__(HOT_NT, 2) hot_kernel(const HotArgs A) {
    asm volatile("griddepcontrol.launch_dependents;");   // the fallback launch may become resident
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int csize = (int)gridDim.x, crank = (int)blockIdx.x;
    cg::cluster_group cluster = cg::this_cluster();

    __shared__ Unit su;
    __shared__ double s_coarse[HOT_NT];
    __shared__ double s_red[HOT_NW];
    __shared__ double s_gather[2][MAXC];   // rank 0's copy collects the cluster's chi^2 partials
    __shared__ int s_gflag[2][MAXC];       // ... and their "my share of the series is unsorted" flags
    __shared__ double s_row[3][12];
    __shared__ glf::TrapNode s_trap[16];
    if (tid < 16) s_trap[tid] = glf::TrapNode{c_trap16[tid].x, c_trap16[tid].y};

    const int S = A.n_ss;
    const float inv_ss = A.inv_ss, doff = A.doff, off0 = A.off0;
    const bool want_chi2 = A.chi2 != nullptr, want_flux = A.flux != nullptr;
    const int ntot = csize * HOT_NT, gtid = crank * HOT_NT + tid;
    int wpar = 0;
    // no CTA may write into rank 0's shared memory before rank 0 runs: arrive now, wait before the
    // first push
    bool started = (csize == 1);
    if (csize > 1) cluster.barrier_arrive();

    const unsigned nunits = (unsigned)A.B * (unsigned)A.nseg;
    for (unsigned un = blockIdx.y; un < nunits; un += gridDim.y) {
        const int wk = A.nseg == 1 ? (int)un : (int)(un / (unsigned)A.nseg);
        const int t_lo = (int)(un - (unsigned)wk * (unsigned)A.nseg) * A.seglen;
        const double* __restrict__ seg = A.times + t_lo;
        const int nT = min(A.seglen, A.T - t_lo);
        const int stride = (nT + HOT_NT - 1) / HOT_NT;
        const int nc = (nT + stride - 1) / stride;
        const double* __restrict__ p = A.params + (size_t)wk * 12;
        float* frow = want_flux ? A.flux + (size_t)wk * A.T + t_lo : nullptr;

        __syncthreads();   // the previous unit's shared data is dead
        GLH_TL(0);
        // ---- 1. coarse samples, order check (this CTA's share of the adjacent pairs, incl. the pair
        // that straddles into the next segment), prelude
        if (tid < nc) s_coarse[tid] = seg[(size_t)tid * stride];
        int unsorted = 0;
        if (!A.sorted_known) {
            const int npairs = min(nT, A.T - t_lo - 1);
            for (int i = gtid; i < npairs; i += ntot) unsorted |= !(seg[i] <= seg[i + 1]);
        }
        // the parameter row: ONE coalesced 96-byte request per prelude warp (it may sit in host memory
        // that the device reads over PCIe: gl_series_loglike), handed to lane 0 through shared memory
        if (warp < 3) {
            if (lane < 12) s_row[warp][lane] = p[lane];
            __syncwarp();
            if (tid == 0) hot_prelude_orbit(s_row[0], A.t_exp, S, seg[0], seg[nT - 1], &su);
            if (tid == 32) hot_prelude_shape(s_row[1], &su);
            if (tid == 64) hot_prelude_ld(s_row[2], &su);
        }
        unsorted = __syncthreads_or(unsorted);
        GLH_TL(1);

        int cls = su.cls_orbit;
        if (cls == CLS_SIMPLE && su.defer_shape) cls = CLS_DEFER;
        const int nep = (cls == CLS_SIMPLE) ? su.nep : 0;

        // ---- 2. index range of every listed epoch: warp = epoch, half-warp = end of the window
        if (warp < nep) {
            const int half = lane >> 4;
            const double q = half ? su.qhi[warp] : su.qlo[warp];
            const int idx = lower_bound_half(seg, nT, s_coarse, nc, stride, q, lane & 15);
            if ((lane & 15) == 0) (half ? su.hi : su.lo)[warp] = idx;
        }
        __syncthreads();
        GLH_TL(2);

        double acc = 0.0;   // this lane's chi^2 terms
        if (cls == CLS_INVALID) {
            if (frow)
                for (int i = gtid; i < nT; i += ntot) frow[i] = __int_as_float(0x7fc00000);
        } else if (cls == CLS_SIMPLE) {
            // index ranges are read from shared memory where they are needed (broadcast reads; nep is 1
            // for a single-transit series): len_k = max(hi_k - lo_k, 0) -- an unsorted share of the
            // series may give anything, the unit is then redone by the fallback kernel
            int M = 0;
            for (int k = 0; k < nep; ++k) M += max(su.hi[k] - su.lo[k], 0);
            auto inwin = [&](int i) {
                bool in = false;
#pragma unroll 1
                for (int k = 0; k < nep; ++k) in = in || (i >= su.lo[k] && i < su.hi[k]);
                return in;
            };
            GLH_TL(3);
            // ---- 4. in-window exposures.  A lane takes JS consecutive sub-exposures of one exposure
            // (JS = 1 unless the list is long), a warp G = 32 / JB whole exposures; groups are dealt
            // from both ends of the list inwards, so that ingress and egress -- the long code path --
            // start first and sit in warps of their own.
            if (M > 0) {
                const float w = su.w, aR = su.aR, bimp = su.bimp, a = su.a, b = su.b;
                const float cpsi = su.cpsi, spsi = su.spsi, k0 = su.k0, k1 = su.k1, k2 = su.k2;
                const float ab = a * b, e2 = (a - b) * (a + b);
                const long long pairs = (long long)M * S;
                const int JS = (int)min((long long)S, max(1LL, pairs / (4LL * ntot)));
                const int JB = (S + JS - 1) / JS, G = 32 / JB;
                const int my_l = lane / JB, my_b = lane - my_l * JB;
                const int W = (M + G - 1) / G;
                // sweep k hands out tasks k nwt .. (k+1) nwt - 1, in warp order on even sweeps and in
                // reverse on odd ones: the warps that opened with the outermost (expensive) groups get
                // the last, innermost ones, if any
                const int nwt = HOT_NW * csize, gw = warp * csize + crank;
                for (int k = 0; k * nwt < W; ++k) {
                    const int t = k * nwt + ((k & 1) ? nwt - 1 - gw : gw);
                    if (t >= W) continue;   // warp-uniform
                    const int g = (t & 1) ? W - 1 - (t >> 1) : (t >> 1);
                    const int v = g * G + my_l;
                    const bool active = (my_l < G) && (v < M);
                    int i = 0;
                    float delta = 0.f, ob = 0.f, rs = 0.f;
                    if (active) {
                        int n = 0, run = 0;
                        i = su.lo[0] + v;
#pragma unroll 1
                        for (int k = 0; k < nep; ++k) {   // which epoch's range holds list entry v
                            if (v >= run) {
                                n = k;
                                i = su.lo[k] + (v - run);
                            }
                            run += max(su.hi[k] - su.lo[k], 0);
                        }
                        const float dtc = (float)(seg[i] - su.tc[n]);
                        if (want_chi2 && my_b == 0) {
                            if (PRE) {
                                const float2 o2 = A.ow[t_lo + i];
                                ob = o2.x;
                                rs = o2.y;
                            } else {
                                ob = (float)(A.obs[t_lo + i] - 1.0);
                                const float sf = (float)A.sigma[t_lo + i];
                                rs = glf::mufu_rcp(sf);
                                rs = rs * fmaf(-sf, rs, 2.f);
                            }
                        }
                        const int j1 = min(S, (my_b + 1) * JS);
                        for (int j = my_b * JS; j < j1; ++j) {
                            const float phi = w * (dtc + fmaf((float)j, doff, off0));
                            float s, c;
                            small_sincos(phi, &s, &c);
                            const float x0 = bimp * c, y0 = aR * s;   // eqs. 9-10, d sin(beta) = b
                            delta += blocked_hot(s_trap, fmaf(cpsi, x0, spsi * y0), fmaf(cpsi, y0, -spsi * x0),
                                                 a, b, ab, e2, k0, k1, k2);
                        }
                    }
                    float sum = 0.f;   // exposure mean, blocks in sub-exposure order (R18)
                    for (int bb = 0; bb < JB; ++bb) sum += __shfl_sync(0xffffffffu, delta, (lane + bb) & 31);
                    if (active && my_b == 0) {
                        const float dbar = sum * inv_ss;
                        if (frow) frow[i] = 1.f - dbar;
                        const float d = dbar * rs;
                        acc += (double)(d * fmaf(2.f * ob, rs, d));   // ((o+dbar) r)^2 - (o r)^2
                    }
                }
            }
            GLH_TL(6);
            // ---- 4b. out-of-window exposures: flux = 1, 16 bytes at a time where the row allows (after the
            // evaluation: nothing waits for these stores)
            if (frow) {
                const int head = (int)((4u - (((uintptr_t)frow >> 2) & 3u)) & 3u);
                if (gtid < head && gtid < nT && !inwin(gtid)) frow[gtid] = 1.f;
                const int nchunk = nT > head ? (nT - head) >> 2 : 0;
                for (int c = gtid; c < nchunk; c += ntot) {
                    const int i0 = head + 4 * c;
                    bool hit = false;
#pragma unroll 1
                    for (int k = 0; k < nep; ++k) hit = hit || (i0 + 3 >= su.lo[k] && i0 < su.hi[k]);
                    if (!hit) {
                        *reinterpret_cast<float4*>(frow + i0) = make_float4(1.f, 1.f, 1.f, 1.f);
                    } else {
#pragma unroll
                        for (int r = 0; r < 4; ++r)
                            if (!inwin(i0 + r)) frow[i0 + r] = 1.f;
                    }
                }
                const int tail0 = head + 4 * nchunk;
                if (gtid < nT - tail0 && !inwin(tail0 + gtid)) frow[tail0 + gtid] = 1.f;
            }
        }
        GLH_TL(4);
        // ---- 5. chi^2 (and the cluster's verdict on the order of the series): CTA sum, partials
        // pushed into rank 0's shared memory, one cluster barrier, rank 0 adds them in rank order
        bool defer = (cls == CLS_DEFER);
        if (want_chi2) {
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, off);
            if (lane == 0) s_red[warp] = acc;
            if (!started) {
                cluster.barrier_wait();
                started = true;
            }
            __syncthreads();
            if (tid == 0) {
                double tot = 0.0;
                for (int k = 0; k < HOT_NW; ++k) tot += s_red[k];
                if (csize > 1) {
                    *cluster.map_shared_rank(&s_gather[wpar][crank], 0) = tot;
                    *cluster.map_shared_rank(&s_gflag[wpar][crank], 0) = unsorted;
                } else {
                    s_gather[wpar][0] = tot;
                    s_gflag[wpar][0] = unsorted;
                }
            }
            if (csize > 1) cluster.sync();
            if (crank == 0 && tid == 0) {
                double d2 = 0.0;
                int uns = 0;
                for (int r = 0; r < csize; ++r) {
                    d2 += s_gather[wpar][r];
                    uns |= s_gflag[wpar][r];
                }
                defer = defer || (uns != 0 && cls != CLS_INVALID);
                // raw series: baseline_kernel, launched before this grid (which may have started early:
                // programmatic dependent launch), writes S into chi2[0..B): wait before touching chi2
                if (!PRE) asm volatile("griddepcontrol.wait;" ::: "memory");
                float out;
                if (cls == CLS_INVALID) {
                    out = __int_as_float(0x7f800000);
                } else if (defer) {
                    out = __uint_as_float(MARK_BITS);
                } else {
                    double Sb = A.S;
                    if (!PRE) Sb = (double)*(volatile float*)&A.chi2[wk];
                    out = (Sb > 1.79769313486231570e308) ? (float)Sb : (float)(Sb + d2);
                }
                A.chi2[wk] = out;
                if (defer && A.status) *A.status = 1;
            }
            GLH_TL(5);
            wpar ^= 1;
        } else if (frow) {
            // flux-only units are single CTAs; the marker goes where this segment's row starts
            defer = defer || (unsorted != 0 && cls != CLS_INVALID);
            __syncthreads();   // every other store of this CTA to frow[0] is behind us
            if (tid == 0 && defer) {
                frow[0] = __uint_as_float(MARK_BITS);
                if (A.status) *A.status = 1;
            }
        }
    }
    if (!started) cluster.barrier_wait();
}

}  // namespace glh
