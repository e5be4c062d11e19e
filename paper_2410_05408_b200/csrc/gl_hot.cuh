// gl_hot.cuh -- hot_kernel: the fp32 transit kernel, built around the COMMON path.
// A walker is "simple" when its orbit is circular (eqs. 9-10 as printed), its transit
// window is short (|phi| <= 0.8 rad), at most MAXEP transits fall inside the series, the star centre can
// never lie inside the outline's evolute while the outline is near the limb (so the outline crosses the
// limb at most twice), and the series is sorted.  Simple walkers take the path described below; every
// other walker is only NOTED by the main loop and done, inside the same launch, by a second loop behind it
// that runs generic_unit() -- the full-featured arithmetic of greenlantern_b200.cu (fp64 phases, Kepler,
// four-crossing search), inlined THERE: behind the common path's code, never fetched unless a walker needs
// it, and with no call inside the main loop.  Invalid walkers: NaN row, chi^2 = +inf.
//
// Why a kernel of its own: round 1's single fused kernel inlined everything -- ~340 KB of SASS (fp64 Kepler, the
// four-crossing search, libm slow paths); on a K2-shaped batch (config 3) it spent its time in
// instruction fetch and barriers, not arithmetic (profiles/r01_v5.md).  This one has no fp64
// arithmetic beyond the epoch bookkeeping of the prelude, the time difference t_i - t_c and the
// chi^2 sum, no libm call, no scan of the series, and one CTA (or one cluster, for long in-window
// ranges) per walker:
//   1. at entry every thread loads one COARSE sample of the series (every stride-th time) into
//      shared memory and, unless the caller vouches for the order, checks its share of adjacent
//      pairs; FOUR threads of four warps run the walker prelude side by side (validity + window
//      angle / outline / limb darkening / period);
//   2. for a sorted series the in-window exposures of transit epoch n are ONE index range
//      [lo_n, hi_n): one warp per range end finds it by two 32-way steps in the coarse table + one
//      round of global loads -- no scan of the series, no ballots over it, no list;
//   3. out-of-window flux = 1 is plain 16-byte stores;
//   4. SPARSE list (a K2-shaped series: all (exposure, sub-exposure) pairs of the walker fit one
//      pass of the CTA): lane = pair, in time order, so neighbouring lanes run the same code path;
//      pairs whose outline is near the limb (the long path: critical points, two crossings, 16-point
//      rule) are compacted into a list and evaluated by TWO lanes each (far/near critical point,
//      first/second crossing, even/odd quadrature nodes in parallel); exposure means through shared
//      memory.  DENSE list (a JWST-shaped series): a thread takes whole exposures, all
//      sub-exposures in turn, with the same arithmetic in the same order (bit-identical values);
//   5. chi^2 = S + sum of d (2 o r + d), d = dbar/sigma (cancellation-free form of
//      ((o + dbar)/sigma)^2 - (o/sigma)^2), S = sum_i ((obs_i-1)/sigma_i)^2 once per series.
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
// CHECKED build (-DGLH_CHECKED; tests/test_gpu_parity.py builds it, the product never does): every
// shared- and global-memory index of the transit kernels is asserted to be in range, and pseudo-random
// per-CTA delays are injected in front of every cluster barrier and DSMEM access, so that
// a protocol that only works by luck of timing shows up as a wrong or irreproducible result.
// (compute-sanitizer is closed on the GPU pool this was developed on: profiles/r02_sanitizer.md.)
#ifdef GLH_CHECKED
#include <assert.h>
#define GLH_ASSERT(c) assert(c)
#define GLH_DELAY(k)                                                                                  \
    do {                                                                                              \
        const unsigned h_ = (blockIdx.x + 1u) * 2654435761u ^ (blockIdx.y + 7u) * 40503u ^ (unsigned)(k) * 977u; \
        const long long n_ = (long long)((h_ >> 9) % 30000u);                                         \
        const long long t0_ = clock64();                                                              \
        while (clock64() - t0_ < n_) { }                                                              \
    } while (0)
#else
#define GLH_ASSERT(c) do { } while (0)
#define GLH_DELAY(k) do { } while (0)
#endif

namespace glh {

namespace cg = cooperative_groups;

constexpr int HOT_NT = 512;           // threads per CTA
constexpr int HOT_NW = HOT_NT / 32;
constexpr int MAXEP = 8;              // transit epochs of one walker inside one series segment
constexpr int MAXC = 8;               // CTAs per cluster (portable limit)
constexpr int CAP = 2 * HOT_NT;       // (exposure, sub-exposure) pairs of the sparse mode

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

// ------------------------------------------------------------------------------------------
// Steps a3 + a4 for an outline that crosses the limb AT MOST TWICE (the caller has
// excluded the evolute regime for the whole walker): the arithmetic of glf::blocked_f32 without its
// generic branch, cut into the pieces the kernel schedules separately.
//   path_of       which rule the pair takes (0 = no overlap; 1, 2, 3 = 6 / 8 / 16 fixed nodes, outline
//                 wholly inside and >= 0.01 from the limb; 4 = near the limb)
//   cheap_delta   paths 1-3
//   near_delta    path 4, by one lane (TWO = false) or by two lanes that share it (TWO = true);
//                 both give the same bits: the one-lane version does the two lanes' parts in turn
//                 and adds them in the same order.
// delta = k0 A_flat + k1 A_lin + k2 A_quad (R8; eqs. 21-23).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int path_of(float r0sq, float a, float* r0_out) {
    const float reach = 1.f + a;
    const float r0 = r0sq * glf::mufu_rsqrt(fmaxf(r0sq, 1e-30f));
    *r0_out = r0;
    if (r0sq >= reach * reach) return 0;
    if (!(r0 + a <= 0.99f)) return 4;
    if (fmaf(4.f, a, r0) <= 1.f || r0 + a <= 0.5f) return 1;
    return (r0 + a + a <= 1.f || r0 + a <= 0.7f) ? 2 : 3;
}

// Part of the trapezoid sum of W(r^2) (2 f_flat) over the whole outline (glf::whole_outline_lin): the
// blocks of four node pairs number first, first + step, ... of the nh/4 blocks; NOT yet scaled by pi/nh.
__device__ __forceinline__ float outline_lin_part(const glf::TrapNode* trap, int nh, int first, int step,
                                                  float xc, float yc, float a, float b, float ab, float u,
                                                  float v) {
    const int stride = 16 / nh;
    float acc = 0.f;
    for (int blk = first; blk * 4 < nh; blk += step) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            const glf::TrapNode nd = trap[(blk * 4 + kk) * stride];
            const float p = a * nd.c, q = b * nd.s;
            const float xp = xc + p, yp = yc + q, xq = xc - p, yq = yc - q;
            const float m2p = fmaf(-xp, xp, fmaf(-yp, yp, 1.f));
            const float m2q = fmaf(-xq, xq, fmaf(-yq, yq, 1.f));
            const float w = fmaf(u, nd.c, v * nd.s);
            acc += glf::pair_term<true>(m2p, ab + w, m2q, ab - w);
        }
    }
    return acc;
}

// Outline wholly inside the disc: A_flat = pi a b, A_quad = pi a b (r0^2 + (a^2 + b^2)/4) in closed
// form, `lin` = the trapezoid sum of the f_lin weight, scaled.
__device__ __forceinline__ float inside_delta(float lin, float a, float b, float ab, float r0sq, float k0,
                                              float k1, float k2) {
    const float in_flat = glf::kPiF * ab;
    const float in_quad = in_flat * fmaf(0.25f, fmaf(a, a, b * b), r0sq);
    return fmaf(k0, in_flat, fmaf(k1 * (1.f / 3.f), lin, k2 * in_quad));
}

// xc, yc >= 0 (already folded).  path = 1, 2 or 3.
__device__ __forceinline__ float cheap_delta(const glf::TrapNode* trap, int path, float xc, float yc,
                                             float r0sq, float a, float b, float ab, float k0, float k1,
                                             float k2) {
    const float u = b * xc, v = a * yc;
    float lin;
    if (path == 1) {
        lin = glf::whole_outline_lin6(xc, yc, a, b, ab, u, v);
    } else {
        const int nh = path == 2 ? 4 : 8;
        lin = outline_lin_part(trap, nh, 0, 1, xc, yc, a, b, ab, u, v) * glf::pi_over_nodes(nh);
    }
    return inside_delta(lin, a, b, ab, r0sq, k0, k1, k2);
}

// glf::critical_point with the sign as an argument (sgn = +1: the maximum of g in the first quadrant,
// -1: the minimum in the third), so that two lanes can run the two searches in one instruction stream.
__device__ __forceinline__ void critical_point_rt(float xc, float yc, float a, float b, float sgn, float* c,
                                                  float* s) {
    for (int it = 0; it < 12; ++it) {
        const float x = fmaf(a, *c, xc), y = fmaf(b, *s, yc);
        const float bc = b * *c, as = a * *s;
        const float h = bc * y - as * x;
        const float hp = fmaf(bc, bc, as * as) - fmaf(b * *s, y, a * *c * x);
        float d = (sgn * hp < 0.f) ? -glf::fast_div(h, hp) : copysignf(0.5f, sgn * h);
        d = fminf(fmaxf(d, -0.5f), 0.5f);
        const float d2 = d * d;
        const float sd = d * fmaf(d2, fmaf(d2, 1.f / 120.f, -1.f / 6.f), 1.f);
        const float cd = fmaf(d2, fmaf(d2, fmaf(d2, -1.f / 720.f, 1.f / 24.f), -0.5f), 1.f);
        float cn = *c * cd - *s * sd, sn = *s * cd + *c * sd;
        cn = sgn * fmaxf(sgn * cn, 0.f);
        sn = sgn * fmaxf(sgn * sn, 0.f);
        const float rn = glf::mufu_rsqrt(fmaf(cn, cn, sn * sn));
        *c = cn * rn;
        *s = sn * rn;
        if (fabsf(d) < 1e-3f) break;
    }
}

template <bool TWO>
__device__ __forceinline__ float near_rest(const glf::TrapNode* trap, float xc, float yc, float r0sq, float a,
                                           float b, float ab, float e2, float k0, float k1, float k2, float cf,
                                           float sf, float cn, float sn, int h, unsigned mask);

// Path 4.  xc, yc >= 0.  TWO: lanes `lane` and `lane ^ 1` of the warp hold the SAME pair; h = lane & 1
// says which half this lane does (mask = the lanes that are in here together: whole lane pairs).
template <bool TWO>
__device__ __forceinline__ float near_delta(const glf::TrapNode* trap, float xc, float yc, float r0sq, float a,
                                            float b, float ab, float e2, float k0, float k1, float k2, int h,
                                            unsigned mask) {
    using namespace glf;
    // ---- critical points of g = x^2 + y^2 - 1 on the outline: the farthest point from the star centre
    // (first quadrant) and the nearest (third quadrant), both started from the direction (a xc, b yc)
    const float Aa = a * xc, Bb = b * yc;
    const float rn = mufu_rsqrt(fmaf(Aa, Aa, Bb * Bb));   // (r0 > 0.49 here: not both zero)
    const float c0 = Aa * rn, s0 = Bb * rn;
    float cf, sf, cn, sn;
    if (TWO) {
        const float sg = h ? -1.f : 1.f;
        float c = sg * c0, s = sg * s0;
        critical_point_rt(xc, yc, a, b, sg, &c, &s);
        const float co = __shfl_xor_sync(mask, c, 1), so = __shfl_xor_sync(mask, s, 1);
        cf = h ? co : c;
        sf = h ? so : s;
        cn = h ? c : co;
        sn = h ? s : so;
    } else {
        cf = c0;
        sf = s0;
        critical_point_rt(xc, yc, a, b, 1.f, &cf, &sf);
        cn = -c0;
        sn = -s0;
    }
    return near_rest<TWO>(trap, xc, yc, r0sq, a, b, ab, e2, k0, k1, k2, cf, sf, cn, sn, h, mask);
}

// The rest of path 4 once the farthest point (cf, sf) is known; (cn, sn) = the nearest point (TWO) or
// the starting direction of its search (one lane: it is searched here, only if needed).
template <bool TWO>
__device__ __forceinline__ float near_rest(const glf::TrapNode* trap, float xc, float yc, float r0sq, float a,
                                           float b, float ab, float e2, float k0, float k1, float k2, float cf,
                                           float sf, float cn, float sn, int h, unsigned mask) {
    using namespace glf;
    const float u = b * xc, v = a * yc;
    const float xf = fmaf(a, cf, xc), yf = fmaf(b, sf, yc);
    const float gfar = fmaf(xf, xf, fmaf(yf, yf, -1.f));
    if (gfar <= 0.f) {
        // wholly inside, close to the limb: 16 nodes, 32 within 0.02 of it; the two halves of the
        // node blocks are summed separately (lane 0 / lane 1) and added
        const int nh = (gfar < -0.04f) ? 8 : 16;
        float p0, p1;
        if (TWO) {
            const float mine = outline_lin_part(trap, nh, h, 2, xc, yc, a, b, ab, u, v);
            const float other = __shfl_xor_sync(mask, mine, 1);
            p0 = h ? other : mine;
            p1 = h ? mine : other;
        } else {
            p0 = outline_lin_part(trap, nh, 0, 2, xc, yc, a, b, ab, u, v);
            p1 = outline_lin_part(trap, nh, 1, 2, xc, yc, a, b, ab, u, v);
        }
        return inside_delta((p0 + p1) * glf::pi_over_nodes(nh), a, b, ab, r0sq, k0, k1, k2);
    }
    // ---- the outline crosses the limb twice (or misses the disc).  tau = t - t_far in [0, 2 pi).
    Arc o = {xc, yc, a, b, cf, sf};
    float tsplit = kPiF;
    const float xo = fmaf(-a, cf, xc), yo = fmaf(-b, sf, yc);   // the point opposite t_far
    float gsplit = fmaf(xo, xo, fmaf(yo, yo, -1.f));
    if (gsplit >= 0.f) {
        // mostly outside: the nearest outline point and its tau
        if (!TWO) critical_point_rt(xc, yc, a, b, -1.f, &cn, &sn);
        const float xn = fmaf(a, cn, xc), yn = fmaf(b, sn, yc);
        gsplit = fmaf(xn, xn, fmaf(yn, yn, -1.f));
        if (gsplit >= 0.f) return 0.f;
        const float dtau = atan2_fast(cf * sn - sf * cn, cf * cn + sf * sn);
        tsplit = dtau < 0.f ? dtau + kTwoPiF : dtau;
    }
    // half-cosine model of g between its maximum and the split point (exact for a circle)
    const float mid = 0.5f * (gfar + gsplit), amp = 0.5f * (gfar - gsplit);
    const float uu = rough_acos(fminf(fmaxf(-fast_div(mid, amp), -1.f), 1.f)) * (1.f / kPiF);
    float t1, s1, c1, t2, s2, c2;
    if (TWO) {
        float s, c;   // ONE call, the lane's half chosen by its arguments: the two lanes stay in step
        const float t = crossing(o, h ? tsplit : 0.f, h ? kTwoPiF : tsplit,
                                 h ? kTwoPiF - uu * (kTwoPiF - tsplit) : uu * tsplit, h != 0, &s, &c);
        const float to = __shfl_xor_sync(mask, t, 1), so = __shfl_xor_sync(mask, s, 1),
                    co = __shfl_xor_sync(mask, c, 1);
        t1 = h ? to : t;
        s1 = h ? so : s;
        c1 = h ? co : c;
        t2 = h ? t : to;
        s2 = h ? s : so;
        c2 = h ? c : co;
    } else {
        t1 = crossing(o, 0.f, tsplit, uu * tsplit, false, &s1, &c1);
        t2 = crossing(o, tsplit, kTwoPiF, kTwoPiF - uu * (kTwoPiF - tsplit), true, &s2, &c2);
    }
    // ---- outline arc [t1, t2] (inside the disc): flat and quad in closed form
    glc::Outline<float> oo = {xc, yc, a, b, e2};
    const glc::ArcCoef<float> k = glc::arc_coefficients(oo);
    const float dt = t2 - t1;
    float f1, q1, f2, q2;
    glc::arc_primitive(k, s1, c1, &f1, &q1);
    glc::arc_primitive(k, s2, c2, &f2, &q2);
    float Aflat = 0.5f * fmaf(k.ab, dt, f2 - f1);
    float Aquad = 0.25f * fmaf(k.k0, dt, q2 - q1);
    // ---- f_lin: 16-point Gauss-Legendre in z, t = tm + hw (3z - z^3)/2; even node pairs (lane 0) and
    // odd ones (lane 1) summed separately, then added
    const float hw = 0.5f * dt;
    float sm, cm;
    abs_trig(o, t1 + hw, &sm, &cm);
    constexpr float gl_phi[8] = GLH_GL_PHI, gl_om[8] = GLH_GL_OM;
    auto node = [&](float phi, float om, float acc) {
        const float dd = hw * phi;   // in [0, pi]
        const float sd = mufu_sin(dd), cd = mufu_cos(dd);
        const float cp = cm * cd - sm * sd, sp = sm * cd + cm * sd;
        const float cq = cm * cd + sm * sd, sq = sm * cd - cm * sd;
        const float xp = fmaf(a, cp, xc), yp = fmaf(b, sp, yc);
        const float xq = fmaf(a, cq, xc), yq = fmaf(b, sq, yc);
        const float m2p = fmaf(-xp, xp, fmaf(-yp, yp, 1.f));
        const float m2q = fmaf(-xq, xq, fmaf(-yq, yq, 1.f));
        const float fp = fmaf(u, cp, fmaf(v, sp, ab)), fq = fmaf(u, cq, fmaf(v, sq, ab));
        return fmaf(om, pair_term<true>(m2p, fp, m2q, fq), acc);
    };
    float part[2] = {0.f, 0.f};
    if (TWO) {
        float mine = 0.f;
#pragma unroll
        for (int ii = 0; ii < 4; ++ii)   // node pair 2 ii + h: the two lanes differ in constants only
            mine = node(h ? gl_phi[2 * ii + 1] : gl_phi[2 * ii], h ? gl_om[2 * ii + 1] : gl_om[2 * ii], mine);
        const float other = __shfl_xor_sync(mask, mine, 1);
        part[0] = h ? other : mine;
        part[1] = h ? mine : other;
    } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) part[i & 1] = node(gl_phi[i], gl_om[i], part[i & 1]);
    }
    float Alin = (1.f / 3.f) * hw * (part[0] + part[1]);
    // ---- limb arc from the exit point (t2) counter-clockwise back to the entry point (t1)
    const float xa = fmaf(a, c2, xc), ya = fmaf(b, s2, yc);
    const float xb = fmaf(a, c1, xc), yb = fmaf(b, s1, yc);
    const float dl = atan2_fast(xa * yb - ya * xb, xa * xb + ya * yb);
    Aflat = fmaf(0.5f, dl, Aflat);
    Alin = fmaf(1.f / 3.f, dl, Alin);
    Aquad = fmaf(0.25f, dl, Aquad);
    return fmaf(k0, Aflat, fmaf(k1, Alin, k2 * Aquad));
}

// One lane, any path: the dense mode's per-sub-exposure call.  xc_in, yc_in of any sign.
__device__ __forceinline__ float blocked_hot(const glf::TrapNode* trap, float xc_in, float yc_in, float a,
                                             float b, float ab, float e2, float k0, float k1, float k2) {
    const float xc = fabsf(xc_in), yc = fabsf(yc_in);   // mirror images have the same areas
    const float r0sq = fmaf(xc, xc, yc * yc);
    float r0;
    const int path = path_of(r0sq, a, &r0);
    if (path == 0) return 0.f;
    if (path < 4) return cheap_delta(trap, path, xc, yc, r0sq, a, b, ab, k0, k1, k2);
    return near_delta<false>(trap, xc, yc, r0sq, a, b, ab, e2, k0, k1, k2, 0, 0xffffffffu);
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
    double S;               // PRE: baseline sum_i ((obs_i - 1)/sigma_i)^2
    double t_exp;
    float inv_ss, doff, off0;   // 1/n_ss, t_exp/n_ss, (0.5/n_ss - 0.5) t_exp: sub-exposure j sits at off0 + j doff (R18)
    unsigned ss_magic;      // ceil(2^32 / n_ss): pair / n_ss = umulhi(pair, ss_magic) for pair < 2^16 (n_ss > 1)
    int B, T, n_ss, nseg, seglen;   // B * nseg < 2^31
    int sorted_known;       // the caller vouches that times is non-decreasing (gl_series checked it)
    int* done_count;        // nullptr, or a zeroed device word: the CTAs count themselves out here ...
    int* done_flag;         // ... and the last one sets this word (pinned host memory) to 1: the host call's
                            // completion signal (gl_series_loglike spins on it instead of synchronising the stream)
};

enum { CLS_SIMPLE = 0, CLS_INVALID = 1, CLS_DEFER = 2 };
constexpr int MAXDEFER_WORDS = 1025;   // one bit per unit of a CTA: B * nseg < 2^31 over >= 65535 grid rows

struct Unit {
    // written by the four prelude threads
    double t0, P, x1, x2, hx;     // x1, x2 = (t_first - t0)/P, (t_last - t0)/P; hx = t_exp/(2P) + 1e-9
    float phimax;                 // half-angle of the window [rad], widened
    float w, aR, bimp, a, b, cpsi, spsi, k0, k1, k2;
    int cls_win, defer_shape, bad_ld, bad_period, never;
    // written by the search warps
    double tc[MAXEP];             // conjunction time of each transit epoch that touches the segment
    int lo[MAXEP], hi[MAXEP];     // its in-window index range [lo, hi) (relative to the segment)
};

// Prelude, thread 1 of 4: validity (the limb-darkening norm is checked by hot_prelude_ld) and the
// half-angle of the transit window.  fin = every entry of the row is finite (voted by the warp).
// PAPER.md:85-87 eqs. 9-10: the centre is within `reach` of the star centre iff
// sin^2(phi) < [(reach/aR)^2 - cos^2 i] / sin^2 i (and cos(phi) > 0).
// e != 0 (or NaN) is deferred whatever else the row holds: the full kernel owns those rules.
__device__ __forceinline__ void hot_prelude_window(const double* p, bool fin, Unit* u) {
    const double P = p[1], aR = p[2], b = p[3], e = p[4], Rp = p[6], f = p[7];
    const bool ok = fin & (P > 0.0) & (Rp > 0.0) & (Rp < 0.5) & (f >= 0.0) & (f < 1.0) & (aR > 1.0) &
                    (fabs(b) <= aR);
    const float aRf = (float)aR, bf = (float)b;
    const float iaR = rcp_nr(aRf);
    const float cosi = bf * iaR, ci2 = cosi * cosi;
    const float reach = (1.f + (float)Rp) * (1.f + 1e-5f);
    const float q = reach * iaR;
    const float S2 = glf::fast_div(q * q - ci2, 1.f - ci2);
    u->phimax = asin_small(glf::mufu_sqrt(fminf(fmaxf(S2, 0.f), 0.25f)) * (1.f + 1e-6f)) * (1.f + 1e-5f);
    u->aR = aRf;
    u->bimp = bf;
    const bool never = (S2 <= 0.f);   // no transit at all
    u->never = never;
    // S2 > 1/4 is a long window (a NaN S2 -- face-on orbit grazing the reach -- fails both tests): deferred
    u->cls_win = !(e == 0.0) ? CLS_DEFER : (!ok ? CLS_INVALID : ((never | (S2 <= 0.25f)) ? CLS_SIMPLE : CLS_DEFER));
}

// Thread 2 of 4: the oblate spheroid's projected outline in closed form -- semi-major axis Rp along
// (sin xi, cos xi), semi-minor Rp sqrt(1 - f(2-f) cos^2 eta) (eqs. 6, 11-13 with a = Rp(1-f),
// b = c = Rp, zeta = 0: SURVEY.md 8(c) "equation checks"; the parity tests compare with the general
// eigen-axes of the full kernel) -- and the evolute exclusion: a second pair of critical points of g
// needs a xc < e2 and b yc < e2 (gl_core.cuh), i.e. r0 < e2 sqrt(1/a^2 + 1/b^2); if that is below
// 0.99 - a, the near-limb path (r0 + a > 0.99) can never see one.
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

// Thread 3 of 4: c0, c1, c2 of R8 over pi (1 - u1/3 - u2/6), and that norm's sign.
__device__ __forceinline__ void hot_prelude_ld(const double* p, Unit* u) {
    const double u1 = p[10], u2 = p[11];
    const double norm = 1.0 - u1 / 3.0 - u2 / 6.0;
    const float ipn = rcp_nr((float)(3.14159265358979323846 * norm));
    u->k0 = (float)(1.0 - u1 - 2.0 * u2) * ipn;
    u->k1 = (float)(u1 + 2.0 * u2) * ipn;
    u->k2 = (float)u2 * ipn;
    u->bad_ld = !(norm > 0.0);
}

// Thread 4 of 4: 1/P in fp64 by Newton from the MUFU reciprocal (P must be in fp32's range for that),
// the angular velocity, and the segment's ends in units of the period.
__device__ __forceinline__ void hot_prelude_period(const double* p, double t_exp, double tfirst, double tlast,
                                                   Unit* u) {
    const double t0 = p[0], P = p[1];
    double inv_P = (double)glf::mufu_rcp((float)P);
    inv_P = inv_P * fma(-P, inv_P, 2.0);
    inv_P = inv_P * fma(-P, inv_P, 2.0);
    u->t0 = t0;
    u->P = P;
    u->w = (float)(6.28318530717958647692 * inv_P);
    u->x1 = (tfirst - t0) * inv_P;
    u->x2 = (tlast - t0) * inv_P;
    u->hx = 0.5 * t_exp * inv_P + 1e-9;
    u->bad_period = !((P > 1e-30) & (P < 1e30));
}

// #{i in [0, n) : seg[i] < q} for a non-decreasing segment, by ONE WARP (every lane calls this with
// the same arguments and gets the same answer).  coarse[k] = seg[k stride] for k stride < n, +inf
// beyond, HOT_NT = 512 entries: two 32-way steps (16 entries apart, then 1 apart) find how many
// coarse samples lie below q, one round of global loads (stride - 1 candidates) does the rest.  On a
// segment that is NOT sorted the answer is meaningless but still in [0, n].
__device__ __forceinline__ int lower_bound_warp(const double* __restrict__ seg, int n, const double* coarse,
                                                int stride, double q, int lane) {
    const int j1 = __popc(__ballot_sync(0xffffffffu, coarse[lane * 16] < q));
    if (j1 == 0) return 0;   // warp-uniform
    const int blk = (j1 - 1) * 16;
    const int j2 = __popc(__ballot_sync(0xffffffffu, lane < 16 && coarse[blk + (lane & 15)] < q));
    const int lo = blk + max(j2, 1);                  // coarse samples below q (>= 1)
    const int base = (lo - 1) * stride, end = min(lo * stride, n);
    int cnt = 0;
    for (int m0 = base + 1; m0 < end; m0 += 32) {      // warp-uniform trip count
        const int m = m0 + lane;
        GLH_ASSERT(m0 >= 0 && end <= n);
        cnt += __popc(__ballot_sync(0xffffffffu, m < end && seg[m] < q));
    }
    return min(base + 1 + cnt, n);
}

// A walker off the common path (eccentric orbit, long window, many transit epochs, evolute regime,
// unsorted series): the CTA (or cluster) does the unit with the full-featured arithmetic of
// greenlantern_b200.cu -- fp64 phase of every exposure, Kepler, generic crossing search -- one exposure
// per lane and pass.  Defined in greenlantern_b200.cu (it needs that file's Walker machinery) and inlined
// into hot_kernel's SECOND loop.  (As a real call -- __noinline__, in either loop -- it cost the common path
// 2 us of 16 on config 3 and 4 of 86 on config 4: the call ABI changes the register allocation of the whole
// kernel.)  Returns CLS_INVALID for an invalid walker (its flux row is NaN-filled), else CLS_SIMPLE with the
// thread's chi^2 terms added to *acc.
__device__ __forceinline__ int generic_unit(const HotArgs& A, bool pre, int wk, int t_lo, int nT, int gtid, int ntot,
                                            const glf::TrapNode* trap, double* acc, float* s_d, int* s_li,
                                            int* s_cnt);   // (s_d[CAP], s_li[CAP], s_cnt[HOT_NW]: the kernel's)

template <bool PRE>
__global__ void __launch_bounds__(HOT_NT, 2) hot_kernel(const HotArgs A) {
    asm volatile("griddepcontrol.launch_dependents;");   // a dependent launch (the GP scan) may become resident
    GLH_TL(15);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int csize = (int)gridDim.x, crank = (int)blockIdx.x;
    cg::cluster_group cluster = cg::this_cluster();

    __shared__ Unit su;
    __shared__ double s_row[4][12];
    __shared__ double s_coarse[HOT_NT];    // every stride-th time of the segment (+inf beyond its end)
    __shared__ double s_red[HOT_NW];
    __shared__ double s_gather[2][MAXC];   // rank 0's copy collects the cluster's chi^2 partials
    __shared__ int s_cnt[2][HOT_NW];       // near-limb pairs per (pair slot, warp)
    __shared__ float s_px[CAP], s_py[CAP]; // sparse mode: folded kernel-frame centre of a near-limb pair
    __shared__ float s_d[CAP];             // ... blocked fraction of every pair
    __shared__ unsigned short s_np[CAP];   // ... the near-limb pairs, in pair order
    __shared__ int s_li[CAP];              // ... index in the segment of in-window exposure e
    __shared__ float2 s_ow[CAP];           // ... its (obs - 1, 1/sigma)
    __shared__ glf::TrapNode s_trap[16];

    const int S = A.n_ss;
    const float inv_ss = A.inv_ss, doff = A.doff, off0 = A.off0;
    const bool want_chi2 = A.chi2 != nullptr, want_flux = A.flux != nullptr;
    const int ntot = csize * HOT_NT, gtid = crank * HOT_NT + tid;
    const unsigned lt_mask = (1u << lane) - 1u;
    int wpar = 0;
    // no CTA may write into rank 0's shared memory before rank 0 runs: arrive now, wait before the
    // first push
    bool started = (csize == 1);
    if (csize > 1) cluster.barrier_arrive();

    // chi^2 of one unit.  Every step below is a fixed tree or a fixed loop: the same bits in every run of a
    // launch shape.  The thread's terms (fp64 accumulator of fp32 terms) are narrowed and summed over the warp
    // in fp32 (5 shuffles; each term carries fp32 rounding already), the <= 16 warp sums go through shared
    // memory to warp 0, which adds them in fp64 by a shuffle tree; lane 0 adds the series' baseline S and
    // writes chi^2 -- or, in a cluster, pushes the CTA's sum into rank 0's shared memory, and rank 0 adds
    // the sums in rank order behind ONE cluster barrier.  A single thread walking the partials (round 1, and
    // this kernel before) took 1.3 us of config 3's 8 us: dependent shared-memory / fp64 round trips cost
    // 60-100 cycles each when nothing else runs.
    // nwsum: only the first nwsum warps can hold non-zero terms (sparse mode: the threads that formed the
    // exposure means); the others are neither reduced nor read.
    auto chi2_unit = [&](double acc, int cls, int wk, int nwsum) {
        if (warp < nwsum) {
            float part = (float)acc;
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) part += __shfl_down_sync(0xffffffffu, part, off);
            if (lane == 0) s_red[warp] = (double)part;
        }
        GLH_TL(8);
        GLH_DELAY(1);
        if (!started) {
            cluster.barrier_wait();
            started = true;
        }
        __syncthreads();
        GLH_TL(9);
        double tot = 0.0;
        if (warp == 0) {
            tot = lane < nwsum ? s_red[lane] : 0.0;
#pragma unroll
            for (int off = HOT_NW / 2; off > 0; off >>= 1)
                if (nwsum > off) tot += __shfl_down_sync(0xffffffffu, tot, off);   // (nwsum is CTA-uniform)
            GLH_DELAY(2);
            if (csize > 1 && lane == 0) *cluster.map_shared_rank(&s_gather[wpar][crank], 0) = tot;
        }
        GLH_TL(10);
        GLH_DELAY(3);
        if (csize > 1) cluster.sync();
        GLH_DELAY(4);
        if (crank == 0 && tid == 0) {
            double d2 = tot;
            if (csize > 1) {
                d2 = 0.0;
                for (int r = 0; r < csize; ++r) d2 += s_gather[wpar][r];
            }
            // raw series: baseline_kernel, launched before this grid (which may have started early:
            // programmatic dependent launch), writes S into chi2[0..B): wait before touching chi2
            if (!PRE) asm volatile("griddepcontrol.wait;" ::: "memory");
            float out;
            if (cls == CLS_INVALID) {
                out = __int_as_float(0x7f800000);
            } else {
                double Sb = A.S;
                if (!PRE) Sb = (double)*(volatile float*)&A.chi2[wk];
                out = (Sb > 1.79769313486231570e308) ? (float)Sb : (float)(Sb + d2);
            }
            A.chi2[wk] = out;
        }
        GLH_TL(5);
        wpar ^= 1;
    };

    // Units off the common path are only NOTED in the main loop (one bit per unit of this CTA) and done in
    // a second loop behind it, so that the main loop holds the common path's code and nothing else.
    __shared__ unsigned s_defer[MAXDEFER_WORDS];
    const unsigned nunits = (unsigned)A.B * (unsigned)A.nseg;
    {
        // (one unit per CTA row unless the batch exceeds the grid: no division then)
        const unsigned mine = blockIdx.y >= nunits ? 0u
                              : (nunits <= gridDim.y ? 1u : (nunits - blockIdx.y + gridDim.y - 1) / gridDim.y);
        GLH_ASSERT((mine + 31) / 32 <= MAXDEFER_WORDS);
        for (unsigned i = tid; i < (mine + 31) / 32; i += HOT_NT) s_defer[i] = 0u;   // (barrier: top of the loop)
    }
    bool any_defer = false;
    unsigned kun = 0;
    for (unsigned un = blockIdx.y; un < nunits; un += gridDim.y, ++kun) {
        const int wk = A.nseg == 1 ? (int)un : (int)(un / (unsigned)A.nseg);
        const int t_lo = (int)(un - (unsigned)wk * (unsigned)A.nseg) * A.seglen;
        const double* __restrict__ seg = A.times + t_lo;
        const int nT = min(A.seglen, A.T - t_lo);
        const double* __restrict__ p = A.params + (size_t)wk * 12;
        float* frow = want_flux ? A.flux + (size_t)wk * A.T + t_lo : nullptr;
        const int stride = (nT + HOT_NT - 1) / HOT_NT;   // coarse table: every stride-th time

        __syncthreads();   // the previous unit's shared data is dead
        GLH_TL(0);
        // ---- 1. coarse samples of the series; order check (this CTA's share of the adjacent pairs,
        // incl. the pair that straddles into the next segment) unless the caller vouches for the order;
        // prelude on four threads of four warps.  The parameter row is ONE coalesced 96-byte request
        // per prelude warp (it may sit in host memory read over PCIe: gl_series_loglike).
        {
            const long long ci = (long long)tid * stride;
            GLH_ASSERT(ci >= 0 && (ci < nT || ci >= nT));
            s_coarse[tid] = ci < nT ? seg[ci] : __longlong_as_double(0x7ff0000000000000LL);
        }
        // the node table of the fixed-angle rules, from constant memory: filled HERE by the last warp, behind
        // the first loads of the unit, and not in front of the kernel's first barrier -- after an L2 flush the
        // constant-cache miss sat on the entry path of every CTA (entry to first unit: 2.0 us flushed, 1.1 warm)
        if (kun == 0 && tid >= HOT_NT - 16) {
            const int k = tid - (HOT_NT - 16);
            s_trap[k] = glf::TrapNode{c_trap16[k].x, c_trap16[k].y};
        }
        int unsorted = 0;
        if (!A.sorted_known) {   // (every CTA of a cluster looks at ALL pairs: the verdict must be the cluster's)
            const int npairs = min(nT, A.T - t_lo - 1);
            for (int i = tid; i < npairs; i += HOT_NT) unsorted |= !(seg[i] <= seg[i + 1]);
        }
        if (warp < 4) {
            const double v = lane < 12 ? p[lane] : 0.0;
            if (lane < 12) s_row[warp][lane] = v;
            const bool fin = __all_sync(0xffffffffu, fabs(v) <= 1.79769313486231570e308);
            __syncwarp();
            if (tid == 0) hot_prelude_window(s_row[0], fin, &su);
            if (tid == 32) hot_prelude_shape(s_row[1], &su);
            if (tid == 64) hot_prelude_ld(s_row[2], &su);
            if (tid == 96) hot_prelude_period(s_row[3], A.t_exp, seg[0], seg[nT - 1], &su);
        }
        unsorted = __syncthreads_or(unsorted);
        GLH_TL(1);
        // every thread: the transit epochs n whose window [t0 + n P - hw, t0 + n P + hw) can touch the
        // segment (hw = half-width of the window in time, hwp in units of the period), and the verdict
        const double P = su.P, t0 = su.t0;
        const double hwp = (double)su.phimax * 0.15915494309189535 + su.hx;
        const double nlo = ceil(su.x1 - hwp - 1e-9);
        const double cnt = floor(su.x2 + hwp + 1e-9) - nlo + 1.0;
        const bool few = (cnt <= (double)MAXEP);   // false for NaN / infinite time stamps too
        int cls = su.cls_win;
        if (cls != CLS_DEFER && su.bad_ld) cls = CLS_INVALID;
        if (cls == CLS_SIMPLE && !su.never &&
            (su.bad_period || su.defer_shape || !few || !(su.phimax + su.w * (float)A.t_exp <= 0.8f)))
            cls = CLS_DEFER;   // (0.8 rad: small_sincos's range)
        if (cls == CLS_SIMPLE && unsorted) cls = CLS_DEFER;
        const int nep = (cls == CLS_SIMPLE && !su.never && cnt > 0.0) ? (int)cnt : 0;

        // ---- 2. for a sorted series the in-window exposures of an epoch are ONE index range: warp
        // 2 k finds where epoch k's window starts, warp 2 k + 1 where it ends
        if (warp < 2 * nep) {
            const double tc = fma(nlo + (double)(warp >> 1), P, t0);
            const double q = (warp & 1) ? tc + hwp * P : tc - hwp * P;
            const int idx = lower_bound_warp(seg, nT, s_coarse, stride, q, lane);
            if (lane == 0) {
                if (warp & 1) {
                    su.hi[warp >> 1] = idx;
                } else {
                    su.lo[warp >> 1] = idx;
                    su.tc[warp >> 1] = tc;
                }
            }
        }
        __syncthreads();
        GLH_TL(2);

        double acc = 0.0;   // this thread's chi^2 terms
        int nwsum = HOT_NW;   // ... and the warps that can hold any
        bool chi2_done = false;
        if (cls == CLS_DEFER) {   // (CTA-uniform, and the same in every CTA of a cluster)
            if (tid == 0) s_defer[kun >> 5] |= 1u << (kun & 31u);
            any_defer = true;
            continue;
        }
        if (cls == CLS_INVALID) {
            if (frow)
                for (int i = gtid; i < nT; i += ntot) frow[i] = __int_as_float(0x7fc00000);
        } else {
            const float w = su.w, aR = su.aR, bimp = su.bimp, a = su.a, b = su.b;
            const float cpsi = su.cpsi, spsi = su.spsi, k0 = su.k0, k1 = su.k1, k2 = su.k2;
            const float ab = a * b, e2 = (a - b) * (a + b);
            // the ranges are read from shared memory where they are needed (broadcast reads; nep is 1
            // for a single-transit series): len_k = max(hi_k - lo_k, 0) -- an unsorted share of the
            // series may give anything: such a unit was classified CLS_DEFER above and never gets here
            int M = 0;   // in-window exposures of the unit (the whole cluster's)
#pragma unroll 1
            for (int k = 0; k < nep; ++k) M += max(su.hi[k] - su.lo[k], 0);   // (nep is 1 for a single-transit series)
            // v-th in-window exposure of the unit -> its index in the segment and its time from the
            // centre of its transit, (float)(t - t_c): the fp64 phase reduction is gone
            auto entry = [&](int v, int* idx) {
                int n = 0, run = 0, i = su.lo[0] + v;
#pragma unroll 1
                for (int k = 1; k < nep; ++k) {
                    run += max(su.hi[k - 1] - su.lo[k - 1], 0);
                    if (v >= run) {
                        n = k;
                        i = su.lo[k] + (v - run);
                    }
                }
                GLH_ASSERT(i >= 0 && i < nT && n >= 0 && n < MAXEP);
                *idx = i;
                return (float)(seg[i] - su.tc[n]);
            };
            // folded kernel-frame position of sub-exposure j of an exposure (eqs. 9-10
            // with d sin(beta) = b; phi = 2 pi dt / P, |phi| <= 0.8)
            auto position = [&](float dtc, int j, float* xc, float* yc) {
                float s, c;
                small_sincos(w * (dtc + fmaf((float)j, doff, off0)), &s, &c);
                const float x0 = bimp * c, y0 = aR * s;
                *xc = fabsf(fmaf(cpsi, x0, spsi * y0));
                *yc = fabsf(fmaf(cpsi, y0, -spsi * x0));
            };
            auto obs_of = [&](int i) {   // (obs - 1, 1/sigma) of exposure i in fp32
                if (PRE) return A.ow[t_lo + i];
                const float sf = (float)A.sigma[t_lo + i];
                float rs = glf::mufu_rcp(sf);
                rs = rs * fmaf(-sf, rs, 2.f);
                return make_float2((float)(A.obs[t_lo + i] - 1.0), rs);
            };
            auto finish = [&](int i, float dbar, float2 o2) {   // exposure i is done: flux, chi^2 term
                GLH_ASSERT(i >= 0 && i < nT);
                if (frow) frow[i] = 1.f - dbar;
                const float d = dbar * o2.y;
                acc += (double)(d * fmaf(2.f * o2.x, o2.y, d));   // ((o + dbar) r)^2 - (o r)^2
            };
            // out-of-window exposures: flux = 1, 16 bytes at a time where the row allows; thread ft of nft
            auto fill = [&](int ft, int nft) {
                auto inwin = [&](int i) {
                    bool in = false;
#pragma unroll 1
                    for (int k = 0; k < nep; ++k) in = in || (i >= su.lo[k] && i < su.hi[k]);
                    return in;
                };
                const int head = (int)((4u - (((uintptr_t)frow >> 2) & 3u)) & 3u);
                if (ft < head && ft < nT && !inwin(ft)) frow[ft] = 1.f;
                const int nchunk = nT > head ? (nT - head) >> 2 : 0;
                // (one transit in the series is the common case: its range sits in registers, not in a loop
                // over shared memory per 16-byte chunk)
                const int lo0 = nep > 0 ? su.lo[0] : 0, hi0 = nep > 0 ? su.hi[0] : 0;
                for (int c = ft; c < nchunk; c += nft) {
                    const int i0 = head + 4 * c;
                    bool hit = (i0 + 3 >= lo0 && i0 < hi0);
#pragma unroll 1
                    for (int k = 1; k < nep; ++k) hit = hit || (i0 + 3 >= su.lo[k] && i0 < su.hi[k]);
                    if (!hit) {
                        GLH_ASSERT(i0 >= 0 && i0 + 3 < nT && (((uintptr_t)(frow + i0)) & 15u) == 0);
                        *reinterpret_cast<float4*>(frow + i0) = make_float4(1.f, 1.f, 1.f, 1.f);
                    } else {
#pragma unroll 1
                        for (int r = 0; r < 4; ++r)
                            if (!inwin(i0 + r)) frow[i0 + r] = 1.f;
                    }
                }
                const int tail0 = head + 4 * nchunk;
                if (ft < nT - tail0 && !inwin(tail0 + ft)) frow[tail0 + ft] = 1.f;
            };
            const long long pairs = (long long)M * S;
            if (csize == 1 && pairs <= CAP) {
                // ---- 3a. SPARSE list: lane = (exposure, sub-exposure) pair, in time order.  Pairs on the
                // short paths (outline wholly inside the disc, away from the limb) are finished at once;
                // the near-limb ones are listed (deterministic order: pair slot, warp, lane).
                const int np = (int)pairs;
                int rank0 = -1, rank1 = -1;
#pragma unroll
                for (int sl = 0; sl < 2; ++sl) {   // (unrolled: the two slots' loads and chains overlap)
                    const int pr = tid + sl * HOT_NT;
                    bool near = false;
                    if (pr < np) {
                        const int e = S == 1 ? pr : (int)__umulhi((unsigned)pr, A.ss_magic);
                        const int j = pr - e * S;
                        int i;
                        const float dtc = entry(e, &i);
                        GLH_ASSERT(e >= 0 && e < M && e < CAP && j >= 0 && j < S);
                        if (j == 0) {
                            s_li[e] = i;
                            if (want_chi2) s_ow[e] = obs_of(i);
                        }
                        float xc, yc, r0;
                        position(dtc, j, &xc, &yc);
                        const float r0sq = fmaf(xc, xc, yc * yc);
                        const int path = path_of(r0sq, a, &r0);
                        near = (path == 4);
                        if (near) {
                            s_px[pr] = xc;
                            s_py[pr] = yc;
                        } else {
                            s_d[pr] = path == 0 ? 0.f : cheap_delta(s_trap, path, xc, yc, r0sq, a, b, ab, k0, k1, k2);
                        }
                    }
                    const unsigned bal = __ballot_sync(0xffffffffu, near);
                    if (lane == 0) s_cnt[sl][warp] = __popc(bal);
                    const int rk = near ? __popc(bal & lt_mask) : -1;
                    if (sl == 0) rank0 = rk; else rank1 = rk;
                }
                __syncthreads();
                // position of (slot, warp) in the list: scan of the 32 counts by every warp for itself
                int L;
                {
                    const int c = s_cnt[lane >> 4][lane & 15];
                    int incl = c;
#pragma unroll
                    for (int off = 1; off < 32; off <<= 1) {
                        const int v = __shfl_up_sync(0xffffffffu, incl, off);
                        if (lane >= off) incl += v;
                    }
                    L = __shfl_sync(0xffffffffu, incl, 31);
                    const int b0 = __shfl_sync(0xffffffffu, incl - c, warp);
                    const int b1 = __shfl_sync(0xffffffffu, incl - c, 16 + warp);
                    GLH_ASSERT(L <= np && L <= CAP && (rank0 < 0 || b0 + rank0 < L) && (rank1 < 0 || b1 + rank1 < L));
                    if (rank0 >= 0) s_np[b0 + rank0] = (unsigned short)tid;
                    if (rank1 >= 0) s_np[b1 + rank1] = (unsigned short)(tid + HOT_NT);
                }
                __syncthreads();
                GLH_TL(3);
                // ---- near-limb pairs: TWO lanes each (16 pairs per warp); the warps that have none fill
                // the out-of-window part of the flux row meanwhile
                const int nearwarps = min((L + 15) >> 4, HOT_NW);
                if (frow && warp >= nearwarps) fill(tid - nearwarps * 32, (HOT_NW - nearwarps) * 32);
                for (int q0 = 0; q0 < L; q0 += HOT_NT / 2) {
                    const int q = q0 + (tid >> 1);
                    if (q < L) {
                        const int pr = s_np[q];
                        GLH_ASSERT(pr >= 0 && pr < np);
                        const float xc = s_px[pr], yc = s_py[pr];
                        const float d = near_delta<true>(s_trap, xc, yc, fmaf(xc, xc, yc * yc), a, b, ab, e2, k0,
                                                         k1, k2, lane & 1, 3u << (lane & 30));
                        if ((lane & 1) == 0) s_d[pr] = d;
                    }
                }
                if (frow && nearwarps == HOT_NW) fill(tid, HOT_NT);
                __syncthreads();
                GLH_TL(6);
                // exposure means, in sub-exposure order (R18)
                nwsum = min((M + 31) >> 5, HOT_NW);
                for (int e = tid; e < M; e += HOT_NT) {
                    GLH_ASSERT(e * S + S <= CAP);
                    float sum = 0.f;
#pragma unroll 4
                    for (int j = 0; j < S; ++j) sum += s_d[e * S + j];
                    finish(s_li[e], sum * inv_ss, want_chi2 ? s_ow[e] : make_float2(0.f, 0.f));
                }
                GLH_TL(7);
                // (the reduction is issued from inside this branch: hanging it behind the if / else ladder
                // measured 0.2 us slower on config 3 -- code placement)
                if (want_chi2) {
                    chi2_unit(acc, cls, wk, nwsum);
                    chi2_done = true;
                }
            } else {
                // ---- 3b. DENSE list (a JWST-shaped series): thread v takes the v-th, (v + ntot)-th, ...
                // in-window exposure, all its sub-exposures in turn; neighbouring lanes hold neighbouring
                // exposures, i.e. nearly the same geometry and code path
                GLH_TL(3);
                for (int v = gtid; v < M; v += ntot) {
                    int i;
                    const float dtc = entry(v, &i);
                    const float2 o2 = want_chi2 ? obs_of(i) : make_float2(0.f, 0.f);
                    float sum = 0.f;
                    for (int j = 0; j < S; ++j) {
                        float xc, yc;
                        position(dtc, j, &xc, &yc);
                        sum += blocked_hot(s_trap, xc, yc, a, b, ab, e2, k0, k1, k2);
                    }
                    finish(i, sum * inv_ss, o2);
                }
                GLH_TL(6);
                if (frow) fill(gtid, ntot);
            }
        }
        GLH_TL(4);
        // ---- 4. chi^2
        if (want_chi2 && !chi2_done) chi2_unit(acc, cls, wk, nwsum);
    }
    if (any_defer) {
        kun = 0;
        for (unsigned un = blockIdx.y; un < nunits; un += gridDim.y, ++kun) {
            __syncthreads();   // generic_unit's shared walker of the previous unit is dead; s_defer is visible
            if (!((s_defer[kun >> 5] >> (kun & 31u)) & 1u)) continue;
            const int wk = A.nseg == 1 ? (int)un : (int)(un / (unsigned)A.nseg);
            const int t_lo = (int)(un - (unsigned)wk * (unsigned)A.nseg) * A.seglen;
            double gacc = 0.0;
            const int cls = generic_unit(A, PRE, wk, t_lo, min(A.seglen, A.T - t_lo), gtid, ntot, s_trap, &gacc,
                                         s_d, s_li, &s_cnt[0][0]);
            if (want_chi2) chi2_unit(gacc, cls, wk, HOT_NW);
        }
    }
    if (!started) cluster.barrier_wait();
    if (A.done_count && tid == 0) {
        // Host completion signal.  Everything this CTA wrote (chi^2: thread 0 of rank 0, possibly straight
        // into mapped host memory) is ordered before its count by a device-scope fence; the last CTA to
        // count sees every other count (atomic at device scope), re-arms the counter for the next launch
        // and publishes the lot to the host with ONE system-scope fence before it raises the flag
        // (causality is cumulative across the two scopes; a system fence per CTA measured +6 us on 256 CTAs).
        __threadfence();
        const int total = (int)(gridDim.x * gridDim.y);
        if (atomicAdd(A.done_count, 1) == total - 1) {
            *A.done_count = 0;
            __threadfence_system();
            *(volatile int*)A.done_flag = 1;
        }
    }
}

}  // namespace glh
