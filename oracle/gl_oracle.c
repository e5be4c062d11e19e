/* gl_oracle.c -- TEST INFRASTRUCTURE ONLY (not part of the product path).
 *
 * Plain, slow, double-precision CPU oracle for the oblate-planet transit model
 * of arXiv:2410.05408 ("greenlantern", Price et al.).  It is written from the
 * paper alone and shares no code, header, table or constant generator with
 * the CUDA path under paper_2410_05408_b200/csrc/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call it.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md):
 *
 *   F_inst = 1 - [c0*A_flat + c1*A_lin + c2*A_quad] / [pi*(1 - u1/3 - u2/6)]
 *
 *   A_flat = closed-contour integral of f_flat  (eq. 21)
 *   A_lin  = closed-contour integral of f_lin   (eq. 22)
 *   A_quad = closed-contour integral of f_quad  (eq. 23)
 *
 * over the boundary of  Omega = (projected ellipsoid outline) n (unit disc),
 * "the closed curve encompassing the area of the projected ellipsoid that is
 * also within the stellar disk".  c0 = 1-u1-2u2, c1 = u1+2u2,
 * c2 = u2 come from expanding the quadratic limb-darkening law
 * I = 1 - u1(1-mu) - u2(1-mu)^2, mu = sqrt(1-r^2), as c0 + c1*mu + c2*r^2
 * (PAPER.md:127 names the three integrals; the combination is DESIGN.md
 * reading R8).  The outline is eqs. 7-13, its derivatives
 * eqs. 14-15, the rotation eq. 6.
 *
 * How (chosen to be plainly correct, and unlike the CUDA path):
 *   - the <=4 crossings of the outline with the unit circle are found by
 *     BRACKETING: critical points of g(theta)=x_e^2+y_e^2-1 from a 1440-point
 *     scan of g' + bisection, then one bisection per sign change of g between
 *     consecutive critical points.  No quartic algebra, no Newton.
 *   - on outline arcs inside the disc, all three integrands of eqs. 21-23 are
 *     integrated NUMERICALLY, exactly as printed, by adaptive Gauss-Legendre
 *     (16-point value, 8-point error estimate, interval bisection).
 *   - on outline arcs outside the disc the contour runs along the stellar
 *     limb ("snapping", eqs. 16-17); eqs. 21-23 evaluated on
 *     (cos l, sin l) have elementary antiderivatives, used here:
 *       f_flat = l'/2,  f_lin = l'/3,  f_quad = l' * (1/4 - cos(4l)/12).
 *   - orbit: eqs. 9-10, generalised to (e, omega) by
 *     Kepler's equation (reading R7), solved by bisection-safeguarded
 *     Newton to machine precision.
 *   - supersampling: midpoint rule (reading R18); chi^2 with
 *     Neumaier-compensated summation (reading R19).
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"):
 *   sphere + quadratic LD vs the radial limb-darkening integral; uniform LD
 *   fully inside = dx*dy2; circle-circle lens area; brute-force pixel grid and
 *   Monte Carlo; out of transit == 1.0 exactly; time-reversal symmetry;
 *   mu-degeneracy (App. A, eq. A1); the paper's literal snap+Simpson algorithm
 *   (gl_oracle_areas_snap_simpson below) at N=2^16.
 *   PARITY UNPINNED by anything external: e>0 orbits, the supersampling
 *   convention and chi^2 (only self-consistency pins exist).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define GLO_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------ */
/* Rotation matrices, eqs. 3-6                              */
/* ------------------------------------------------------------------------ */

static void mat3_mul(const double *A, const double *B, double *C) {
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double s = 0.0;
            for (int k = 0; k < 3; k++) s += A[3 * i + k] * B[3 * k + j];
            C[3 * i + j] = s;
        }
}

/* R(zeta,eta,xi) = R_x(zeta) R_y(eta) R_z(xi), row-major r1..r9 (eq. 6). */
void gl_oracle_rotation(double zeta, double eta, double xi, double *r) {
    const double Rx[9] = {1, 0, 0, 0, cos(zeta), -sin(zeta), 0, sin(zeta), cos(zeta)}; /* eq. 3 */
    const double Ry[9] = {cos(eta), 0, sin(eta), 0, 1, 0, -sin(eta), 0, cos(eta)};     /* eq. 4 */
    const double Rz[9] = {cos(xi), -sin(xi), 0, sin(xi), cos(xi), 0, 0, 0, 1};         /* eq. 5 */
    double T[9];
    mat3_mul(Rx, Ry, T);
    mat3_mul(T, Rz, r);
}

/* Outline amplitudes, eqs. 11-13.  out = {dx, dy1, dy2}. */
void gl_oracle_outline(double a, double b, double c, double zeta, double eta, double xi,
                       double *out) {
    double r[9];
    gl_oracle_rotation(zeta, eta, xi, r);
    const double r1 = r[0], r2 = r[1], r3 = r[2], r4 = r[3], r5 = r[4], r6 = r[5], r7 = r[6],
                 r8 = r[7], r9 = r[8];
    const double dx = sqrt(a * a * r1 * r1 + b * b * r4 * r4 + c * c * r7 * r7);          /* eq. 11 */
    const double dy1 = (a * a * r1 * r2 + b * b * r4 * r5 + c * c * r7 * r8) / dx;        /* eq. 12 */
    const double dy2 =
        sqrt(a * a * b * b * r9 * r9 + a * a * c * c * r6 * r6 + b * b * c * c * r3 * r3) / dx; /* eq. 13 */
    out[0] = dx;
    out[1] = dy1;
    out[2] = dy2;
}

/* Tidally locked outline, eqs. B14-B16; alpha, beta as in eq. B13. */
void gl_oracle_outline_locked(double a, double b, double c, double zeta, double eta, double xi,
                              double alpha, double beta, double *out) {
    double r[9];
    gl_oracle_rotation(zeta, eta, xi, r);
    const double ca = cos(alpha), sa = sin(alpha), cb = cos(beta), sb = sin(beta);
    const double p1 = sb * (r[2] * ca + r[1] * sa) - r[0] * cb;
    const double p2 = sb * (r[5] * ca + r[4] * sa) - r[3] * cb;
    const double p3 = sb * (r[8] * ca + r[7] * sa) - r[6] * cb;
    const double q1 = r[2] * sa - r[1] * ca;
    const double q2 = r[5] * sa - r[4] * ca;
    const double q3 = r[8] * sa - r[7] * ca;
    const double s1 = r[6] * sb + cb * (r[8] * ca + r[7] * sa);
    const double s2 = r[3] * sb + cb * (r[5] * ca + r[4] * sa);
    const double s3 = r[0] * sb + cb * (r[2] * ca + r[1] * sa);
    const double dx = sqrt(a * a * p1 * p1 + b * b * p2 * p2 + c * c * p3 * p3);           /* B14 */
    const double dy1 = (a * a * p1 * q1 + b * b * p2 * q2 + c * c * p3 * q3) / dx;         /* B15 */
    const double dy2 =
        sqrt(a * a * b * b * s1 * s1 + a * a * c * c * s2 * s2 + b * b * c * c * s3 * s3) / dx; /* B16 */
    out[0] = dx;
    out[1] = dy1;
    out[2] = dy2;
}

/* ------------------------------------------------------------------------ */
/* Outline point and integrands                                              */
/* ------------------------------------------------------------------------ */

typedef struct {
    double x0, y0, dx, dy1, dy2;
} outline_t;

/* eqs. 7-8 and 14-15 */
static void outline_point(const outline_t *o, double th, double *x, double *y, double *xp,
                          double *yp) {
    const double c = cos(th), s = sin(th);
    *x = o->x0 + o->dx * c;                 /* eq. 7  */
    *y = o->y0 + o->dy1 * c + o->dy2 * s;   /* eq. 8  */
    *xp = -o->dx * s;                       /* eq. 14 */
    *yp = -o->dy1 * s + o->dy2 * c;         /* eq. 15 */
}

/* [1 - (1-s)^{3/2}] / s for s = r^2 in [0,1]; 1-r^2 clamped at 0 (reading R11);
 * the 0/0 at r=0 has the limit 3/2 (reading R9).  expm1/log1p keep full
 * precision for small s without a series switch. */
static double lin_factor(double s) {
    if (s >= 1.0) return 1.0 / s;
    if (s <= 0.0) return 1.5;
    return -expm1(1.5 * log1p(-s)) / s;
}

/* eqs. 21-23 at a point (x,y) with tangent (xp,yp); out = {f_flat, f_lin, f_quad} */
static void integrands(double x, double y, double xp, double yp, double *f) {
    const double r2 = x * x + y * y;
    const double fflat = 0.5 * (x * yp - y * xp);                                   /* eq. 21 */
    const double flin = (2.0 / 3.0) * lin_factor(r2) * fflat;                       /* eq. 22 */
    const double fquad =
        0.5 * (x * (x * x / 3.0 + y * y) * yp - y * (x * x + y * y / 3.0) * xp);    /* eq. 23 */
    f[0] = fflat;
    f[1] = flin;
    f[2] = fquad;
}

static void integrands_on_outline(const outline_t *o, double th, double *f) {
    double x, y, xp, yp;
    outline_point(o, th, &x, &y, &xp, &yp);
    integrands(x, y, xp, yp, f);
}

/* g(theta) = x_e^2 + y_e^2 - 1 and its derivative */
static double g_of(const outline_t *o, double th) {
    double x, y, xp, yp;
    outline_point(o, th, &x, &y, &xp, &yp);
    return x * x + y * y - 1.0;
}
static double gp_of(const outline_t *o, double th) {
    double x, y, xp, yp;
    outline_point(o, th, &x, &y, &xp, &yp);
    return 2.0 * (x * xp + y * yp);
}

/* ------------------------------------------------------------------------ */
/* Gauss-Legendre nodes (computed, not transcribed) and adaptive quadrature  */
/* ------------------------------------------------------------------------ */

#define GLO_NHI 16
#define GLO_NLO 8
static double glx_hi[GLO_NHI], glw_hi[GLO_NHI], glx_lo[GLO_NLO], glw_lo[GLO_NLO];
static int gl_tables_ready = 0;

/* Nodes = roots of the Legendre polynomial P_n (Newton on the three-term
 * recurrence); weights = 2 / ((1-x^2) P_n'(x)^2). */
void gl_oracle_leggauss(int n, double *x, double *w) {
    for (int i = 0; i < n; i++) {
        double z = cos(GLO_PI * (i + 0.75) / (n + 0.5));
        double pp = 1.0;
        for (int it = 0; it < 100; it++) {
            double p0 = 1.0, p1 = z;
            for (int k = 2; k <= n; k++) {
                const double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            pp = n * (z * p1 - p0) / (z * z - 1.0);
            const double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        /* one more derivative evaluation at the converged node */
        {
            double p0 = 1.0, p1 = z;
            for (int k = 2; k <= n; k++) {
                const double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            pp = n * (z * p1 - p0) / (z * z - 1.0);
        }
        x[n - 1 - i] = z;
        w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

static void ensure_tables(void) {
    if (gl_tables_ready) return;
#ifdef _OPENMP
#pragma omp critical(glo_tables)
#endif
    {
        if (!gl_tables_ready) {
            gl_oracle_leggauss(GLO_NHI, glx_hi, glw_hi);
            gl_oracle_leggauss(GLO_NLO, glx_lo, glw_lo);
            gl_tables_ready = 1;
        }
    }
}

static void gl_fixed(const outline_t *o, double lo, double hi, int n, const double *xs,
                     const double *ws, double *out) {
    const double m = 0.5 * (lo + hi), h = 0.5 * (hi - lo);
    double acc[3] = {0, 0, 0};
    for (int i = 0; i < n; i++) {
        double f[3];
        integrands_on_outline(o, m + h * xs[i], f);
        for (int k = 0; k < 3; k++) acc[k] += ws[i] * f[k];
    }
    for (int k = 0; k < 3; k++) out[k] = h * acc[k];
}

/* adaptive: accept the 16-point value when it agrees with the 8-point value */
static void adaptive(const outline_t *o, double lo, double hi, int depth, double *acc) {
    double hi16[3], lo8[3];
    gl_fixed(o, lo, hi, GLO_NHI, glx_hi, glw_hi, hi16);
    gl_fixed(o, lo, hi, GLO_NLO, glx_lo, glw_lo, lo8);
    double err = 0.0, mag = 0.0;
    for (int k = 0; k < 3; k++) {
        err = fmax(err, fabs(hi16[k] - lo8[k]));
        mag = fmax(mag, fabs(hi16[k]));
    }
    if (err <= 1e-18 + 2e-16 * mag || depth >= 60 || !(hi - lo > 1e-15)) {
        for (int k = 0; k < 3; k++) acc[k] += hi16[k];
        return;
    }
    const double mid = 0.5 * (lo + hi);
    adaptive(o, lo, mid, depth + 1, acc);
    adaptive(o, mid, hi, depth + 1, acc);
}

/* ------------------------------------------------------------------------ */
/* Crossings by bracketing                                                   */
/* ------------------------------------------------------------------------ */

static double bisect(const outline_t *o, double (*fn)(const outline_t *, double), double lo,
                     double hi) {
    /* fn(lo) and fn(hi) have opposite "positive" flags */
    const int plo = fn(o, lo) > 0.0;
    for (int it = 0; it < 200; it++) {
        const double mid = 0.5 * (lo + hi);
        if (!(mid > lo && mid < hi)) break;
        if ((fn(o, mid) > 0.0) == plo)
            lo = mid;
        else
            hi = mid;
    }
    return 0.5 * (lo + hi);
}

static int cmp_double(const void *a, const void *b) {
    const double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

#define GLO_NSCAN 1440

/* Areas {A_flat, A_lin, A_quad} of Omega; returns the number of crossings found
 * (0, 2 or 4), or -1 when Omega is empty. */
int gl_oracle_areas(double x0, double y0, double dx, double dy1, double dy2, double *A) {
    ensure_tables();
    const outline_t o = {x0, y0, dx, dy1, dy2};
    A[0] = A[1] = A[2] = 0.0;

    /* 0. trivially disjoint: every outline point is at least
     * r0 - (dx + |dy1| + dy2) from the star centre (triangle inequality on
     * eqs. 7-8), so nothing overlaps the unit disc */
    if (sqrt(x0 * x0 + y0 * y0) - (dx + fabs(dy1) + dy2) >= 1.0) return -1;

    /* 1. critical points of g: sign changes of g' on the scan, then bisection */
    double crit[16];
    int ncrit = 0;
    /* the scan starts at an offset so that the exact zeros of g' that symmetric
     * configurations put at theta = 0, pi/2, pi ... do not sit on scan points,
     * and it closes on the very value it started with (exact periodicity) */
    const double step = 2.0 * GLO_PI / GLO_NSCAN;
    const double th_off = 0.5 * step * 0.61803398874989;
    const double first = gp_of(&o, th_off);
    double prev = first;
    for (int k = 1; k <= GLO_NSCAN && ncrit < 16; k++) {
        const double th = th_off + k * step;
        const double cur = (k == GLO_NSCAN) ? first : gp_of(&o, th);
        if ((prev > 0.0) != (cur > 0.0)) crit[ncrit++] = bisect(&o, gp_of, th - step, th);
        prev = cur;
    }

    /* 2. breakpoints = critical points + one bisected root per sign change of g */
    double brk[32];
    int nbrk = 0, nroots = 0;
    if (ncrit == 0) {
        /* g is constant (circle centred on the star): a single arc [0, 2pi] */
        brk[nbrk++] = 0.0;
    } else {
        for (int i = 0; i < ncrit; i++) {
            const double ta = crit[i];
            const double tb = (i + 1 < ncrit) ? crit[i + 1] : crit[0] + 2.0 * GLO_PI;
            brk[nbrk++] = ta;
            if ((g_of(&o, ta) > 0.0) != (g_of(&o, tb) > 0.0)) {
                brk[nbrk++] = bisect(&o, g_of, ta, tb);
                nroots++;
            }
        }
    }
    qsort(brk, nbrk, sizeof(double), cmp_double);

    /* 3. walk the arcs between consecutive breakpoints */
    int any_inside = 0;
    for (int i = 0; i < nbrk; i++) {
        const double ta = brk[i];
        const double tb = (i + 1 < nbrk) ? brk[i + 1] : brk[0] + 2.0 * GLO_PI;
        if (!(tb > ta)) continue;
        const double gm = g_of(&o, 0.5 * (ta + tb));
        if (gm < 0.0) {
            /* inside the disc: integrate eqs. 21-23 along the outline */
            any_inside = 1;
            adaptive(&o, ta, tb, 0, A);
        } else {
            /* outside: the contour follows the limb between the radial
             * projections (eqs. 16-17) of the arc's end points */
            double xa, ya, xb, yb, t1, t2;
            outline_point(&o, ta, &xa, &ya, &t1, &t2);
            outline_point(&o, tb, &xb, &yb, &t1, &t2);
            const double la = atan2(ya, xa);                                 /* eq. 16 */
            const double dl = atan2(xa * yb - ya * xb, xa * xb + ya * yb);   /* in (-pi, pi] */
            const double lb = la + dl;
            A[0] += dl / 2.0;
            A[1] += dl / 3.0;
            A[2] += dl / 4.0 - (sin(4.0 * lb) - sin(4.0 * la)) / 48.0;
        }
    }
    if (!any_inside) {
        A[0] = A[1] = A[2] = 0.0;
        return -1;
    }
    return nroots;
}

/* The paper's literal algorithm: radial snapping of outside
 * points, eqs. 16-20, and composite Simpson's rule over theta in [0, 2pi] with N
 * (even) intervals.  An independent route to the same three numbers. */
void gl_oracle_areas_snap_simpson(double x0, double y0, double dx, double dy1, double dy2,
                                  long N, double *A) {
    const outline_t o = {x0, y0, dx, dy1, dy2};
    if (N % 2) N++;
    const double h = 2.0 * GLO_PI / (double)N;
    double acc[3] = {0, 0, 0}, comp[3] = {0, 0, 0};
    for (long k = 0; k <= N; k++) {
        double x, y, xp, yp, f[3];
        outline_point(&o, k * h, &x, &y, &xp, &yp);
        const double r2 = x * x + y * y;
        if (r2 > 1.0) {
            const double lam = atan2(y, x);                    /* eq. 16 */
            const double dlam = (-y * xp + x * yp) / r2;       /* eq. 19 */
            x = cos(lam);                                      /* eq. 17 */
            y = sin(lam);
            xp = -y * dlam;                                    /* eq. 18 */
            yp = x * dlam;
        }
        integrands(x, y, xp, yp, f);
        const double wk = (k == 0 || k == N) ? 1.0 : ((k % 2) ? 4.0 : 2.0);
        for (int j = 0; j < 3; j++) { /* Neumaier-compensated accumulation */
            const double v = wk * f[j], t = acc[j] + v;
            comp[j] += (fabs(acc[j]) >= fabs(v)) ? (acc[j] - t) + v : (v - t) + acc[j];
            acc[j] = t;
        }
    }
    for (int j = 0; j < 3; j++) A[j] = (acc[j] + comp[j]) * h / 3.0;
}

/* Instantaneous relative flux for a planet whose outline is (x0,y0,dx,dy1,dy2). */
double gl_oracle_flux_outline(double x0, double y0, double dx, double dy1, double dy2, double u1,
                              double u2) {
    double A[3];
    if (gl_oracle_areas(x0, y0, dx, dy1, dy2, A) < 0) return 1.0;
    const double c0 = 1.0 - u1 - 2.0 * u2, c1 = u1 + 2.0 * u2, c2 = u2;
    const double norm = GLO_PI * (1.0 - u1 / 3.0 - u2 / 6.0);
    return 1.0 - (c0 * A[0] + c1 * A[1] + c2 * A[2]) / norm;
}

/* ------------------------------------------------------------------------ */
/* Orbit (eqs. 9-10 + Kepler, reading R7)                                    */
/* ------------------------------------------------------------------------ */

/* Solve E - e sin E = M; Newton safeguarded by bisection on [M-e, M+e]. */
double gl_oracle_kepler(double M, double e) {
    if (e == 0.0) return M;
    double lo = M - e, hi = M + e, E = M;
    for (int it = 0; it < 200; it++) {
        const double fE = E - e * sin(E) - M;
        if (fE > 0.0) hi = E; else lo = E;
        double En = E - fE / (1.0 - e * cos(E));
        if (!(En > lo && En < hi)) En = 0.5 * (lo + hi);
        if (En == E) break;
        E = En;
    }
    return E;
}

/* Sky-plane position of the planet centre at time t.  p = the 12-vector
 * (t0, P, a/R*, b, e, omega, Rp_eq, f, xi, eta, u1, u2).  Returns 1 when the
 * planet is in front of the star (cos phi > 0), else 0. */
int gl_oracle_orbit(const double *p, double t, double *x0, double *y0, double *phi_out);
int gl_oracle_position(const double *p, double t, double *x0, double *y0) {
    double phi;
    return gl_oracle_orbit(p, t, x0, y0, &phi);
}

/* The same, also returning the orbital angle from conjunction phi (alpha of eqs. 9-10). */
int gl_oracle_orbit(const double *p, double t, double *x0, double *y0, double *phi_out) {
    const double t0 = p[0], P = p[1], aR = p[2], b = p[3], e = p[4], om = p[5];
    const double nuc = 0.5 * GLO_PI - om;
    const double Ec = 2.0 * atan2(sqrt(1.0 - e) * sin(0.5 * nuc), sqrt(1.0 + e) * cos(0.5 * nuc));
    const double Mc = Ec - e * sin(Ec);
    /* the phase is reduced before multiplying by 2 pi so that long baselines
     * keep full precision */
    double ph = (t - t0) / P;
    ph -= floor(ph + 0.5);
    const double M = Mc + 2.0 * GLO_PI * ph;
    const double E = gl_oracle_kepler(M, e);
    const double nu = 2.0 * atan2(sqrt(1.0 + e) * sin(0.5 * E), sqrt(1.0 - e) * cos(0.5 * E));
    const double r = aR * (1.0 - e * cos(E));
    const double phi = nu + om - 0.5 * GLO_PI;
    const double cosi = (b / aR) * (1.0 + e * sin(om)) / (1.0 - e * e);
    *x0 = r * cos(phi) * cosi;   /* eq. 9 with alpha -> phi, d -> r, sin(beta) = cos i */
    *y0 = r * sin(phi);          /* eq. 10 */
    *phi_out = phi;
    return cos(phi) > 0.0;
}

/* Per-walker validity. */
int gl_oracle_params_valid(const double *p) {
    for (int k = 0; k < 12; k++)
        if (!isfinite(p[k])) return 0;
    const double P = p[1], aR = p[2], b = p[3], e = p[4], om = p[5], Rp = p[6], f = p[7];
    const double u1 = p[10], u2 = p[11];
    if (!(P > 0.0) || !(e >= 0.0 && e < 1.0)) return 0;
    if (!(Rp > 0.0 && Rp < 0.5) || !(f >= 0.0 && f < 1.0)) return 0;
    if (!(aR * (1.0 - e) > 1.0)) return 0;
    if (!(fabs(b) * (1.0 + e * sin(om)) <= aR * (1.0 - e * e))) return 0;
    if (!(1.0 - u1 / 3.0 - u2 / 6.0 > 0.0)) return 0;
    return 1;
}

/* Oblate spheroid: a = Rp_eq (1-f) along x' (polar), b = c = Rp_eq; zeta = 0
 * (App. A :368; readings R4, R5). */
static void walker_outline(const double *p, double *d3) {
    const double Rp = p[6], f = p[7], xi = p[8], eta = p[9];
    gl_oracle_outline(Rp * (1.0 - f), Rp, Rp, 0.0, eta, xi, d3);
}

/* Exposure-averaged flux of walker p at time t (midpoint rule, reading R18). */
double gl_oracle_flux_time(const double *p, double t, double t_exp, int n_ss) {
    if (!gl_oracle_params_valid(p)) return NAN;
    double d3[3];
    walker_outline(p, d3);
    double sum = 0.0;
    for (int j = 0; j < n_ss; j++) {
        const double tj = t + ((j + 0.5) / n_ss - 0.5) * t_exp;
        double x0, y0, F = 1.0;
        if (gl_oracle_position(p, tj, &x0, &y0))
            F = gl_oracle_flux_outline(x0, y0, d3[0], d3[1], d3[2], p[10], p[11]);
        sum += F;
    }
    return sum / n_ss;
}

/* ------------------------------------------------------------------------ */
/* NEXT-2: general triaxial ellipsoids and tidally locked    */
/* planets.  Extended row p[16]: columns 0-11 as above, then                   */
/*   12 zeta [rad] (third Euler angle of eq. 6)                */
/*   13 rb, 14 rc: semi-axes b = Rp_eq rb along y', c = Rp_eq rc along z'      */
/*      (a = Rp_eq (1-f) along x' as before; the oblate model is rb = rc = 1)  */
/*   15 locked: 0 = orientation fixed in the observer frame (eq. 2, eqs.       */
/*      11-13), 1 = tidally locked (eq. B13): the outline amplitudes follow    */
/*      eqs. B14-B16 with alpha = the orbital angle from    */
/*      conjunction (phi of reading R7; alpha of eqs. 9-10 for e = 0) and      */
/*      sin(beta) = cos i; the centre still moves by eqs. 9-10.                */
/* ------------------------------------------------------------------------ */
int gl_oracle_params_ex_valid(const double *p) {
    if (!gl_oracle_params_valid(p)) return 0;
    for (int k = 12; k < 16; k++)
        if (!isfinite(p[k])) return 0;
    const double Rp = p[6], rb = p[13], rc = p[14];
    if (!(rb > 0.0) || !(rc > 0.0) || !(Rp * rb < 0.5) || !(Rp * rc < 0.5)) return 0;
    if (!(p[15] == 0.0 || p[15] == 1.0)) return 0;
    return 1;
}

double gl_oracle_flux_time_ex(const double *p, double t, double t_exp, int n_ss) {
    if (!gl_oracle_params_ex_valid(p)) return NAN;
    const double Rp = p[6], f = p[7], xi = p[8], eta = p[9], zeta = p[12];
    const double sa = Rp * (1.0 - f), sb = Rp * p[13], sc = Rp * p[14];
    const int locked = p[15] == 1.0;
    double d3[3];
    gl_oracle_outline(sa, sb, sc, zeta, eta, xi, d3);
    const double e = p[4], om = p[5];
    const double cosi = (p[3] / p[2]) * (1.0 + e * sin(om)) / (1.0 - e * e);
    const double beta = asin(cosi);   /* eq. 9: x0 = d cos(alpha) sin(beta) */
    double sum = 0.0;
    for (int j = 0; j < n_ss; j++) {
        const double tj = t + ((j + 0.5) / n_ss - 0.5) * t_exp;
        double x0, y0, alpha, F = 1.0;
        if (gl_oracle_orbit(p, tj, &x0, &y0, &alpha)) {
            if (locked) gl_oracle_outline_locked(sa, sb, sc, zeta, eta, xi, alpha, beta, d3);
            F = gl_oracle_flux_outline(x0, y0, d3[0], d3[1], d3[2], p[10], p[11]);
        }
        sum += F;
    }
    return sum / n_ss;
}

/* ------------------------------------------------------------------------ */
/* NEXT-3: the paper's sampling parameters (App. A,           */
/* PAPER.md:366-430).  mu, nu replace (f, eta); q1, q2 replace (u1, u2)        */
/* (Kipping's map, as in BASELINE.json config 3); the mean radius r replaces   */
/* the equatorial one, R_eq = r / (1-f)^(1/3) (volume-equivalent sphere:       */
/* a b c = R_eq^3 (1-f); SURVEY.md ambiguity 22).                              */
/* ------------------------------------------------------------------------ */

/* eqs. A1 and A4: (f, eta) -> (mu, nu). */
void gl_oracle_munu_of(double f, double eta, double *out2) {
    const double c2 = cos(2.0 * eta), g = f * (f - 2.0);
    out2[0] = (f - 1.0) * (f - 1.0) + g * c2;                                         /* A1 */
    out2[1] = (2.0 + 2.0 * g * cos(eta) * cos(eta) + (f - 1.0) * sqrt(4.0 + 2.0 * g * (1.0 + c2))) /
              (2.0 + g * (1.0 + c2));                                                 /* A4 */
}

/* eqs. A2-A3 and A1 solved for eta in [0, pi/2]: (mu, nu) -> (f, eta). */
void gl_oracle_feta_of(double mu, double nu, double *out2) {
    const double fmin = 1.0 - sqrt(0.5 * (mu + 1.0));                                 /* A2 */
    const double f = fmin + (1.0 - fmin) * nu;                                        /* A3 */
    double c2 = (f > 0.0) ? (mu - (f - 1.0) * (f - 1.0)) / (f * (f - 2.0)) : 1.0;     /* A1 */
    if (c2 > 1.0) c2 = 1.0;
    if (c2 < -1.0) c2 = -1.0;
    out2[0] = f;
    out2[1] = 0.5 * acos(c2);
}

/* eq. A6: ln p(mu, nu). */
double gl_oracle_log_prior_munu(double mu, double nu) {
    const double q = nu * (nu - 2.0) * (mu * (nu - 1.0) * (nu - 1.0) + nu * (nu - 2.0) - 1.0);
    if (!(mu > -1.0 && mu < 1.0 && nu > 0.0 && nu <= 1.0) || !(q > 0.0)) return -INFINITY;
    return -1.5 * log(2.0) - 0.5 * log(q);
}

/* eqs. A10 and A12: two uniform variates (u, w) -> (mu, nu) distributed as eq. A6. */
void gl_oracle_munu_from_uniform(double u, double w, double *out2) {
    const double nu = u * u / (u * u - 2.0 * u + 2.0);                                /* A10 */
    const double s = sqrt(nu * (2.0 - nu)), d = (nu - 1.0) * (nu - 1.0);
    out2[0] = (4.0 * w + 4.0 * (w * w - w) * s + 2.0 * (nu * (nu - 2.0) - 1.0) * w * w - d) / d; /* A12 */
    out2[1] = nu;
}

/* Sampling row (t0, P, a/R*, b, e, omega, r_mean, mu, nu, xi, q1, q2) -> model row
 * (t0, P, a/R*, b, e, omega, Rp_eq, f, xi, eta, u1, u2) and ln p(mu, nu).  A row outside
 * mu in (-1,1), nu in (0,1], q1, q2 in [0,1], r_mean > 0 gives NaNs and -inf. */
void gl_oracle_params_from_munu(const double *srow, double *prow, double *logprior) {
    const double r = srow[6], mu = srow[7], nu = srow[8], q1 = srow[10], q2 = srow[11];
    const double lp = gl_oracle_log_prior_munu(mu, nu);
    int ok = isfinite(lp) && (r > 0.0) && (q1 >= 0.0 && q1 <= 1.0) && (q2 >= 0.0 && q2 <= 1.0);
    for (int k = 0; k < 12; k++) ok = ok && isfinite(srow[k]);
    if (!ok) {
        for (int k = 0; k < 12; k++) prow[k] = NAN;
        if (logprior) *logprior = -INFINITY;
        return;
    }
    double fe[2];
    gl_oracle_feta_of(mu, nu, fe);
    for (int k = 0; k < 6; k++) prow[k] = srow[k];
    prow[6] = r / cbrt(1.0 - fe[0]);
    prow[7] = fe[0];
    prow[8] = srow[9];
    prow[9] = fe[1];
    prow[10] = 2.0 * sqrt(q1) * q2;
    prow[11] = sqrt(q1) * (1.0 - 2.0 * q2);
    if (logprior) *logprior = lp;
}

static int pick_threads(int nthreads) {
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
    return nthreads;
#else
    (void)nthreads;
    return 1;
#endif
}

/* flux[B,T] for params[B,12], times[T].  Returns the thread count used. */
int gl_oracle_lightcurve(const double *params, int B, const double *times, int T, double t_exp,
                         int n_ss, double *flux, int nthreads) {
    ensure_tables();
    nthreads = pick_threads(nthreads);
    const long total = (long)B * T;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
#endif
    for (long k = 0; k < total; k++) {
        const int b = (int)(k / T), i = (int)(k % T);
        flux[k] = gl_oracle_flux_time(params + 12 * (long)b, times[i], t_exp, n_ss);
    }
    return nthreads;
}

/* chi2[B] = sum_i ((obs_i - F_b(t_i)) / sigma_i)^2, Neumaier-summed; flux may
 * be NULL.  Invalid walkers: flux row NaN, chi2 = +inf. */
int gl_oracle_loglike(const double *params, int B, const double *times, int T, double t_exp,
                      int n_ss, const double *obs, const double *sigma, double *chi2,
                      double *flux, int nthreads) {
    ensure_tables();
    nthreads = pick_threads(nthreads);
    double *tmp = flux ? flux : (double *)malloc(sizeof(double) * (size_t)B * T);
    gl_oracle_lightcurve(params, B, times, T, t_exp, n_ss, tmp, nthreads);
    for (int b = 0; b < B; b++) {
        if (!gl_oracle_params_valid(params + 12 * (long)b)) {
            chi2[b] = INFINITY;
            continue;
        }
        double acc = 0.0, comp = 0.0;
        for (int i = 0; i < T; i++) {
            const double r = (obs[i] - tmp[(long)b * T + i]) / sigma[i];
            const double v = r * r, t = acc + v;
            comp += (fabs(acc) >= fabs(v)) ? (acc - t) + v : (v - t) + acc;
            acc = t;
        }
        chi2[b] = acc + comp;
    }
    if (!flux) free(tmp);
    return nthreads;
}

/* flux[B,T] for params_ex[B,16] (NEXT-2). */
int gl_oracle_lightcurve_ex(const double *params, int B, const double *times, int T, double t_exp,
                            int n_ss, double *flux, int nthreads) {
    ensure_tables();
    nthreads = pick_threads(nthreads);
    const long total = (long)B * T;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16) num_threads(nthreads)
#endif
    for (long k = 0; k < total; k++) {
        const int b = (int)(k / T), i = (int)(k % T);
        flux[k] = gl_oracle_flux_time_ex(params + 16 * (long)b, times[i], t_exp, n_ss);
    }
    return nthreads;
}

/* Bare geometries (config 5): row = (d, Rp, f_proj, PA, u1, u2); planet centre
 * at (d, 0), semi-major Rp at position angle PA (counter-clockwise from the
 * star-centre -> planet-centre direction), semi-minor Rp (1 - f_proj).
 * The outline amplitudes are the lower-Cholesky factor of the 2x2 covariance
 * of that ellipse -- the same object eqs. 11-13 produce. */
int gl_oracle_flux_geometry(const double *geom, long N, double *flux, int nthreads) {
    ensure_tables();
    nthreads = pick_threads(nthreads);
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 64) num_threads(nthreads)
#endif
    for (long k = 0; k < N; k++) {
        const double *g = geom + 6 * k;
        const double d = g[0], Rp = g[1], fp = g[2], pa = g[3], u1 = g[4], u2 = g[5];
        int ok = 1;
        for (int j = 0; j < 6; j++) ok = ok && isfinite(g[j]);
        if (!ok || !(d >= 0.0) || !(Rp > 0.0 && Rp < 0.5) || !(fp >= 0.0 && fp < 1.0) ||
            !(1.0 - u1 / 3.0 - u2 / 6.0 > 0.0)) {
            flux[k] = NAN;
            continue;
        }
        const double a = Rp, b = Rp * (1.0 - fp);
        const double c = cos(pa), s = sin(pa);
        const double Cxx = a * a * c * c + b * b * s * s;
        const double Cxy = (a * a - b * b) * c * s;
        const double dx = sqrt(Cxx), dy1 = Cxy / dx, dy2 = a * b / dx;
        flux[k] = gl_oracle_flux_outline(d, 0.0, dx, dy1, dy2, u1, u2);
    }
    return nthreads;
}
