/* greenlantern_b200.h -- C ABI of the B200 (sm_100a) oblate-planet transit library.
 *
 * The model is the one of arXiv:2410.05408 (Price et al., the `greenlantern` code); citations
 * are PAPER.md:<line> (+ equation) of the paper text and DESIGN.md "Readings" (R<n>) where the
 * paper is silent.  The library holds hand-written CUDA only; there is no CPU fallback.
 *
 * Conventions common to every entry point
 *   - Unless a parameter is marked HOST, every pointer is a CUDA DEVICE pointer owned by the
 *     caller.  The library never frees, retains or reallocates it.
 *   - Work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream) and the call returns WITHOUT synchronising.  Buffers must stay alive until the
 *     stream has passed the work.
 *   - The device-pointer entry points allocate nothing and keep no per-call state: they are
 *     re-entrant and may be issued concurrently on different streams.  What the library DOES keep:
 *     (1) per device, the quadrature tables in constant memory, uploaded once by the first call on that
 *     device (immutable afterwards); (2) per calling thread and device, for the *_host wrappers only,
 *     one non-blocking stream and one private cudaMemPool that keeps its scratch between calls (the
 *     device's default pool is not touched); both live until the thread ends; (3) what a gl_series
 *     handle owns (see gl_series_create).  Nothing is read from the environment.
 *   - Return value: GL_OK or a negative gl_status.  Argument errors (GL_EINVAL) enqueue nothing.
 *     B == 0, T == 0 or N == 0 is GL_OK and enqueues nothing.
 *   - Parameters, times, observations and sigmas cross the boundary as fp64 whatever the compute
 *     dtype: an fp32 time stamp at |t| ~ 40 d is coarser than the whole flux error budget
 *     (DESIGN.md "Precision plan").
 *
 * Parameter row, GL_NPARAMS = 12 doubles (north_star of BASELINE.json; R4-R7):
 *    0 t0      time of inferior conjunction (same unit as `times`)
 *    1 P       orbital period
 *    2 a/R*    semi-major axis in stellar radii
 *    3 b       signed sky-plane x-offset of the planet centre at t0, in stellar radii
 *              (x0(t0) = b, eq. 9 with d sin(beta) = b)
 *    4 e       eccentricity, 0 <= e < 1          5 omega   argument of periastron [rad]
 *    6 Rp_eq   equatorial radius / R*, 0 < Rp_eq < 0.5
 *    7 f       flattening (R_eq - R_pol)/R_eq, 0 <= f < 1        (eq. 1)
 *    8 xi      sky-projected obliquity [rad]: rotation about z' in eq. 6
 *    9 eta     tilt of the spin axis out of the sky plane [rad]: rotation about y' in eq. 6
 *   10 u1, 11 u2   quadratic limb darkening I = 1 - u1(1-mu) - u2(1-mu)^2
 *
 * What a flux value is (SURVEY.md 8(c); PAPER.md:127-135 eqs. 21-23, :145):
 *    F_inst = 1 - [c0 A_flat + c1 A_lin + c2 A_quad] / [pi (1 - u1/3 - u2/6)],
 *    A_flat, A_lin, A_quad = integrals of 1, sqrt(1-r^2), r^2 over (projected outline) n (unit
 *    disc), c0 = 1-u1-2u2, c1 = u1+2u2, c2 = u2; F_inst = 1 when the overlap is empty or the
 *    planet is behind the star.  F(t_i) = mean of F_inst over n_ss sub-exposures at
 *    t_i + ((j+1/2)/n_ss - 1/2) t_exp, j = 0..n_ss-1 (midpoint rule, R18).
 *
 * Per-walker invalid parameters do not fail a call: that walker's flux row is NaN and its
 * chi^2 is +inf.  Invalid = any non-finite entry, P <= 0, e outside [0,1), Rp_eq outside
 * (0,0.5), f outside [0,1), a/R* (1-e) <= 1, |b|(1+e sin omega) > a/R* (1-e^2),
 * 1 - u1/3 - u2/6 <= 0.
 */
#ifndef GREENLANTERN_B200_H
#define GREENLANTERN_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define GL_NPARAMS 12
#define GL_NGEOM 6
#define GL_NPARAMS_EX 16   /* extended row of gl_lightcurve_ex / gl_loglike_ex */

typedef enum { GL_F32 = 0, GL_F64 = 1 } gl_dtype; /* arithmetic AND output precision */

typedef enum {
    GL_OK = 0,
    GL_EINVAL = -1,       /* null pointer, negative size, n_ss < 1, unknown dtype, t_exp not finite */
    GL_ECUDA = -2,        /* a CUDA runtime call or a launch failed; see gl_last_cuda_error() */
    GL_EUNSUPPORTED = -3, /* size outside what one launch can index (B*T or N >= 2^40)         */
    GL_ECAPACITY = -4     /* size beyond the fixed capacity of a static-scratch entry point    */
} gl_status;

/* gl_lightcurve: flux_out[b*T + i] = F_b(times[i]).
 *   params  [B, GL_NPARAMS] row-major fp64 (device)      times [T] fp64 (device)
 *   t_exp   exposure length (HOST scalar, same unit as times; >= 0)   n_ss >= 1 sub-exposures
 *   flux_out [B, T] row-major, float (GL_F32) or double (GL_F64) (device), fully overwritten.
 * Steps: Kepler + sky position (eqs. 9-10, R7), outline (PAPER.md:89-96
 * eqs. 11-13), outline/limb crossings (R3), boundary integrals (eqs. 21-23),
 * exposure mean -- one fused launch, nothing per-sub-sample is stored (GL_F32: hot_kernel, see gl_loglike;
 * GL_F64: the full kernel). */
int gl_lightcurve(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                  void* flux_out, gl_dtype dtype, void* stream);

/* gl_loglike: chi2_out[b] = sum_i ((obs[i] - F_b(times[i])) / sigma[i])^2   (R19).
 *   obs, sigma [T] fp64 (device), sigma > 0 (a non-positive or non-finite sigma makes every
 *   chi^2 +inf).  chi2_out [B] float/double per dtype, fully overwritten.
 *   flux_out_or_null: optional [B, T] output as in gl_lightcurve; NULL => the model flux never
 *   leaves registers.  The residual sum is accumulated in fp64 in both dtypes.
 *   GL_F64: one launch of the full transit kernel, everything per walker in fp64.
 *   GL_F32 (12-column rows): TWO launches on `stream`, chained by programmatic dependent launch:
 *   (1) a one-CTA kernel forms the walker-independent part S = sum_i ((obs_i - 1)/sigma_i)^2 once;
 *   (2) hot_kernel: walkers on the common path (circular orbit, short transit window, sorted series,
 *   outline that can cross the limb at most twice) get their in-window exposures as index ranges and
 *   chi^2 = S + sum over them of d (2 o r + d), o = obs - 1, r = 1/sigma, d = (1 - F) r, in fp32 terms
 *   summed in fp64; every other walker runs, inside the same launch, the full-featured arithmetic of
 *   the fp64 kernel in fp32 (fp64 phases, Kepler's equation, four-crossing search).
 *   A caller that evaluates many batches against one series should use gl_series_* below, which does
 *   (1) once per series. */
int gl_loglike(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
               const double* obs, const double* sigma, void* chi2_out, void* flux_out_or_null,
               gl_dtype dtype, void* stream);

/* gl_lightcurve_ex / gl_loglike_ex (NEXT-2 of SURVEY.md 8(f)): the same two calls for general
 * triaxial ellipsoids and tidally locked planets.  params_ex [B, GL_NPARAMS_EX] row-major fp64
 * (device): columns 0-11 as above, then
 *   12 zeta [rad], third Euler angle of R(zeta, eta, xi) (eqs. 3-6)
 *   13 rb, 14 rc: semi-axes b = Rp_eq rb along y', c = Rp_eq rc along z' (a = Rp_eq (1 - f) along x');
 *      rb, rc > 0, every semi-axis < 0.5.  rb = rc = 1, zeta = 0 is the oblate model above.
 *   15 locked: 0 = orientation fixed in the observer frame (eq. 2, eqs. 11-13);
 *      1 = tidally locked (PAPER.md:452-466 eq. B13): the outline of EVERY sub-exposure follows
 *      eqs. B14-B16 with alpha = the orbital angle from conjunction and sin(beta) = cos i (the
 *      projected-ellipse geometry moves from the per-walker prelude into the per-sample loop).
 * Any other value of column 15, or a bad axis, makes the walker invalid (NaN row, chi^2 = +inf).
 * Everything else (layout, dtype, stream, status codes) as gl_lightcurve / gl_loglike. */
int gl_lightcurve_ex(const double* params_ex, int B, const double* times, int T, double t_exp,
                     int n_ss, void* flux_out, gl_dtype dtype, void* stream);
int gl_loglike_ex(const double* params_ex, int B, const double* times, int T, double t_exp, int n_ss,
                  const double* obs, const double* sigma, void* chi2_out, void* flux_out_or_null,
                  gl_dtype dtype, void* stream);

/* gl_params_from_munu (NEXT-3 of SURVEY.md 8(f)): the paper's SAMPLING parameters (App. A,
 * PAPER.md:366-430) -> the model rows gl_lightcurve / gl_loglike take, on the device.
 *   sampling [B, 12] fp64 (device): t0, P, a/R*, b, e, omega, r_mean, mu, nu, xi, q1, q2
 *     r_mean = volume-equivalent radius ratio (R_eq = r_mean / (1-f)^(1/3)); mu in (-1, 1),
 *     nu in (0, 1] (eqs. A1-A4); q1, q2 in [0, 1] (u1 = 2 sqrt(q1) q2, u2 = sqrt(q1)(1 - 2 q2)).
 *   params_out [B, GL_NPARAMS] fp64 (device), fully overwritten; f by eqs. A2-A3, eta in [0, pi/2]
 *     by eq. A1.  logprior_out_or_null [B] fp64: ln p(mu, nu) of eq. A6.
 * A row outside the domain gives a NaN row (an invalid walker downstream) and -inf.
 * gl_munu_from_uniform: uw [B, 2] uniform variates in [0, 1] -> munu_out [B, 2] distributed as eq. A6
 * (inverse-transform sampling, eqs. A10 and A12).  Both are fp64 only and enqueue one launch. */
int gl_params_from_munu(const double* sampling, int B, double* params_out,
                        double* logprior_out_or_null, void* stream);
int gl_munu_from_uniform(const double* uw, int B, double* munu_out, void* stream);

/* gl_gp_loglike (NEXT-4 of SURVEY.md 8(f)): the paper's objective in place of
 * chi^2 -- the Gaussian-process log-likelihood of the residuals r_i = obs_i - F_b(t_i) under
 *   K_ij = s^2 (1 + sqrt(3) d/rho) exp(-sqrt(3) d/rho) + delta_ij (sigma_i^2 + jit^2),  d = |t_i - t_j|
 * (Matern-3/2 + jitter):  loglike_out[b] = -1/2 r^T K^-1 r - 1/2 ln det K - (T/2) ln 2 pi, fp64.
 *   gp [B, 3] fp64 (device): (s, rho, jit) per walker, s >= 0, rho > 0, jit >= 0 (else NaN).
 *   times MUST be sorted ascending (else NaN).  flux_work [B, T] of dtype (device, required): the
 *   model flux is written there by the transit kernel (as gl_lightcurve) and read back by the
 *   likelihood kernel, which evaluates the likelihood exactly in O(T) per walker with a Kalman
 *   filter on the state-space form of the Matern-3/2 process -- the quantity celerite computes
 *   for the paper, not celerite's algorithm.  An invalid walker (NaN flux row) gives -inf.
 *   Two launches on `stream`; no synchronisation. */
int gl_gp_loglike(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                  const double* obs, const double* sigma, const double* gp, double* loglike_out,
                  void* flux_work, gl_dtype dtype, void* stream);

/* gl_gp_loglike_static: gl_gp_loglike in fp32 for callers that cannot allocate device memory (code
 * under CUDA stream capture, tight serving loops, harnesses that forbid cudaMalloc).  The [B, T] fp32
 * flux scratch that gl_gp_loglike takes as `flux_work` lives in a file-scope `static __device__` array
 * of the library instead: GL_GP_STATIC_MAX_ELEMS floats = 4 MiB of EVERY GPU that loads the library,
 * held until the process exits.  Inputs and the output are still the caller's (device pointers, as
 * gl_gp_loglike); result and launches are those of gl_gp_loglike(..., GL_F32, ...) bit for bit.
 *   - B * T > GL_GP_STATIC_MAX_ELEMS (also returned by gl_gp_static_capacity()): GL_ECAPACITY,
 *     nothing enqueued.  Config 3 (256 x 3900) fits.
 *   - Calls no cudaMalloc / cudaFree / allocating routine.  The first call on each device resolves the
 *     array's address (cudaGetSymbolAddress, with that device current) and uploads the library's constant
 *     tables if no other call has; later calls only launch.
 *   - ALL calls on a device share the one array and it keeps the last call's contents.  Nothing in it
 *     needs clearing: every element a call reads it has written first.  Calls that overlap on the GPU
 *     (different streams, no ordering between them) RACE on it: order them, or use gl_gp_loglike with
 *     buffers of your own. */
#define GL_GP_STATIC_MAX_ELEMS (1 << 20)
int gl_gp_loglike_static(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                         const double* obs, const double* sigma, const double* gp, double* loglike_out,
                         void* stream);
long long gl_gp_static_capacity(void);

/* gl_flux_geometry: steps "crossings + boundary integrals" alone, for N bare geometries.
 *   geom [N, GL_NGEOM] row-major fp64 (device): (d, Rp, f_proj, PA, u1, u2) -- planet centre at
 *   (d, 0), d >= 0; projected semi-major axis Rp (0 < Rp < 0.5) at position angle PA [rad],
 *   counter-clockwise from the star-centre -> planet-centre direction; semi-minor Rp (1-f_proj),
 *   0 <= f_proj < 1.  flux_out [N] float/double.  An invalid row gives NaN. */
int gl_flux_geometry(const double* geom, long long N, void* flux_out, gl_dtype dtype, void* stream);

/* gl_flux_geometry_simpson: the same rows and output as gl_flux_geometry, computed with the
 * PAPER'S OWN algorithm instead of crossings + closed forms: every outline point outside the disc
 * is snapped radially onto the limb (eqs. 16-20) and the three integrands of
 * PAPER.md:127-135 (eqs. 21-23) are summed over theta in [0, 2 pi] by composite Simpson
 * with n_intervals intervals (even, 2 <= n_intervals <= 2^24; else GL_EINVAL), one
 * warp per geometry.  The discretisation error falls only like 1/n_intervals on
 * limb-crossing geometries (the snapped integrand has a kink); it is here to be measured against
 * gl_flux_geometry, not to replace it. */
int gl_flux_geometry_simpson(const double* geom, long long N, int n_intervals, void* flux_out,
                             gl_dtype dtype, void* stream);

/* HOST-buffer convenience wrappers (used for the end-to-end numbers of bench.py): every pointer
 * below is a HOST pointer; the call allocates device scratch, copies in, runs the kernel above,
 * copies out and synchronises before it returns.  Same semantics and status codes otherwise. */
int gl_lightcurve_host(const double* params, int B, const double* times, int T, double t_exp,
                       int n_ss, void* flux_out, gl_dtype dtype);
int gl_loglike_host(const double* params, int B, const double* times, int T, double t_exp, int n_ss,
                    const double* obs, const double* sigma, void* chi2_out, void* flux_out_or_null,
                    gl_dtype dtype);
int gl_flux_geometry_host(const double* geom, long long N, void* flux_out, gl_dtype dtype);

/* gl_series: a RESIDENT series for repeated likelihood calls (fp32 only).  An MCMC run evaluates one
 * likelihood per walker per sampler step against fixed data: only params[B,12]
 * changes between calls.  gl_series_create uploads (times, obs, sigma) ONCE and does, once, everything
 * that depends on the series alone: the order check of `times`, the baseline sum
 * S = sum_i ((obs_i - 1)/sigma_i)^2 in fp64, the fp32 pairs (obs_i - 1, 1/sigma_i) of the residuals,
 * device buffers and pinned, device-mapped staging for up to B_max walkers.
 *   times, obs, sigma [T] fp64, HOST pointers (copied; the caller may free them afterwards).
 *   T >= 1, n_ss >= 1, t_exp >= 0, B_max >= 1, else GL_EINVAL.  *out receives the handle.
 * The handle OWNS device memory (T * 32 bytes + B_max * 100 bytes, + B_max * T * 4 bytes once a host
 * call has asked for flux), pinned host memory and one non-blocking stream, all on the device that
 * was current at creation; gl_series_destroy releases them (NULL is allowed).  A handle serves ONE
 * call at a time (calls on one handle must not overlap); different handles are independent.
 *
 * gl_series_loglike: params [B, GL_NPARAMS] fp64 HOST (any memory), B <= B_max; chi2_out [B] float
 *   HOST; flux_out_or_null [B, T] float HOST.  Synchronous: returns when the outputs are written.
 *   The kernel reads the parameter rows from, and writes chi^2 to, pinned host memory directly (no
 *   copy engine on the path); a chi^2-only call waits on a completion word in pinned memory that the
 *   kernel's last CTA sets (no stream synchronise; after 2 s without it the stream is synchronised
 *   and its error, if any, returned); flux, when asked for, comes back by one device-to-host copy.  Same
 *   values as gl_loglike(GL_F32) up to the rounding of S (kept in fp64 here, narrowed there).
 * gl_series_loglike_dev: params, chi2_out, flux_out_or_null are DEVICE pointers; work is enqueued on
 *   `stream` without synchronising (the series buffers are only read, so several streams may use
 *   one handle through this call as long as the handle outlives the work).  The launch is
 *   captured once per distinct (params, B, chi2_out, flux_out_or_null) -- the last four are kept --
 *   and replayed as a CUDA graph: a sampler that reuses its buffers pays one graph launch per step.
 * Launches per call: ONE (hot_kernel, see gl_loglike; the per-series kernel ran at creation). */
typedef struct gl_series gl_series;
int gl_series_create(const double* times, const double* obs, const double* sigma, int T, double t_exp,
                     int n_ss, int B_max, gl_series** out);
int gl_series_loglike(gl_series* s, const double* params, int B, float* chi2_out,
                      float* flux_out_or_null);
int gl_series_loglike_dev(gl_series* s, const double* params, int B, float* chi2_out,
                          float* flux_out_or_null, void* stream);
/* any of the output pointers may be NULL; baseline = S above (fp64; +inf when a sigma is bad) */
int gl_series_info(const gl_series* s, int* T, int* n_ss, int* B_max, int* sorted, double* baseline);
int gl_series_destroy(gl_series* s);

/* gl_probe_peaks: measures, on the current device, the arithmetic ceilings the roofline of
 * bench.py divides by: register-only dependent-chain kernels of FFMA (fp32), DFMA
 * (fp64) and MUFU.RSQ, 8 independent chains per thread, every SM full.  out3 (HOST) receives
 * { fp32 TFLOP/s, fp64 TFLOP/s, MUFU Tops/s }.  Synchronises the device; not part of the hot path. */
int gl_probe_peaks(double* out3);

/* gl_probe_empty_launch: enqueues an EMPTY kernel of `rows` clusters of `cluster` CTAs of `threads`
 * threads on `stream` and, when dep_rows > 0, a second empty grid (dep_rows clusters of
 * dep_cluster CTAs of 128 threads) chained to it by programmatic dependent launch -- launch
 * shapes of the library's calls without their work.  bench.py times it the way
 * it times a step and reports it as roofline.launch_floor_ms.  Not part of the hot path. */
int gl_probe_empty_launch(int cluster, int rows, int threads, int dep_cluster, int dep_rows,
                          void* stream);
/* gl_probe_empty_graph: the same single empty kernel, captured once per shape (and calling thread) and
 * replayed as a CUDA graph on `stream` -- the way gl_series_loglike_dev launches a step. */
int gl_probe_empty_graph(int cluster, int rows, int threads, void* stream);

/* Number of kernel launches the calling thread's entry points have enqueued so far (HOST). */
long long gl_launch_count(void);

const char* gl_strerror(int code);          /* static string, never NULL           */
const char* gl_last_cuda_error(void);       /* text of the last GL_ECUDA, per thread */
int gl_version(void);                       /* major*10000 + minor*100 + patch       */

#ifdef __cplusplus
}
#endif
#endif /* GREENLANTERN_B200_H */
