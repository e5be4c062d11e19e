"""CPU oracle for the oblate-transit model of arXiv:2410.05408 -- TEST INFRASTRUCTURE ONLY.

A thin numpy/ctypes front end over ``gl_oracle.c`` (plain C, fp64; see that file's
header for the passages it follows and for what pins it).  Nothing in the product
package ``paper_2410_05408_b200`` imports this module, and this module imports
nothing from it.  Allowed callers: ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs.

PARITY UNPINNED (no external pin exists; self-consistency pins only): e>0
orbits, the supersampling convention, chi^2.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gl_oracle.c"
_LIB = _HERE / "libgl_oracle.so"

_dp = ctypes.POINTER(ctypes.c_double)
_lib = None


def build(force: bool = False) -> Path:
    """Compile gl_oracle.c with gcc (-O2, OpenMP) into oracle/libgl_oracle.so."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math",
               "-ffp-contract=off", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        d, i, l = ctypes.c_double, ctypes.c_int, ctypes.c_long
        lib.gl_oracle_rotation.argtypes = [d, d, d, _dp]
        lib.gl_oracle_outline.argtypes = [d, d, d, d, d, d, _dp]
        lib.gl_oracle_outline_locked.argtypes = [d, d, d, d, d, d, d, d, _dp]
        lib.gl_oracle_leggauss.argtypes = [i, _dp, _dp]
        lib.gl_oracle_areas.argtypes = [d, d, d, d, d, _dp]
        lib.gl_oracle_areas.restype = i
        lib.gl_oracle_areas_snap_simpson.argtypes = [d, d, d, d, d, l, _dp]
        lib.gl_oracle_flux_outline.argtypes = [d, d, d, d, d, d, d]
        lib.gl_oracle_flux_outline.restype = d
        lib.gl_oracle_kepler.argtypes = [d, d]
        lib.gl_oracle_kepler.restype = d
        lib.gl_oracle_position.argtypes = [_dp, d, _dp, _dp]
        lib.gl_oracle_position.restype = i
        lib.gl_oracle_params_valid.argtypes = [_dp]
        lib.gl_oracle_params_valid.restype = i
        lib.gl_oracle_flux_time.argtypes = [_dp, d, d, i]
        lib.gl_oracle_flux_time.restype = d
        lib.gl_oracle_lightcurve.argtypes = [_dp, i, _dp, i, d, i, _dp, i]
        lib.gl_oracle_lightcurve_ex.argtypes = [_dp, i, _dp, i, d, i, _dp, i]
        lib.gl_oracle_params_ex_valid.argtypes = [_dp]
        lib.gl_oracle_munu_of.argtypes = [d, d, _dp]
        lib.gl_oracle_feta_of.argtypes = [d, d, _dp]
        lib.gl_oracle_log_prior_munu.argtypes = [d, d]
        lib.gl_oracle_log_prior_munu.restype = d
        lib.gl_oracle_munu_from_uniform.argtypes = [d, d, _dp]
        lib.gl_oracle_params_from_munu.argtypes = [_dp, _dp, _dp]
        lib.gl_oracle_lightcurve.restype = i
        lib.gl_oracle_loglike.argtypes = [_dp, i, _dp, i, d, i, _dp, _dp, _dp, _dp, i]
        lib.gl_oracle_loglike.restype = i
        lib.gl_oracle_flux_geometry.argtypes = [_dp, l, _dp, i]
        lib.gl_oracle_flux_geometry.restype = i
        _lib = lib
    return _lib


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def rotation(zeta, eta, xi):
    """R(zeta,eta,xi) = Rx Ry Rz as a 3x3 array (eq. 6)."""
    out = np.zeros(9)
    _load().gl_oracle_rotation(zeta, eta, xi, out.ctypes.data_as(_dp))
    return out.reshape(3, 3)


def outline(a, b, c, zeta, eta, xi):
    """(dx, dy1, dy2) of eqs. 11-13."""
    out = np.zeros(3)
    _load().gl_oracle_outline(a, b, c, zeta, eta, xi, out.ctypes.data_as(_dp))
    return out


def outline_locked(a, b, c, zeta, eta, xi, alpha, beta):
    """(dx, dy1, dy2) of eqs. B14-B16."""
    out = np.zeros(3)
    _load().gl_oracle_outline_locked(a, b, c, zeta, eta, xi, alpha, beta,
                                     out.ctypes.data_as(_dp))
    return out


def leggauss(n):
    x, w = np.zeros(n), np.zeros(n)
    _load().gl_oracle_leggauss(n, x.ctypes.data_as(_dp), w.ctypes.data_as(_dp))
    return x, w


def areas(x0, y0, dx, dy1, dy2):
    """(A_flat, A_lin, A_quad), n_crossings (or -1 when the overlap is empty)."""
    A = np.zeros(3)
    n = _load().gl_oracle_areas(x0, y0, dx, dy1, dy2, A.ctypes.data_as(_dp))
    return A, n


def areas_snap_simpson(x0, y0, dx, dy1, dy2, N):
    """The paper's literal snap + Simpson algorithm with N intervals."""
    A = np.zeros(3)
    _load().gl_oracle_areas_snap_simpson(x0, y0, dx, dy1, dy2, int(N), A.ctypes.data_as(_dp))
    return A


def flux_outline(x0, y0, dx, dy1, dy2, u1, u2):
    return _load().gl_oracle_flux_outline(x0, y0, dx, dy1, dy2, u1, u2)


def kepler(M, e):
    return _load().gl_oracle_kepler(M, e)


def position(params12, t):
    """(x0, y0, in_front) of the planet centre at time t."""
    p, pp = _c(params12)
    x, y = ctypes.c_double(), ctypes.c_double()
    front = _load().gl_oracle_position(pp, float(t), ctypes.byref(x), ctypes.byref(y))
    return x.value, y.value, bool(front)


def params_valid(params12):
    p, pp = _c(params12)
    return bool(_load().gl_oracle_params_valid(pp))


def flux_time(params12, t, t_exp=0.0, n_ss=1):
    p, pp = _c(params12)
    return _load().gl_oracle_flux_time(pp, float(t), float(t_exp), int(n_ss))


def lightcurve(params, times, t_exp=0.0, n_ss=1, nthreads=0):
    """flux[B,T] (fp64).  ``nthreads`` <= 0 uses every host core."""
    p, pp = _c(np.atleast_2d(params))
    t, tp = _c(times)
    flux = np.empty((p.shape[0], t.shape[0]))
    _load().gl_oracle_lightcurve(pp, p.shape[0], tp, t.shape[0], float(t_exp), int(n_ss),
                                 flux.ctypes.data_as(_dp), int(nthreads))
    return flux


def lightcurve_ex(params16, times, t_exp=0.0, n_ss=1, nthreads=0):
    """flux[B,T] for the extended rows [B,16] of NEXT-2: triaxial and/or tidally locked planets
    (columns 12-15 = zeta, b-axis/Rp_eq, c-axis/Rp_eq, locked flag)."""
    p, pp = _c(np.atleast_2d(params16))
    assert p.shape[1] == 16
    t, tp = _c(times)
    flux = np.empty((p.shape[0], t.shape[0]))
    _load().gl_oracle_lightcurve_ex(pp, p.shape[0], tp, t.shape[0], float(t_exp), int(n_ss),
                                    flux.ctypes.data_as(_dp), int(nthreads))
    return flux


def params_ex_valid(params16):
    p, pp = _c(params16)
    return bool(_load().gl_oracle_params_ex_valid(pp))


def munu_of(f, eta):
    """(mu, nu) of eqs. A1, A4."""
    o = np.zeros(2)
    _load().gl_oracle_munu_of(float(f), float(eta), o.ctypes.data_as(_dp))
    return o


def feta_of(mu, nu):
    """(f, eta) from eqs. A2-A3 and A1 solved for eta in [0, pi/2]."""
    o = np.zeros(2)
    _load().gl_oracle_feta_of(float(mu), float(nu), o.ctypes.data_as(_dp))
    return o


def log_prior_munu(mu, nu):
    """ln p(mu, nu), eq. A6."""
    return _load().gl_oracle_log_prior_munu(float(mu), float(nu))


def munu_from_uniform(u, w):
    """(mu, nu) drawn by inverse-transform sampling, eqs. A10, A12."""
    o = np.zeros(2)
    _load().gl_oracle_munu_from_uniform(float(u), float(w), o.ctypes.data_as(_dp))
    return o


def params_from_munu(sampling):
    """Sampling rows [B,12] (t0,P,a/R*,b,e,omega,r_mean,mu,nu,xi,q1,q2) -> (model rows [B,12],
    ln p(mu,nu) [B])."""
    srows, _ = _c(np.atleast_2d(sampling))
    out = np.empty_like(srows)
    lp = np.empty(srows.shape[0])
    one = np.zeros(1)
    for k in range(srows.shape[0]):
        r, rp = _c(srows[k])
        o = np.zeros(12)
        _load().gl_oracle_params_from_munu(rp, o.ctypes.data_as(_dp), one.ctypes.data_as(_dp))
        out[k], lp[k] = o, one[0]
    return out, lp


def matern32(dt, s, rho):
    """Matern-3/2 covariance s^2 (1 + sqrt(3)|dt|/rho) exp(-sqrt(3)|dt|/rho)."""
    x = np.sqrt(3.0) * np.abs(dt) / rho
    return s * s * (1.0 + x) * np.exp(-x)


def gp_loglike_dense(resid, times, sigma, s, rho, jit):
    """NEXT-4, the plain definition: ln N(resid; 0, K) with
    K = Matern-3/2(s, rho) + diag(sigma^2 + jit^2), by a dense Cholesky factorisation (O(T^3): small T)."""
    r = np.asarray(resid, dtype=np.float64)
    t = np.asarray(times, dtype=np.float64)
    K = matern32(t[:, None] - t[None, :], s, rho) + np.diag(np.asarray(sigma, dtype=np.float64) ** 2 + jit * jit)
    L = np.linalg.cholesky(K)
    z = np.linalg.solve(L, r)            # r^T K^-1 r = |L^-1 r|^2
    return -0.5 * (z @ z) - np.log(np.diag(L)).sum() - 0.5 * r.size * np.log(2.0 * np.pi)


def loglike(params, times, t_exp, n_ss, obs, sigma, nthreads=0, return_threads=False):
    """(chi2[B], flux[B,T]) in fp64."""
    p, pp = _c(np.atleast_2d(params))
    t, tp = _c(times)
    o, op = _c(obs)
    s, sp = _c(sigma)
    flux = np.empty((p.shape[0], t.shape[0]))
    chi2 = np.empty(p.shape[0])
    used = _load().gl_oracle_loglike(pp, p.shape[0], tp, t.shape[0], float(t_exp), int(n_ss),
                                     op, sp, chi2.ctypes.data_as(_dp),
                                     flux.ctypes.data_as(_dp), int(nthreads))
    if return_threads:
        return chi2, flux, used
    return chi2, flux


def flux_geometry(geom, nthreads=0, return_threads=False):
    """flux[N] for rows (d, Rp, f_proj, PA, u1, u2) (config 5)."""
    g, gp = _c(np.atleast_2d(geom))
    out = np.empty(g.shape[0])
    used = _load().gl_oracle_flux_geometry(gp, g.shape[0], out.ctypes.data_as(_dp),
                                           int(nthreads))
    if return_threads:
        return out, used
    return out
