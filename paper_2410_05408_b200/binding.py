"""Thin ctypes binding over the C ABI of include/greenlantern_b200.h.

Argument marshalling only: every step of the path runs inside the CUDA library.  torch is used
for device memory and streams.  There is NO CPU fallback: if the shared library is missing or a
tensor is not on a CUDA device, the call raises.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np

GL_F32, GL_F64 = 0, 1
GL_NPARAMS, GL_NGEOM, GL_NPARAMS_EX = 12, 6, 16
_LIBPATH = Path(__file__).resolve().parent / "csrc" / "libgreenlantern_b200.so"
_lib = None

EXPORTS = ("gl_lightcurve", "gl_loglike", "gl_lightcurve_ex", "gl_loglike_ex", "gl_params_from_munu", "gl_munu_from_uniform", "gl_gp_loglike", "gl_gp_loglike_static", "gl_gp_static_capacity", "gl_flux_geometry", "gl_flux_geometry_simpson", "gl_lightcurve_host",
           "gl_loglike_host", "gl_flux_geometry_host", "gl_series_create", "gl_series_loglike",
           "gl_series_loglike_dev", "gl_series_info", "gl_series_destroy", "gl_probe_peaks",
           "gl_probe_empty_launch", "gl_probe_empty_graph", "gl_launch_count", "gl_strerror",
           "gl_last_cuda_error", "gl_version")


class GreenlanternError(RuntimeError):
    pass


def load_library():
    """dlopen csrc/libgreenlantern_b200.so (built by paper_2410_05408_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIBPATH.exists():
        raise GreenlanternError(
            f"{_LIBPATH} is missing: run `python -m paper_2410_05408_b200.build` (needs nvcc). "
            "There is no CPU fallback.")
    lib = ctypes.CDLL(str(_LIBPATH))
    vp, i, d, ll = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_longlong
    lib.gl_lightcurve.argtypes = [vp, i, vp, i, d, i, vp, i, vp]
    lib.gl_loglike.argtypes = [vp, i, vp, i, d, i, vp, vp, vp, vp, i, vp]
    lib.gl_lightcurve_ex.argtypes = lib.gl_lightcurve.argtypes
    lib.gl_loglike_ex.argtypes = lib.gl_loglike.argtypes
    lib.gl_lightcurve_ex.restype = lib.gl_loglike_ex.restype = i
    lib.gl_params_from_munu.argtypes = [vp, i, vp, vp, vp]
    lib.gl_munu_from_uniform.argtypes = [vp, i, vp, vp]
    lib.gl_params_from_munu.restype = lib.gl_munu_from_uniform.restype = i
    lib.gl_gp_loglike.argtypes = [vp, i, vp, i, d, i, vp, vp, vp, vp, vp, i, vp]
    lib.gl_gp_loglike.restype = i
    lib.gl_gp_loglike_static.argtypes = [vp, i, vp, i, d, i, vp, vp, vp, vp, vp]
    lib.gl_gp_loglike_static.restype = i
    lib.gl_gp_static_capacity.argtypes = []
    lib.gl_gp_static_capacity.restype = ll
    lib.gl_flux_geometry.argtypes = [vp, ll, vp, i, vp]
    lib.gl_flux_geometry_simpson.argtypes = [vp, ll, i, vp, i, vp]
    lib.gl_flux_geometry_simpson.restype = i
    lib.gl_lightcurve_host.argtypes = [vp, i, vp, i, d, i, vp, i]
    lib.gl_loglike_host.argtypes = [vp, i, vp, i, d, i, vp, vp, vp, vp, i]
    lib.gl_flux_geometry_host.argtypes = [vp, ll, vp, i]
    for name in ("gl_lightcurve", "gl_loglike", "gl_flux_geometry", "gl_lightcurve_host",
                 "gl_loglike_host", "gl_flux_geometry_host", "gl_version"):
        getattr(lib, name).restype = i
    lib.gl_series_create.argtypes = [vp, vp, vp, i, d, i, i, ctypes.POINTER(vp)]
    lib.gl_series_loglike.argtypes = [vp, vp, i, vp, vp]
    lib.gl_series_loglike_dev.argtypes = [vp, vp, i, vp, vp, vp]
    lib.gl_series_info.argtypes = [vp, ctypes.POINTER(i), ctypes.POINTER(i), ctypes.POINTER(i),
                                   ctypes.POINTER(i), ctypes.POINTER(d)]
    lib.gl_series_destroy.argtypes = [vp]
    for name in ("gl_series_create", "gl_series_loglike", "gl_series_loglike_dev", "gl_series_info",
                 "gl_series_destroy"):
        getattr(lib, name).restype = i
    lib.gl_probe_empty_launch.argtypes = [i, i, i, i, i, vp]
    lib.gl_probe_empty_launch.restype = i
    lib.gl_probe_empty_graph.argtypes = [i, i, i, vp]
    lib.gl_probe_empty_graph.restype = i
    lib.gl_probe_peaks.argtypes = [vp]
    lib.gl_probe_peaks.restype = i
    lib.gl_launch_count.restype = ll
    lib.gl_strerror.argtypes = [i]
    lib.gl_strerror.restype = ctypes.c_char_p
    lib.gl_last_cuda_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(rc):
    if rc != 0:
        lib = load_library()
        msg = lib.gl_strerror(rc).decode()
        if rc == -2:
            msg += ": " + lib.gl_last_cuda_error().decode()
        raise GreenlanternError(f"greenlantern_b200 status {rc}: {msg}")


def _torch():
    import torch
    return torch


def _dev_f64(x, shape_tail=None):
    torch = _torch()
    if not isinstance(x, torch.Tensor) or not x.is_cuda:
        raise GreenlanternError("expected a CUDA torch.Tensor (no CPU fallback exists)")
    if x.dtype != torch.float64 or not x.is_contiguous():
        raise GreenlanternError("inputs must be contiguous float64 tensors")
    if shape_tail is not None and (x.dim() != 2 or x.shape[1] != shape_tail):
        raise GreenlanternError(f"expected shape [*, {shape_tail}]")
    return x


def _tdtype(dtype):
    torch = _torch()
    if dtype in (GL_F32, "f32", "float32", torch.float32):
        return GL_F32, torch.float32
    if dtype in (GL_F64, "f64", "float64", torch.float64):
        return GL_F64, torch.float64
    raise GreenlanternError(f"unknown dtype {dtype!r}")


def _stream(x):
    return ctypes.c_void_p(_torch().cuda.current_stream(x.device).cuda_stream)


def gl_lightcurve(params, times, t_exp=0.0, n_ss=1, dtype="f32", out=None):
    """flux[B, T] for params[B, 12] and times[T] (device tensors, fp64)."""
    return _lightcurve("gl_lightcurve", GL_NPARAMS, params, times, t_exp, n_ss, dtype, out)


def gl_lightcurve_ex(params_ex, times, t_exp=0.0, n_ss=1, dtype="f32", out=None):
    """flux[B, T] for the extended rows params_ex[B, 16] (triaxial / tidally locked, NEXT-2)."""
    return _lightcurve("gl_lightcurve_ex", GL_NPARAMS_EX, params_ex, times, t_exp, n_ss, dtype, out)


def _lightcurve(fname, width, params, times, t_exp, n_ss, dtype, out):
    torch = _torch()
    lib = load_library()
    params, times = _dev_f64(params, width), _dev_f64(times)
    code, td = _tdtype(dtype)
    B, T = params.shape[0], times.shape[0]
    if out is None:
        out = torch.empty((B, T), dtype=td, device=params.device)
    with torch.cuda.device(params.device):
        _check(getattr(lib, fname)(params.data_ptr(), B, times.data_ptr(), T, float(t_exp),
                                   int(n_ss), out.data_ptr(), code, _stream(params)))
    return out


def gl_loglike(params, times, t_exp, n_ss, obs, sigma, dtype="f32", want_flux=False):
    """chi2[B] (and flux[B, T] when want_flux) -- one fused launch."""
    return _loglike("gl_loglike", GL_NPARAMS, params, times, t_exp, n_ss, obs, sigma, dtype, want_flux)


def gl_loglike_ex(params_ex, times, t_exp, n_ss, obs, sigma, dtype="f32", want_flux=False):
    """gl_loglike for the extended rows params_ex[B, 16] (triaxial / tidally locked, NEXT-2)."""
    return _loglike("gl_loglike_ex", GL_NPARAMS_EX, params_ex, times, t_exp, n_ss, obs, sigma, dtype,
                    want_flux)


def _loglike(fname, width, params, times, t_exp, n_ss, obs, sigma, dtype, want_flux):
    torch = _torch()
    lib = load_library()
    params, times = _dev_f64(params, width), _dev_f64(times)
    obs, sigma = _dev_f64(obs), _dev_f64(sigma)
    code, td = _tdtype(dtype)
    B, T = params.shape[0], times.shape[0]
    if obs.shape[0] != T or sigma.shape[0] != T:
        raise GreenlanternError("obs and sigma must have the length of times")
    chi2 = torch.empty((B,), dtype=td, device=params.device)
    flux = torch.empty((B, T), dtype=td, device=params.device) if want_flux else None
    with torch.cuda.device(params.device):
        _check(getattr(lib, fname)(params.data_ptr(), B, times.data_ptr(), T, float(t_exp),
                                   int(n_ss), obs.data_ptr(), sigma.data_ptr(), chi2.data_ptr(),
                                   flux.data_ptr() if want_flux else None, code, _stream(params)))
    return (chi2, flux) if want_flux else chi2


def gl_params_from_munu(sampling, want_logprior=True):
    """Sampling rows [B, 12] (t0, P, a/R*, b, e, omega, r_mean, mu, nu, xi, q1, q2; App. A of the paper)
    -> model rows [B, 12] (and ln p(mu, nu) [B])."""
    torch = _torch()
    lib = load_library()
    sampling = _dev_f64(sampling, GL_NPARAMS)
    B = sampling.shape[0]
    params = torch.empty((B, GL_NPARAMS), dtype=torch.float64, device=sampling.device)
    lp = torch.empty((B,), dtype=torch.float64, device=sampling.device) if want_logprior else None
    with torch.cuda.device(sampling.device):
        _check(lib.gl_params_from_munu(sampling.data_ptr(), B, params.data_ptr(),
                                       lp.data_ptr() if want_logprior else None, _stream(sampling)))
    return (params, lp) if want_logprior else params


def gl_munu_from_uniform(uw):
    """[B, 2] uniform variates -> [B, 2] (mu, nu) distributed as eq. A6 of the paper."""
    torch = _torch()
    lib = load_library()
    uw = _dev_f64(uw, 2)
    out = torch.empty_like(uw)
    with torch.cuda.device(uw.device):
        _check(lib.gl_munu_from_uniform(uw.data_ptr(), uw.shape[0], out.data_ptr(), _stream(uw)))
    return out


def gl_gp_loglike(params, times, t_exp, n_ss, obs, sigma, gp, dtype="f32", want_flux=False):
    """ln L[B] (fp64) of the residuals under a Matern-3/2 + jitter Gaussian process (NEXT-4);
    gp[B, 3] = (amplitude, timescale, jitter); times sorted ascending."""
    torch = _torch()
    lib = load_library()
    params, times = _dev_f64(params, GL_NPARAMS), _dev_f64(times)
    obs, sigma, gp = _dev_f64(obs), _dev_f64(sigma), _dev_f64(gp, 3)
    code, td = _tdtype(dtype)
    B, T = params.shape[0], times.shape[0]
    if obs.shape[0] != T or sigma.shape[0] != T or gp.shape[0] != B:
        raise GreenlanternError("obs, sigma must have the length of times and gp one row per walker")
    out = torch.empty((B,), dtype=torch.float64, device=params.device)
    flux = torch.empty((B, T), dtype=td, device=params.device)
    with torch.cuda.device(params.device):
        _check(lib.gl_gp_loglike(params.data_ptr(), B, times.data_ptr(), T, float(t_exp), int(n_ss),
                                 obs.data_ptr(), sigma.data_ptr(), gp.data_ptr(), out.data_ptr(),
                                 flux.data_ptr(), code, _stream(params)))
    return (out, flux) if want_flux else out


def gl_gp_static_capacity():
    """Largest B * T gl_gp_loglike_static accepts (elements of its file-scope fp32 scratch array)."""
    return int(load_library().gl_gp_static_capacity())


def gl_gp_loglike_static(params, times, t_exp, n_ss, obs, sigma, gp, out=None):
    """gl_gp_loglike in fp32 with the flux scratch inside the library (no device allocation by the
    library; B * T <= gl_gp_static_capacity(), else GreenlanternError).  `out`: optional preallocated
    CUDA float64 [B] tensor, so that the call allocates nothing at all.  Calls that overlap on the GPU
    share the scratch and race: keep them on one stream."""
    torch = _torch()
    lib = load_library()
    params, times = _dev_f64(params, GL_NPARAMS), _dev_f64(times)
    obs, sigma, gp = _dev_f64(obs), _dev_f64(sigma), _dev_f64(gp, 3)
    B, T = params.shape[0], times.shape[0]
    if obs.shape[0] != T or sigma.shape[0] != T or gp.shape[0] != B:
        raise GreenlanternError("obs, sigma must have the length of times and gp one row per walker")
    if out is None:
        out = torch.empty((B,), dtype=torch.float64, device=params.device)
    elif not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and tuple(out.shape) == (B,)):
        raise GreenlanternError(f"out must be a contiguous CUDA float64 tensor of shape ({B},)")
    with torch.cuda.device(params.device):
        _check(lib.gl_gp_loglike_static(params.data_ptr(), B, times.data_ptr(), T, float(t_exp), int(n_ss),
                                        obs.data_ptr(), sigma.data_ptr(), gp.data_ptr(), out.data_ptr(),
                                        _stream(params)))
    return out


def gl_flux_geometry(geom, dtype="f32"):
    """flux[N] for rows (d, Rp, f_proj, PA, u1, u2) (device tensor, fp64)."""
    torch = _torch()
    lib = load_library()
    geom = _dev_f64(geom, GL_NGEOM)
    code, td = _tdtype(dtype)
    out = torch.empty((geom.shape[0],), dtype=td, device=geom.device)
    with torch.cuda.device(geom.device):
        _check(lib.gl_flux_geometry(geom.data_ptr(), geom.shape[0], out.data_ptr(), code,
                                    _stream(geom)))
    return out


def gl_flux_geometry_simpson(geom, n_intervals, dtype="f32"):
    """The paper's snap + Simpson algorithm (NEXT-1) on [N, 6] geometry rows; one warp per row."""
    torch = _torch()
    lib = load_library()
    geom = _dev_f64(geom, GL_NGEOM)
    code, td = _tdtype(dtype)
    out = torch.empty((geom.shape[0],), dtype=td, device=geom.device)
    with torch.cuda.device(geom.device):
        _check(lib.gl_flux_geometry_simpson(geom.data_ptr(), geom.shape[0], int(n_intervals),
                                            out.data_ptr(), code, _stream(geom)))
    return out


def _host_f64(x):
    return np.ascontiguousarray(x, dtype=np.float64)


_C_CHAR = ctypes.c_char


def _addr(a):
    """Address of a numpy array's first byte.  `a.ctypes.data` builds a helper object per call (~2 us);
    the buffer-protocol route is several times cheaper and matters for the 20-us host call."""
    try:
        return ctypes.addressof(_C_CHAR.from_buffer(a))
    except (TypeError, ValueError, BufferError):      # read-only or empty arrays
        return a.ctypes.data


def _host_out(out, shape, nd):
    """A caller-supplied HOST output buffer (e.g. pinned memory), checked, or a fresh array."""
    if out is None:
        return np.empty(shape, dtype=nd)
    if not (isinstance(out, np.ndarray) and out.dtype == nd and out.shape == tuple(shape)
            and out.flags["C_CONTIGUOUS"] and out.flags["WRITEABLE"]):
        raise GreenlanternError(f"out must be a writable C-contiguous {nd.__name__}{tuple(shape)} array")
    return out


def gl_loglike_host(params, times, t_exp, n_ss, obs, sigma, dtype="f32", want_flux=False,
                    chi2_out=None, flux_out=None):
    """HOST numpy in, HOST numpy out; the library does the copies (end-to-end path).
    chi2_out / flux_out: optional preallocated HOST arrays (pinned memory makes the D2H copy
    asynchronous and fast)."""
    lib = load_library()
    params, times, obs, sigma = map(_host_f64, (np.atleast_2d(params), times, obs, sigma))
    code = GL_F64 if dtype in (GL_F64, "f64", "float64") else GL_F32
    nd = np.float64 if code == GL_F64 else np.float32
    B, T = params.shape[0], times.shape[0]
    chi2 = _host_out(chi2_out, (B,), nd)
    flux = _host_out(flux_out, (B, T), nd) if want_flux else None
    _check(lib.gl_loglike_host(params.ctypes.data, B, times.ctypes.data, T, float(t_exp),
                               int(n_ss), obs.ctypes.data, sigma.ctypes.data, chi2.ctypes.data,
                               flux.ctypes.data if want_flux else None, code))
    return (chi2, flux) if want_flux else chi2


def gl_lightcurve_host(params, times, t_exp=0.0, n_ss=1, dtype="f32"):
    lib = load_library()
    params, times = _host_f64(np.atleast_2d(params)), _host_f64(times)
    code = GL_F64 if dtype in (GL_F64, "f64", "float64") else GL_F32
    flux = np.empty((params.shape[0], times.shape[0]),
                    dtype=np.float64 if code == GL_F64 else np.float32)
    _check(lib.gl_lightcurve_host(params.ctypes.data, params.shape[0], times.ctypes.data,
                                  times.shape[0], float(t_exp), int(n_ss), flux.ctypes.data, code))
    return flux


def gl_flux_geometry_host(geom, dtype="f32"):
    lib = load_library()
    geom = _host_f64(np.atleast_2d(geom))
    code = GL_F64 if dtype in (GL_F64, "f64", "float64") else GL_F32
    out = np.empty(geom.shape[0], dtype=np.float64 if code == GL_F64 else np.float32)
    _check(lib.gl_flux_geometry_host(geom.ctypes.data, geom.shape[0], out.ctypes.data, code))
    return out


class GlSeries:
    """A resident series (gl_series_* of the C ABI): upload times/obs/sigma once, then evaluate
    chi^2 for many parameter batches.  ``loglike`` takes HOST numpy arrays and is synchronous;
    ``loglike_dev`` takes CUDA tensors and enqueues on torch's current stream."""

    def __init__(self, times, obs, sigma, t_exp, n_ss, B_max, device=None):
        lib = load_library()
        times, obs, sigma = map(_host_f64, (times, obs, sigma))
        if not (times.ndim == 1 and obs.shape == times.shape and sigma.shape == times.shape):
            raise GreenlanternError("times, obs and sigma must be 1-d arrays of one length")
        self._h = ctypes.c_void_p()
        self._loglike = lib.gl_series_loglike
        self._p_obj = self._p_shape = self._p_addr = self._c_obj = self._c_addr = None
        self.T, self.B_max = int(times.shape[0]), int(B_max)
        self._device = device
        if device is not None:
            with _torch().cuda.device(device):
                rc = lib.gl_series_create(times.ctypes.data, obs.ctypes.data, sigma.ctypes.data, self.T,
                                          float(t_exp), int(n_ss), self.B_max, ctypes.byref(self._h))
        else:
            rc = lib.gl_series_create(times.ctypes.data, obs.ctypes.data, sigma.ctypes.data, self.T,
                                      float(t_exp), int(n_ss), self.B_max, ctypes.byref(self._h))
        _check(rc)

    def info(self):
        i, d = ctypes.c_int, ctypes.c_double
        T, S, Bm, so, base = i(), i(), i(), i(), d()
        _check(load_library().gl_series_info(self._h, ctypes.byref(T), ctypes.byref(S), ctypes.byref(Bm),
                                             ctypes.byref(so), ctypes.byref(base)))
        return {"T": T.value, "n_ss": S.value, "B_max": Bm.value, "sorted": bool(so.value),
                "baseline": base.value}

    def loglike(self, params, want_flux=False, chi2_out=None, flux_out=None):
        # An MCMC loop calls this every ~20 us with the SAME arrays: the checks and the address look-ups of
        # the last params / chi2_out objects are remembered (a reference is held, so identity means the same
        # live buffer; the shape is compared again because it can be reassigned in place).
        if params is self._p_obj and params.shape == self._p_shape:
            paddr, B = self._p_addr, self._p_shape[0]
        else:
            obj = params
            if not (type(params) is np.ndarray and params.ndim == 2 and params.dtype == np.float64
                    and params.flags.c_contiguous):
                params = _host_f64(np.atleast_2d(params))
            if params.shape[1] != GL_NPARAMS:
                raise GreenlanternError(f"expected shape [*, {GL_NPARAMS}]")
            paddr, B = _addr(params), params.shape[0]
            if obj is params:      # (a converted copy is not worth remembering)
                self._p_obj, self._p_shape, self._p_addr = params, params.shape, paddr
        if chi2_out is not None and chi2_out is self._c_obj and chi2_out.shape == (B,):
            chi2, caddr = chi2_out, self._c_addr
        else:
            chi2 = _host_out(chi2_out, (B,), np.float32)
            caddr = _addr(chi2)
            if chi2_out is not None:
                self._c_obj, self._c_addr = chi2, caddr
        flux = _host_out(flux_out, (B, self.T), np.float32) if want_flux else None
        _check(self._loglike(self._h, paddr, B, caddr, _addr(flux) if want_flux else None))
        return (chi2, flux) if want_flux else chi2

    def loglike_dev(self, params, want_flux=False, chi2_out=None, flux_out=None):
        torch = _torch()
        params = _dev_f64(params, GL_NPARAMS)
        B = params.shape[0]
        chi2 = chi2_out if chi2_out is not None else torch.empty((B,), dtype=torch.float32, device=params.device)
        flux = None
        if want_flux:
            flux = flux_out if flux_out is not None else torch.empty((B, self.T), dtype=torch.float32,
                                                                     device=params.device)
        for t, shape in ((chi2, (B,)), (flux, (B, self.T))):
            if t is not None and not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
                                      and tuple(t.shape) == shape):
                raise GreenlanternError(f"output must be a contiguous CUDA float32 tensor of shape {shape}")
        with torch.cuda.device(params.device):
            _check(load_library().gl_series_loglike_dev(self._h, params.data_ptr(), B, chi2.data_ptr(),
                                                        flux.data_ptr() if want_flux else None,
                                                        _stream(params)))
        return (chi2, flux) if want_flux else chi2

    def close(self):
        if self._h:
            _check(load_library().gl_series_destroy(self._h))
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def gl_probe_peaks():
    """{fp32 TFLOP/s, fp64 TFLOP/s, MUFU Tops/s} of the current device (FMA / MUFU chain kernels)."""
    out = (ctypes.c_double * 3)()
    _check(load_library().gl_probe_peaks(out))
    return {"fp32_tflops": out[0], "fp64_tflops": out[1], "mufu_tops": out[2]}


def gl_probe_empty_launch(cluster, rows, threads, dep_cluster=1, dep_rows=0, device=None):
    """Enqueue an empty kernel of the given shape (and, optionally, a dependent empty grid) on torch's
    current stream: the launch floor bench.py reports."""
    torch = _torch()
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else device
    st = ctypes.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
    _check(load_library().gl_probe_empty_launch(int(cluster), int(rows), int(threads), int(dep_cluster),
                                                int(dep_rows), st))


def gl_probe_empty_graph(cluster, rows, threads, device=None):
    """The empty kernel of gl_probe_empty_launch replayed as a CUDA graph on torch's current stream."""
    torch = _torch()
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else device
    st = ctypes.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
    _check(load_library().gl_probe_empty_graph(int(cluster), int(rows), int(threads), st))


def gl_launch_count():
    return int(load_library().gl_launch_count())


def gl_version():
    return int(load_library().gl_version())


def gl_strerror(code):
    return load_library().gl_strerror(int(code)).decode()
