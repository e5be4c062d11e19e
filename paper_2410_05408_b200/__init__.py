"""greenlantern-b200: batched oblate-planet transit light curves on B200 (sm_100a).

The public API is the thin binding in :mod:`paper_2410_05408_b200.binding`
(``gl_lightcurve``, ``gl_loglike``, ``gl_flux_geometry``) over the C-ABI
library ``csrc/libgreenlantern_b200.so`` declared in
``include/greenlantern_b200.h``.  There is no CPU fallback: calling the API
without the built CUDA library raises.
"""
__version__ = "0.1.0"

_API = ("gl_lightcurve", "gl_loglike", "gl_lightcurve_ex", "gl_loglike_ex", "gl_params_from_munu", "gl_munu_from_uniform", "gl_gp_loglike", "gl_gp_loglike_static", "gl_gp_static_capacity", "gl_flux_geometry", "gl_flux_geometry_simpson", "gl_lightcurve_host", "gl_loglike_host",
        "gl_flux_geometry_host", "GlSeries", "gl_probe_peaks", "gl_probe_empty_launch", "gl_probe_empty_graph", "gl_launch_count", "gl_version", "gl_strerror", "load_library",
        "GreenlanternError")


def __getattr__(name):
    if name in _API:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
