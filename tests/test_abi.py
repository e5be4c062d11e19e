"""Host-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/greenlantern_b200.h declares; argument errors are rejected before any CUDA call."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


def declared_symbols():
    text = (ROOT / "include" / "greenlantern_b200.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gl_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2410_05408_b200 import build
    build.build()
    import paper_2410_05408_b200 as g
    return g.load_library()


def test_every_declared_symbol_is_exported(lib):
    syms = declared_symbols()
    assert {"gl_lightcurve", "gl_loglike", "gl_flux_geometry", "gl_strerror", "gl_version"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s


def test_binding_lists_the_same_names():
    from paper_2410_05408_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_argument_errors_need_no_gpu(lib):
    assert lib.gl_version() >= 100
    assert lib.gl_strerror(0) == b"ok" and lib.gl_strerror(-1) == b"invalid argument"
    # negative sizes, n_ss < 1, bad dtype: GL_EINVAL; empty batches: GL_OK -- all before any CUDA call
    assert lib.gl_lightcurve(None, -1, None, 0, 0.0, 1, None, 0, None) == -1
    assert lib.gl_lightcurve(None, 1, None, 1, 0.0, 0, None, 0, None) == -1
    assert lib.gl_lightcurve(None, 1, None, 1, 0.0, 1, None, 7, None) == -1
    assert lib.gl_lightcurve(None, 1, None, 1, 0.0, 1, None, 0, None) == -1      # null pointers
    assert lib.gl_lightcurve(None, 0, None, 5, 0.0, 1, None, 0, None) == 0
    assert lib.gl_flux_geometry(None, 0, None, 0, None) == 0
    assert lib.gl_flux_geometry(None, 5, None, 0, None) == -1
    assert lib.gl_loglike(None, 1, None, 1, float("nan"), 1, None, None, None, None, 0, None) == -1
    assert lib.gl_launch_count() == 0


def test_no_cpu_fallback_on_host_tensors(lib):
    import numpy as np
    import torch
    import paper_2410_05408_b200 as g
    with pytest.raises(g.GreenlanternError):
        g.gl_lightcurve(torch.zeros(1, 12, dtype=torch.float64), torch.zeros(4, dtype=torch.float64))
    with pytest.raises(g.GreenlanternError):
        g.gl_flux_geometry(np.zeros((3, 6)))


def test_product_does_not_import_the_oracle():
    pat = re.compile(r"^\s*(import\s+oracle|from\s+oracle|#\s*include\s+.*oracle)|gl_oracle|libgl_oracle",
                     re.M)
    for f in (ROOT / "paper_2410_05408_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cuh", ".h"):
            assert not pat.search(f.read_text()), f
