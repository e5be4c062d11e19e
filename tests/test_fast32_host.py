"""CPU check of the CUDA path's fp32 production arithmetic (csrc/gl_fast32.cuh).

The header compiles as plain C++ (exact libm in place of the MUFU approximations), so steps a3 + a4
of the fp32 path -- fixed-node trapezoid tiers, rotation Newton for t_far, crossing solve, smoothed
Gauss-Legendre, limb closed forms -- are compared with the oracle here, without a GPU.  The GPU
parity tests remain the gate for the real (MUFU) arithmetic."""
import ctypes
import subprocess
from pathlib import Path

import numpy as np
import pytest

import oracle as orc
from paper_2410_05408_b200 import workloads as wl

HERE = Path(__file__).resolve().parent


@pytest.fixture(scope="module")
def host_lib(tmp_path_factory):
    so = tmp_path_factory.mktemp("fast32") / "libfast32_host.so"
    subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", str(so),
                    str(HERE / "host_fast32_harness.cpp"), "-lm"], check=True)
    lib = ctypes.CDLL(str(so))
    lib.host_flux_geometry_f32.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p]
    return lib


def run(lib, geom):
    geom = np.ascontiguousarray(geom, dtype=np.float64)
    out = np.empty(geom.shape[0])
    assert lib.host_flux_geometry_f32(geom.ctypes.data, geom.shape[0], out.ctypes.data) == 0
    return out


def test_fast32_matches_oracle_on_config5_mix(host_lib):
    geom, cls = wl.config5(N=60_000)
    out = run(host_lib, geom)
    err = np.abs(out - orc.flux_geometry(geom))
    for c in range(5):
        assert err[cls == c].max() <= 5e-7, (c, err[cls == c].max())
    assert np.all(out[geom[:, 0] >= 1.0 + geom[:, 1]] == 1.0)      # no overlap: exactly 1


def test_fast32_trapezoid_tiers(host_lib):
    """Whole-outline-inside geometries at every tier boundary (gap = 0.5, 3a, a, 0.3, 0.01, ~0)."""
    rows = []
    for rp, f in ((0.066, 0.5), (0.2, 0.9), (0.1, 0.0), (0.02, 0.3)):
        for pa in (0.0, 0.7, np.pi / 2, 2.5):
            for gap in (0.7, 0.5001, 0.4999, rp * 3.001, rp * 2.999, 0.3001, 0.2999, rp * 1.001, rp * 0.999,
                        0.0101, 0.0099, 1e-3, 1e-5):
                d = 1.0 - gap - rp
                if d > 0:
                    rows.append((d, rp, f, pa, 0.4, 0.25))
    geom = np.array(rows)
    err = np.abs(run(host_lib, geom) - orc.flux_geometry(geom))
    assert err.max() <= 3e-7, err.max()


def test_fast32_golden_pins(host_lib):
    """SURVEY.md 8(c) pin P9 rows (mpmath values), through the fp32 arithmetic."""
    geom = np.array([(0.98, 0.2, 0.95, np.pi / 2, 0.4, 0.25), (0.95, 0.15, 0.6, 0.7, 0.4, 0.25),
                     (1.0, 0.1, 0.5, 2.0, 0.7, -0.1)])
    want = np.array([0.998815344408319, 0.994809529489372, 0.998408554994727])
    assert np.abs(run(host_lib, geom) - want).max() <= 5e-7


def test_hot_kernel_literal_tables_match_the_generator(host_lib):
    """csrc/gl_hot.cuh carries the quadrature tables as literals (immediates in the unrolled loop, a
    statically initialised constant array): they must be the generator's values, bit for bit."""
    import re
    text = (HERE.parent / "paper_2410_05408_b200" / "csrc" / "gl_hot.cuh").read_text()

    def floats(body):
        return np.array([np.float32(x) for x in re.findall(r"(-?\d+\.?\d*(?:e-?\d+)?)f", body)], dtype=np.float32)
    phi = floats(re.search(r"#define GLH_GL_PHI \{([^}]*)\}", text).group(1))
    om = floats(re.search(r"#define GLH_GL_OM \{([^}]*)\}", text).group(1))
    trap = floats(re.search(r"c_trap16\[16\] = \{(.*?)\};", text, re.S).group(1))
    assert phi.size == 8 and om.size == 8 and trap.size == 32
    p, o, t = np.zeros(8, np.float32), np.zeros(8, np.float32), np.zeros(32, np.float32)
    host_lib.host_tables(p.ctypes.data_as(ctypes.c_void_p), o.ctypes.data_as(ctypes.c_void_p),
                         t.ctypes.data_as(ctypes.c_void_p))
    assert np.array_equal(phi, p) and np.array_equal(om, o) and np.array_equal(trap, t)
