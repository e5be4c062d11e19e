"""Pins of the oracle's per-walker validity rules (gl_oracle_params_valid / _ex_valid): every
condition is walked across its boundary and compared with the verdicts written out by hand in
tests/validity_cases.py from include/greenlantern_b200.h:41-44 / SURVEY.md 8(b).  Also: what an
invalid walker returns (NaN row, chi^2 = +inf) and what a valid walker that never transits returns
(flux exactly 1, chi^2 = the baseline sum)."""
import math

import numpy as np

import oracle as orc
from validity_cases import CASES_EX, geom_rows, rows12, rows16

TIMES = np.concatenate([np.linspace(-0.3, 0.3, 61), [2.5, 5.0, 7.5]])


def test_every_12_column_rule_across_its_boundary():
    rows, valid, names = rows12()
    assert valid.sum() >= 15 and (~valid).sum() >= 50
    for r, v, n in zip(rows, valid, names):
        assert orc.params_valid(r) == bool(v), n


def test_every_extended_rule_across_its_boundary():
    rows, valid, names = rows16()
    for r, v, n in zip(rows, valid, names):
        assert orc.params_ex_valid(r) == bool(v), n
    assert len(CASES_EX) >= 15


def test_invalid_rows_give_nan_flux_and_infinite_chi2_valid_ones_finite():
    rows, valid, names = rows12()
    rng = np.random.default_rng(3)
    sigma = rng.uniform(1e-4, 3e-4, TIMES.size)
    obs = 1.0 + rng.normal(0.0, 1.0, TIMES.size) * sigma
    chi2, flux = orc.loglike(rows, TIMES, 0.01, 3, obs, sigma)
    base = math.fsum(((obs - 1.0) / sigma) ** 2)
    for k, (v, n) in enumerate(zip(valid, names)):
        if v:
            assert np.all(np.isfinite(flux[k])) and np.isfinite(chi2[k]), n
            if not n.startswith("LD"):   # (u1 = 2 is a limb-BRIGHTENED star: flux > 1 is right)
                assert flux[k].max() <= 1.0 and flux[k].min() > 0.0, n
        else:
            assert np.all(np.isnan(flux[k])), n
            assert np.isinf(chi2[k]) and chi2[k] > 0, n
        if n.startswith("never transits") or n.startswith("|b| = aR") or n.startswith("b = -aR"):
            assert np.all(flux[k] == 1.0), n                  # exactly 1, bit for bit (pin P5)
            assert abs(chi2[k] - base) <= 1e-12 * base, n     # chi^2 = the baseline sum
    # the extended entry point agrees on which rows are valid
    rows_ex, valid_ex, names_ex = rows16()
    fx = orc.lightcurve_ex(rows_ex, TIMES, 0.01, 3)
    for k, (v, n) in enumerate(zip(valid_ex, names_ex)):
        assert bool(np.all(np.isnan(fx[k]))) == (not v), n
        assert bool(np.all(np.isfinite(fx[k]))) == bool(v), n


def test_geometry_rows_validity():
    rows, valid = geom_rows()
    out = orc.flux_geometry(rows)
    assert np.array_equal(np.isnan(out), ~valid)
    assert np.all(np.isfinite(out[valid])) and np.all(out[valid] > 0.0)
