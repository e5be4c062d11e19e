"""Seeded synthetic inputs for the five configurations of BASELINE.json.

This module serves BOTH the CUDA path (tests, bench.py) and the CPU oracle's
tests.  It holds input recipes only -- no transit-model arithmetic: nothing
here evaluates an outline, an intersection, a boundary integral or a flux.
It imports numpy and nothing else from this repository.

The paper's data (K2 C5/C18 photometry of HIP 41378; the
PandExo/NIRISS simulation) are not available; the arrays
below stand in for them with the same shapes: 29.4-min / 5-s cadences, an
80-day baseline with one transit of a P = 542 d, d/R* ~ 231, r ~ 0.067 planet
(Table 2), 100 ppm / 30 ppm white noise.  DESIGN.md section
"Input recipe" states every draw; SURVEY.md section 8(d) is the source.

Parameter row (north_star, include/greenlantern_b200.h):
    0 t0   1 P   2 a/R*   3 b   4 e   5 omega   6 Rp_eq/R*   7 f
    8 xi (sky-projected obliquity)   9 eta (tilt out of the sky plane)
    10 u1   11 u2
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

NPARAMS = 12
MINUTE = 1.0 / 1440.0
SECOND = 1.0 / 86400.0

SEED_CFG2_NOISE = 4137802
SEED_CFG3_WALKERS = 4137803
SEED_CFG4_WALKERS = 4137804
SEED_CFG4_NOISE = 4137814
SEED_CFG5 = 4137805


@dataclass
class Workload:
    name: str
    params: np.ndarray            # [B, 12] float64
    times: np.ndarray             # [T] float64 (days)
    t_exp: float
    n_ss: int
    obs: np.ndarray | None = None     # [T]
    sigma: np.ndarray | None = None   # [T]
    meta: dict = field(default_factory=dict)

    @property
    def B(self):
        return self.params.shape[0]

    @property
    def T(self):
        return self.times.shape[0]


def transit_duration(P, aR, b, k):
    """T14 as BASELINE.json's configs 1 and 4 use it (reading R17)."""
    sini = np.sqrt(1.0 - (b / aR) ** 2)
    return P / np.pi * np.arcsin(np.sqrt((1.0 + k) ** 2 - b * b) / (aR * sini))


def kipping_to_u(q1, q2):
    """Kipping (2013) (q1, q2) -> (u1, u2) (Table 1 note f)."""
    sq = np.sqrt(q1)
    return 2.0 * sq * q2, sq * (1.0 - 2.0 * q2)


def synthetic_observation(row, times, sigma, seed):
    """A transit-SHAPED stand-in for the K2 / JWST photometry (not a model).

    Straight-chord kinematics, small-planet depth k^2 I(z)/<I> inside the disc,
    a linear ramp across the limb, plus seeded Gaussian noise.  It only has to
    look like the data (depth, duration, noise level); both the CUDA path and
    the oracle receive the very same array as their `obs` input.
    """
    t0, P, aR, b, k, u1, u2 = row[0], row[1], row[2], row[3], row[6], row[10], row[11]
    v = 2.0 * np.pi * aR / P
    z = np.sqrt(b * b + (v * (times - t0)) ** 2)
    mu = np.sqrt(np.clip(1.0 - np.minimum(z, 1.0) ** 2, 0.0, None))
    inten = (1.0 - u1 * (1.0 - mu) - u2 * (1.0 - mu) ** 2) / (1.0 - u1 / 3.0 - u2 / 6.0)
    ramp = np.clip((1.0 + k - z) / (2.0 * k), 0.0, 1.0)
    clean = 1.0 - k * k * inten * ramp
    rng = np.random.default_rng(seed)
    return clean + rng.normal(0.0, sigma, size=times.shape[0])


# --------------------------------------------------------------------------
# config 1: single light curve, uniform limb darkening, no supersampling
# --------------------------------------------------------------------------
def config1():
    row = np.array([0.0, 10.0, 20.0, 0.3, 0.0, 0.0, 0.1, 0.3,
                    np.deg2rad(30.0), np.deg2rad(20.0), 0.0, 0.0])
    T14 = transit_duration(10.0, 20.0, 0.3, 0.1)
    times = -1.5 * T14 + np.arange(1000) * (3.0 * T14 / 999.0)
    return Workload("cfg1_single_uniform_T1000", row[None, :], times, 0.0, 1,
                    meta={"T14": float(T14)})


# --------------------------------------------------------------------------
# config 2: long-period sub-Neptune, K2-shaped series
# --------------------------------------------------------------------------
CFG2_ROW = np.array([0.0, 542.0, 230.0, 0.2, 0.0, 0.0, 0.066, 0.5,
                     np.deg2rad(45.0), np.deg2rad(30.0), 0.40, 0.25])


def k2_times():
    dt = 29.4 * MINUTE
    return (np.arange(3900) - 1949.5) * dt, dt


def config2():
    times, dt = k2_times()
    sph = CFG2_ROW.copy()
    sph[7] = 0.0
    sigma = np.full(times.shape[0], 1e-4)
    obs = synthetic_observation(sph, times, 1e-4, SEED_CFG2_NOISE)
    return Workload("cfg2_k2_single_T3900_S15", CFG2_ROW[None, :].copy(), times, dt, 15,
                    obs, sigma)


def draw_walkers(B, seed):
    """Column-wise draws, in this order: f, xi, eta, Rp, b, a/R*, t0, q1, q2."""
    rng = np.random.default_rng(seed)
    f = rng.uniform(0.0, 0.9, B)
    xi = rng.uniform(0.0, np.pi / 2, B)
    eta = rng.uniform(0.0, np.pi / 2, B)
    rp = rng.uniform(0.06, 0.072, B)
    b = rng.uniform(0.0, 0.5, B)
    aR = rng.uniform(200.0, 260.0, B)
    t0 = rng.normal(0.0, 0.01, B)
    q1 = rng.uniform(0.0, 1.0, B)
    q2 = rng.uniform(0.0, 1.0, B)
    u1, u2 = kipping_to_u(q1, q2)
    P = np.full(B, 542.0)
    z = np.zeros(B)
    return np.column_stack([t0, P, aR, b, z, z, rp, f, xi, eta, u1, u2])


# --------------------------------------------------------------------------
# config 3: 256-walker MCMC batch on config 2's series (the headline workload)
# --------------------------------------------------------------------------
def config3(B=256):
    base = config2()
    params = draw_walkers(B, SEED_CFG3_WALKERS)
    return Workload(f"cfg3_k2_mcmc_B{B}_T3900_S15", params, base.times, base.t_exp, 15,
                    base.obs, base.sigma)


# --------------------------------------------------------------------------
# config 4: JWST-shaped high-cadence batch
# --------------------------------------------------------------------------
def config4(B=128, T=20000):
    dt = 5.0 * SECOND
    times = (np.arange(T) - (T - 1) / 2.0) * dt
    sph = CFG2_ROW.copy()
    sph[7] = 0.0
    sigma = np.full(T, 3e-5)
    obs = synthetic_observation(sph, times, 3e-5, SEED_CFG4_NOISE)
    params = draw_walkers(B, SEED_CFG4_WALKERS)
    return Workload(f"cfg4_jwst_B{B}_T{T}_S3", params, times, dt, 3, obs, sigma)


# --------------------------------------------------------------------------
# config 5: edge-geometry stress, rows (d, Rp, f_proj, PA, u1, u2)
# --------------------------------------------------------------------------
EPS_CYCLE = np.array([0.0, 1e-12, -1e-12, 1e-9, -1e-9, 1e-6, -1e-6, 1e-4, -1e-4])


def _tangent_rows(rng, n, internal):
    """Ellipses constructed tangent to the unit circle, by textbook geometry:
    in the ellipse's own frame the boundary point p = (a cos psi, b sin psi) has
    outward unit normal n ~ (b cos psi, a sin psi); a unit circle touching the
    ellipse at p from outside is centred at p + n, one touching it with the
    ellipse on its inner side at p - n."""
    rp = rng.uniform(0.01, 0.2, n)
    f = rng.uniform(0.0, 0.95, n)
    psi = rng.uniform(0.0, 2 * np.pi, n)
    a, b = rp, rp * (1.0 - f)
    px, py = a * np.cos(psi), b * np.sin(psi)
    nx, ny = b * np.cos(psi), a * np.sin(psi)
    nn = np.hypot(nx, ny)
    sgn = -1.0 if internal else 1.0
    cx, cy = px + sgn * nx / nn, py + sgn * ny / nn      # star centre, ellipse frame
    d = np.hypot(cx, cy)
    # PA: major axis (ellipse-frame x) measured from the star->planet direction (-c)
    pa = np.mod(-np.arctan2(-cy, -cx), np.pi)
    d = np.abs(d + EPS_CYCLE[np.arange(n) % EPS_CYCLE.size])
    return rp, f, pa, d


def config5(N=1_000_000, forced_fraction=0.1):
    rng = np.random.default_rng(SEED_CFG5)
    d = rng.uniform(0.0, 1.2, N)
    rp = rng.uniform(0.01, 0.2, N)
    f = rng.uniform(0.0, 0.95, N)
    f[::1000] = 0.0
    pa = rng.uniform(0.0, np.pi, N)
    u1 = rng.uniform(0.0, 1.0, N)
    u2 = rng.uniform(-0.2, 0.5, N)
    nf = int(N * forced_fraction) // 4
    start = N - 4 * nf
    cls = np.zeros(N, dtype=np.int8)
    if nf > 0:
        # (i) external tangency, (ii) internal tangency
        for j, internal in enumerate((False, True)):
            sl = slice(start + j * nf, start + (j + 1) * nf)
            rp[sl], f[sl], pa[sl], d[sl] = _tangent_rows(rng, nf, internal)
            cls[sl] = 1 + j
        # (iii) planet centre on the limb
        sl = slice(start + 2 * nf, start + 3 * nf)
        d[sl] = 1.0 + EPS_CYCLE[np.arange(nf) % EPS_CYCLE.size]
        cls[sl] = 3
        # (iv) flat side across the limb: tips outside, waist inside => 4 crossings
        sl = slice(start + 3 * nf, start + 4 * nf)
        rp4 = rng.uniform(0.15, 0.2, nf)
        f4 = rng.uniform(0.9, 0.95, nf)
        b4 = rp4 * (1.0 - f4)
        lo, hi = np.sqrt(1.0 - rp4 ** 2), 1.0 - b4
        half = nf // 2
        frac = rng.uniform(0.02, 0.98, nf)
        d4 = lo + frac * (hi - lo)
        pa4 = np.pi / 2 + rng.uniform(-0.02, 0.02, nf)
        # second half: untilted, sitting on the two ends of the 4-crossing window
        k = np.arange(nf - half)
        ends = np.where(k % 2 == 0, lo[half:], hi[half:])
        d4[half:] = ends + EPS_CYCLE[(k // 2) % EPS_CYCLE.size]
        pa4[half:] = np.pi / 2
        rp[sl], f[sl], pa[sl], d[sl] = rp4, f4, pa4, d4
        cls[sl] = 4
    geom = np.column_stack([d, rp, f, pa, u1, u2])
    return geom, cls


def get(name, **kw):
    return {"cfg1": config1, "cfg2": config2, "cfg3": config3, "cfg4": config4}[name](**kw)
