"""Pins for the CPU oracle (oracle/gl_oracle.c) against what the paper and the
mathematics fix -- never against the oracle itself and never against the CUDA path.

Each test names the passage it pins (PAPER.md line / equation; SURVEY.md 8(c) pin id)
and is chosen so that a plausible slip in the oracle (dropped term, wrong sign,
transposed operand, wrong index) fails it.
"""
from pathlib import Path

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate, optimize

import oracle as orc

GOLDEN = Path(__file__).parent / "golden" / "survey_probe_pins.txt"
PI = np.pi


def _golden(kind):
    rows = []
    for line in GOLDEN.read_text().splitlines():
        line = line.split("#")[0].split()
        if line and line[0] == kind:
            rows.append([float(v) for v in line[1:]])
    return rows


def oblate_outline(rp, f, eta, xi):
    return orc.outline(rp * (1 - f), rp, rp, 0.0, eta, xi)


def flux_from_areas(A, u1, u2):
    c0, c1, c2 = 1 - u1 - 2 * u2, u1 + 2 * u2, u2
    return 1 - (c0 * A[0] + c1 * A[1] + c2 * A[2]) / (PI * (1 - u1 / 3 - u2 / 6))


# --------------------------------------------------------------------------
# eqs. 3-6: rotation
# --------------------------------------------------------------------------
def test_rotation_matches_eq6_product_and_is_proper():
    rng = np.random.default_rng(1)
    for _ in range(20):
        z, e, x = rng.uniform(-PI, PI, 3)
        Rx = np.array([[1, 0, 0], [0, np.cos(z), -np.sin(z)], [0, np.sin(z), np.cos(z)]])
        Ry = np.array([[np.cos(e), 0, np.sin(e)], [0, 1, 0], [-np.sin(e), 0, np.cos(e)]])
        Rz = np.array([[np.cos(x), -np.sin(x), 0], [np.sin(x), np.cos(x), 0], [0, 0, 1]])
        R = orc.rotation(z, e, x)
        assert np.allclose(R, Rx @ Ry @ Rz, atol=1e-15)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-14)
        assert abs(np.linalg.det(R) - 1) < 1e-14
    # oblate case, zeta = 0: first row is the spin axis (SURVEY.md 8(c) equation checks)
    R = orc.rotation(0.0, 0.3, 0.7)
    assert np.allclose(R[0], [np.cos(0.3) * np.cos(0.7), -np.cos(0.3) * np.sin(0.7), np.sin(0.3)],
                       atol=1e-15)


# --------------------------------------------------------------------------
# eqs. 7-13: outline of the projected ellipsoid
# --------------------------------------------------------------------------
def test_outline_is_cholesky_factor_of_projected_covariance():
    """eqs. 11-13 == lower Cholesky factor of [R^T diag(a^2,b^2,c^2) R]_{xy}."""
    rng = np.random.default_rng(2)
    for _ in range(50):
        a, b, c = rng.uniform(0.02, 0.3, 3)
        z, e, x = rng.uniform(-PI, PI, 3)
        R = orc.rotation(z, e, x)
        C = (R.T @ np.diag([a * a, b * b, c * c]) @ R)[:2, :2]
        L = np.linalg.cholesky(C)
        d = orc.outline(a, b, c, z, e, x)
        assert np.allclose([d[0], d[1], d[2]], [L[0, 0], L[1, 0], L[1, 1]], rtol=1e-12, atol=1e-15)


def test_outline_bounds_brute_force_projection_of_the_ellipsoid():
    """Project a dense cloud of surface points of the rotated ellipsoid (eq. 2) onto
    the sky; the support function of the cloud must equal that of eqs. 7-8."""
    rng = np.random.default_rng(3)
    u = np.linspace(0, PI, 1501)[:, None]
    v = np.linspace(0, 2 * PI, 3001)[None, :]
    sph = np.stack([np.sin(u) * np.cos(v), np.sin(u) * np.sin(v), np.cos(u) * np.ones_like(v)], -1)
    sph = sph.reshape(-1, 3)
    for _ in range(4):
        a, b, c = rng.uniform(0.05, 0.3, 3)
        z, e, x = rng.uniform(-PI, PI, 3)
        R = orc.rotation(z, e, x)
        prim = sph * np.array([a, b, c])          # surface points in the primed frame
        obs = prim @ R                            # x = R^T x'  (eq. 2, planet-centred)
        dx, dy1, dy2 = orc.outline(a, b, c, z, e, x)
        for ang in rng.uniform(0, 2 * PI, 6):
            n = np.array([np.cos(ang), np.sin(ang)])
            brute = (obs[:, :2] @ n).max()
            model = np.hypot(n[0] * dx + n[1] * dy1, n[1] * dy2)
            assert abs(brute - model) < 2e-6 * max(a, b, c) + 1e-9


def test_outline_golden_and_oblate_axes():
    for rp, f, eta, xi, dx, dy1, dy2 in _golden("outline"):
        d = oblate_outline(rp, f, np.deg2rad(eta), np.deg2rad(xi))
        assert np.allclose(d, [dx, dy1, dy2], rtol=0, atol=2e-14)
    # semi-axes Rp and Rp sqrt(1 - f(2-f) cos^2 eta); minor axis along (cos xi, -sin xi)
    rp, f, eta, xi = 0.13, 0.4, 0.5, 0.9
    dx, dy1, dy2 = oblate_outline(rp, f, eta, xi)
    C = np.array([[dx * dx, dx * dy1], [dx * dy1, dy1 * dy1 + dy2 * dy2]])
    w, V = np.linalg.eigh(C)
    assert np.allclose(np.sqrt(w), [rp * np.sqrt(1 - f * (2 - f) * np.cos(eta) ** 2), rp], rtol=1e-13)
    minor = V[:, 0] * np.sign(V[0, 0])
    assert np.allclose(minor, [np.cos(xi), -np.sin(xi)], atol=1e-12)


def test_locked_outline_reduces_to_free_outline_at_conjunction_geometry():
    """eqs. B14-B16 with alpha = beta = 0 describe the same body as eqs. 11-13 seen
    through the same rotation, up to the frame flip of eq. B13 (x -> -x, y -> -y...):
    the projected covariance must agree, i.e. dx, |dy1|, dy2 are equal."""
    rng = np.random.default_rng(4)
    for _ in range(20):
        a, b, c = rng.uniform(0.02, 0.3, 3)
        z, e, x = rng.uniform(-PI, PI, 3)
        d0 = orc.outline(a, b, c, z, e, x)
        d1 = orc.outline_locked(a, b, c, z, e, x, 0.0, 0.0)
        assert np.allclose([d0[0], abs(d0[1]), d0[2]], [d1[0], abs(d1[1]), d1[2]], rtol=1e-12)


def test_locked_outline_matches_brute_force_projection():
    """eq. B13: x' = R [Rx(-alpha) Ry(beta) x + (0,0,d)]; sky projection of the surface."""
    rng = np.random.default_rng(5)
    u = np.linspace(0, PI, 1201)[:, None]
    v = np.linspace(0, 2 * PI, 2401)[None, :]
    sph = np.stack([np.sin(u) * np.cos(v), np.sin(u) * np.sin(v), np.cos(u) * np.ones_like(v)], -1)
    sph = sph.reshape(-1, 3)
    for _ in range(3):
        a, b, c = rng.uniform(0.05, 0.3, 3)
        z, e, x = rng.uniform(-PI, PI, 3)
        al, be = rng.uniform(-0.5, 0.5), rng.uniform(-0.3, 0.3)
        R = orc.rotation(z, e, x)
        Rxm = np.array([[1, 0, 0], [0, np.cos(al), np.sin(al)], [0, -np.sin(al), np.cos(al)]])
        Ryb = np.array([[np.cos(be), 0, np.sin(be)], [0, 1, 0], [-np.sin(be), 0, np.cos(be)]])
        M = R @ Rxm @ Ryb                          # x' = M x + const  =>  x = M^T (x' - const)
        obs = (sph * np.array([a, b, c])) @ M      # rows: M^T x'
        dx, dy1, dy2 = orc.outline_locked(a, b, c, z, e, x, al, be)
        for ang in rng.uniform(0, 2 * PI, 6):
            n = np.array([np.cos(ang), np.sin(ang)])
            brute = (obs[:, :2] @ n).max()
            model = np.hypot(n[0] * dx + n[1] * dy1, n[1] * dy2)
            assert abs(brute - model) < 3e-6 * max(a, b, c) + 1e-9


# --------------------------------------------------------------------------
# quadrature tables
# --------------------------------------------------------------------------
@pytest.mark.parametrize("n", [8, 16, 31])
def test_leggauss_matches_numpy(n):
    x, w = orc.leggauss(n)
    xn, wn = np.polynomial.legendre.leggauss(n)
    assert np.allclose(x, xn, atol=1e-15) and np.allclose(w, wn, atol=1e-15)


# --------------------------------------------------------------------------
# eqs. 21-23 + Green's theorem: a fully-inside ellipse has textbook area moments
# --------------------------------------------------------------------------
def test_green_integrals_of_inside_ellipse_match_area_moments():
    rng = np.random.default_rng(6)
    for _ in range(6):
        rp, f = rng.uniform(0.03, 0.2), rng.uniform(0, 0.9)
        eta, xi = rng.uniform(0, PI / 2, 2)
        r0, ang = rng.uniform(0.0, 0.7), rng.uniform(0, 2 * PI)
        x0, y0 = r0 * np.cos(ang), r0 * np.sin(ang)
        dx, dy1, dy2 = oblate_outline(rp, f, eta, xi)
        A, n = orc.areas(x0, y0, dx, dy1, dy2)
        assert n == 0
        area = PI * dx * dy2
        assert abs(A[0] - area) < 1e-15                                    # curl f_flat = 1
        trC = dx * dx + dy1 * dy1 + dy2 * dy2
        assert abs(A[2] - area * (r0 * r0 + trC / 4)) < 1e-15              # curl f_quad = r^2

        # curl f_lin = sqrt(1-r^2): 2-D quadrature over the unit disc of the ellipse map
        def integrand(rho, t):
            px = x0 + dx * rho * np.cos(t)
            py = y0 + dy1 * rho * np.cos(t) + dy2 * rho * np.sin(t)
            return np.sqrt(1 - px * px - py * py) * rho * dx * dy2
        ref, _ = integrate.dblquad(integrand, 0, 2 * PI, 0, 1, epsabs=1e-13, epsrel=1e-13)
        assert abs(A[1] - ref) < 1e-12


def test_limb_closed_forms_match_eqs_21_23_on_the_unit_circle():
    """f_flat, f_lin, f_quad on (cos l, sin l): numeric integral over an arc must equal
    dl/2, dl/3, dl/4 - [sin 4l]/48 (the forms the oracle uses on limb arcs)."""
    def f_all(lam):
        x, y, xp, yp = np.cos(lam), np.sin(lam), -np.sin(lam), np.cos(lam)
        fl = 0.5 * (x * yp - y * xp)
        return fl, (2 / 3) * fl, 0.5 * (x * (x * x / 3 + y * y) * yp - y * (x * x + y * y / 3) * xp)
    la, lb = 0.37, 1.91
    for k, closed in enumerate([(lb - la) / 2, (lb - la) / 3,
                                (lb - la) / 4 - (np.sin(4 * lb) - np.sin(4 * la)) / 48]):
        num, _ = integrate.quad(lambda l: f_all(l)[k], la, lb, epsabs=1e-14)
        assert abs(num - closed) < 1e-13
    # full circle: pi, 2 pi/3, pi/2
    assert np.allclose([2 * PI / 2, 2 * PI / 3, 2 * PI / 4], [PI, 2 * PI / 3, PI / 2])


# --------------------------------------------------------------------------
# P1: sphere with quadratic limb darkening == radial limb-darkening integral
# --------------------------------------------------------------------------
def sphere_flux_radial(p, z, u1, u2):
    """1 - (1/norm) * int I(r) * 2 kappa(r) r dr, kappa = half-angle of the circle of
    radius r covered by a disc of radius p centred at distance z (definition-level)."""
    mp.mp.dps = 30
    p, z, u1, u2 = map(mp.mpf, (p, z, u1, u2))

    def inten(r):
        mu = mp.sqrt(max(mp.mpf(0), 1 - r * r))
        return 1 - u1 * (1 - mu) - u2 * (1 - mu) ** 2

    def kappa(r):
        if z + r <= p:
            return mp.pi
        if r <= abs(z - p) and z > p:
            return mp.mpf(0)
        if r + p <= z or abs(z - p) >= r and z > p:
            return mp.mpf(0)
        if r <= p - z:
            return mp.pi
        c = (r * r + z * z - p * p) / (2 * r * z)
        return mp.acos(max(-1, min(1, c)))

    lo, hi = max(mp.mpf(0), z - p), min(mp.mpf(1), z + p)
    if hi <= lo:
        return mp.mpf(1)
    pts = [lo, hi]
    if z < p:
        pts = [mp.mpf(0), p - z, hi]
    blocked = mp.quad(lambda r: inten(r) * 2 * kappa(r) * r, pts)
    return 1 - blocked / (mp.pi * (1 - u1 / 3 - u2 / 6))


@pytest.mark.parametrize("p,z,u1,u2", [
    (0.1, 0.0, 0.4, 0.25), (0.1, 0.5, 0.4, 0.25), (0.1, 0.95, 0.4, 0.25), (0.1, 1.05, 0.4, 0.25),
    (0.066, 0.2, 0.4, 0.25), (0.2, 0.85, 0.9, -0.1), (0.3, 0.1, 0.6, 0.1), (0.05, 0.999, 0.3, 0.3),
    (0.15, 1.149, 0.2, 0.4)])
def test_P1_sphere_matches_radial_integral(p, z, u1, u2):
    ref = float(sphere_flux_radial(p, z, u1, u2))
    # place the sphere at a generic polar angle and a generic (irrelevant) orientation
    ang = 0.7
    dx, dy1, dy2 = orc.outline(p, p, p, 0.3, 0.4, 1.1)
    got = orc.flux_outline(z * np.cos(ang), z * np.sin(ang), dx, dy1, dy2, u1, u2)
    assert abs(got - ref) < 2e-14


def test_P1_golden_sphere_values():
    for p, z, u1, u2, flux in _golden("sphere"):
        assert abs(orc.flux_outline(z, 0.0, p, 0.0, p, u1, u2) - flux) < 2e-15
        assert abs(float(sphere_flux_radial(p, z, u1, u2)) - flux) < 2e-15


# --------------------------------------------------------------------------
# P2: uniform limb darkening, fully inside: blocked fraction = dx*dy2 = (pi a b)/pi
# --------------------------------------------------------------------------
def test_P2_uniform_inside_blocks_projected_area():
    rng = np.random.default_rng(7)
    for _ in range(20):
        rp, f = rng.uniform(0.02, 0.3), rng.uniform(0, 0.95)
        eta, xi = rng.uniform(-PI / 2, PI / 2), rng.uniform(0, PI)
        dx, dy1, dy2 = oblate_outline(rp, f, eta, xi)
        F = orc.flux_outline(0.2, -0.3, dx, dy1, dy2, 0.0, 0.0)
        exact = rp * rp * np.sqrt(1 - f * (2 - f) * np.cos(eta) ** 2)
        assert abs((1 - F) - exact) < 3e-16
    rp, f, eta, depth = _golden("depth")[0]
    dx, dy1, dy2 = oblate_outline(rp, f, np.deg2rad(eta), np.deg2rad(30))
    assert abs((1 - orc.flux_outline(0.3, 0.0, dx, dy1, dy2, 0, 0)) - depth) < 1e-15


# --------------------------------------------------------------------------
# P3: uniform limb darkening, sphere straddling the limb == circle-circle lens area
# --------------------------------------------------------------------------
def lens_area(p, z):
    """Textbook circle-circle intersection area (radii p and 1, centres z apart), in
    30-digit arithmetic: the float formula itself cancels at the 1e-14 level."""
    mp.mp.dps = 30
    p, z = mp.mpf(p), mp.mpf(z)
    if z >= 1 + p:
        return mp.mpf(0)
    if z <= 1 - p:
        return mp.pi * p * p
    k1 = mp.acos((z * z + p * p - 1) / (2 * z * p))
    k0 = mp.acos((z * z + 1 - p * p) / (2 * z))
    return p * p * k1 + k0 - mp.sqrt((1 + p - z) * (z + p - 1) * (z - p + 1) * (z + p + 1)) / 2


@pytest.mark.parametrize("p,z", [(0.1, 0.95), (0.1, 1.0), (0.1, 1.09), (0.3, 0.8), (0.02, 1.01),
                                 (0.45, 0.7), (0.2, 1.1999), (0.2, 0.8001)])
def test_P3_lens_area(p, z):
    A, n = orc.areas(z, 0.0, p, 0.0, p)
    assert n == 2
    assert abs(A[0] - float(lens_area(p, z))) < 5e-16
    # and at a generic polar angle (positions rounded, so a looser bound)
    A, n = orc.areas(z * np.cos(2.1), z * np.sin(2.1), p, 0.0, p)
    assert n == 2 and abs(A[0] - float(lens_area(p, z))) < 2e-15


# --------------------------------------------------------------------------
# P4: brute force on tiny inputs (pixel grid and Monte Carlo)
# --------------------------------------------------------------------------
BRUTE_CASES = [  # x0, y0, Rp, f, eta, xi, u1, u2
    (0.3, 0.0, 0.1, 0.3, 0.35, 0.52, 0.40, 0.25),
    (0.3, 0.88, 0.1, 0.3, 0.35, 0.52, 0.40, 0.25),
    (0.3, 0.93, 0.1, 0.3, 0.35, 0.52, 0.40, 0.25),
    (-0.6, 0.75, 0.2, 0.6, 0.1, 1.2, 0.7, -0.1),
    (0.98, 0.0, 0.2, 0.95, 0.0, 0.0, 0.4, 0.25),     # flat side across the limb (4 crossings)
    (0.0, 0.02, 0.3, 0.5, 0.0, 0.3, 0.5, 0.2),       # star centre inside the outline
    (0.7, 0.72, 0.15, 0.8, 0.2, 2.3, 0.0, 0.0),
    (0.55, -0.8, 0.066, 0.5, 0.52, 0.79, 0.2, 0.5),
]


def brute_grid_flux(x0, y0, dx, dy1, dy2, u1, u2, n=3000):
    """Midpoint pixel integration of I over (ellipse n disc) on the outline's bounding box."""
    hx, hy = dx, np.hypot(dy1, dy2)
    xs = x0 - hx + (np.arange(n) + 0.5) * (2 * hx / n)
    ys = y0 - hy + (np.arange(n) + 0.5) * (2 * hy / n)
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    # inside the outline: invert eqs. 7-8 for (cos t, sin t)
    c = (X - x0) / dx
    s = (Y - y0 - dy1 * c) / dy2
    r2 = X * X + Y * Y
    m = (c * c + s * s <= 1.0) & (r2 <= 1.0)
    mu = np.sqrt(np.clip(1 - r2, 0, None))
    inten = 1 - u1 * (1 - mu) - u2 * (1 - mu) ** 2
    blocked = (inten * m).sum() * (2 * hx / n) * (2 * hy / n)
    return 1 - blocked / (PI * (1 - u1 / 3 - u2 / 6))


@pytest.mark.parametrize("case", BRUTE_CASES)
def test_P4_pixel_grid(case):
    x0, y0, rp, f, eta, xi, u1, u2 = case
    dx, dy1, dy2 = oblate_outline(rp, f, eta, xi)
    got = orc.flux_outline(x0, y0, dx, dy1, dy2, u1, u2)
    ref = brute_grid_flux(x0, y0, dx, dy1, dy2, u1, u2)
    assert abs(got - ref) < 4e-7


def test_P4_monte_carlo():
    rng = np.random.default_rng(8)
    for case in BRUTE_CASES[:5]:
        x0, y0, rp, f, eta, xi, u1, u2 = case
        dx, dy1, dy2 = oblate_outline(rp, f, eta, xi)
        n = 2_000_000
        rho, t = np.sqrt(rng.uniform(0, 1, n)), rng.uniform(0, 2 * PI, n)   # uniform in the outline
        X = x0 + dx * rho * np.cos(t)
        Y = y0 + dy1 * rho * np.cos(t) + dy2 * rho * np.sin(t)
        r2 = X * X + Y * Y
        mu = np.sqrt(np.clip(1 - r2, 0, None))
        val = (1 - u1 * (1 - mu) - u2 * (1 - mu) ** 2) * (r2 <= 1)
        scale = PI * dx * dy2 / (PI * (1 - u1 / 3 - u2 / 6))
        est, err = 1 - val.mean() * scale, val.std() * scale / np.sqrt(n)
        got = orc.flux_outline(x0, y0, dx, dy1, dy2, u1, u2)
        assert abs(got - est) < 5 * err + 1e-9


# --------------------------------------------------------------------------
# P5: out of transit is exactly 1
# --------------------------------------------------------------------------
def test_P5_out_of_transit_is_exactly_one():
    row = np.array([0.0, 10.0, 20.0, 0.3, 0.0, 0.0, 0.1, 0.3, 0.5, 0.3, 0.4, 0.25])
    for t in (0.5, 2.0, -3.3, 4.99):
        assert orc.flux_time(row, t) == 1.0
    # secondary eclipse (reading R16): planet over the disc but behind the star
    assert orc.flux_time(row, 5.0) == 1.0
    x0, y0, front = orc.position(row, 5.0)
    assert not front and np.hypot(x0, y0) < 1.0
    # just outside by any outline, including grazing distance
    dx, dy1, dy2 = oblate_outline(0.1, 0.3, 0.3, 0.5)
    assert orc.flux_outline(1.2, 0.0, dx, dy1, dy2, 0.4, 0.25) == 1.0
    assert orc.flux_outline(0.0, 1.1000001, 0.1, 0.0, 0.1, 0.4, 0.25) == 1.0


# --------------------------------------------------------------------------
# P6: symmetry about mid-transit
# --------------------------------------------------------------------------
def test_P6_time_reversal_symmetry():
    base = np.array([0.1, 10.0, 20.0, 0.3, 0.0, 0.0, 0.1, 0.4, 0.0, 0.35, 0.4, 0.25])
    taus = np.linspace(0.0, 0.1, 23)
    for tau in taus:                                      # xi = 0: the curve is even in tau
        assert abs(orc.flux_time(base, 0.1 + tau) - orc.flux_time(base, 0.1 - tau)) < 1e-14
    tilted, mirrored = base.copy(), base.copy()
    tilted[8], mirrored[8] = 0.6, -0.6
    asym = 0.0
    for tau in taus:                                      # F(t0+tau; xi) = F(t0-tau; -xi)
        a, b = orc.flux_time(tilted, 0.1 + tau), orc.flux_time(mirrored, 0.1 - tau)
        assert abs(a - b) < 1e-14
        asym = max(asym, abs(a - orc.flux_time(tilted, 0.1 - tau)))
    assert asym > 1e-6                                    # and xi != 0 really is asymmetric


# --------------------------------------------------------------------------
# P7: App. A mu-degeneracy (eq. A1; reading R22: R_eq fixed)
# --------------------------------------------------------------------------
def test_P7_mu_degeneracy():
    def mu_of(f, eta):
        return (f - 1) ** 2 + f * (f - 2) * np.cos(2 * eta)       # eq. A1
    f1, eta1 = 0.3, 0.2
    target = mu_of(f1, eta1)
    f2 = 0.5
    eta2 = optimize.brentq(lambda e: mu_of(f2, e) - target, 0.0, PI / 2)
    assert abs(eta2 - eta1) > 0.1
    r1 = np.array([0.0, 10.0, 20.0, 0.3, 0.0, 0.0, 0.1, f1, 0.6, eta1, 0.4, 0.25])
    r2 = r1.copy()
    r2[7], r2[9] = f2, eta2
    for t in np.linspace(-0.12, 0.12, 25):
        assert abs(orc.flux_time(r1, t) - orc.flux_time(r2, t)) < 1e-14
    # eq. A2: f_min = 1 - sqrt((mu+1)/2) is the projected flattening
    dx, dy1, dy2 = oblate_outline(0.1, f1, eta1, 0.6)
    C = np.array([[dx * dx, dx * dy1], [dx * dy1, dy1 * dy1 + dy2 * dy2]])
    w = np.sqrt(np.linalg.eigvalsh(C))
    assert abs((1 - w[0] / w[1]) - (1 - np.sqrt((target + 1) / 2))) < 1e-13


# --------------------------------------------------------------------------
# P8: the paper's literal algorithm (snapping eqs. 16-20 + Simpson) agrees
# --------------------------------------------------------------------------
@pytest.mark.parametrize("x0,y0", [(0.3, 0.0), (0.3, 0.88), (0.3, 0.93), (0.3, 0.99), (0.6, 0.85)])
def test_P8_snap_simpson_agrees(x0, y0):
    """Snapping keeps f_flat and f_lin continuous in theta (they only see the angular
    rate, eq. 19) but makes f_quad JUMP at each limb crossing (it also sees the radial
    part of the tangent), so Simpson converges O(h^2)-or-better for the first two and
    only O(h) for A_quad (SURVEY.md headline: snap+Simpson converges O(1/N))."""
    dx, dy1, dy2 = oblate_outline(0.1, 0.3, np.deg2rad(20), np.deg2rad(30))
    A, _ = orc.areas(x0, y0, dx, dy1, dy2)
    S = orc.areas_snap_simpson(x0, y0, dx, dy1, dy2, 2 ** 16)
    u1, u2 = 0.4, 0.25
    assert abs(flux_from_areas(A, u1, u2) - flux_from_areas(S, u1, u2)) < 1e-7
    assert abs(A[0] - S[0]) < 1e-9 and abs(A[1] - S[1]) < 1e-9 and abs(A[2] - S[2]) < 1e-6


def test_P8_snap_simpson_converges_to_the_oracle():
    dx, dy1, dy2 = oblate_outline(0.1, 0.3, np.deg2rad(20), np.deg2rad(30))
    A, _ = orc.areas(0.3, 0.93, dx, dy1, dy2)
    errs = [np.abs(orc.areas_snap_simpson(0.3, 0.93, dx, dy1, dy2, 2 ** k) - A) for k in (12, 16, 21)]
    assert errs[2][2] < 5e-8 and errs[2][0] < 1e-12 and errs[2][1] < 1e-12
    assert errs[0][2] > errs[1][2] > errs[2][2]


# --------------------------------------------------------------------------
# P9: survey probe values (mpmath, independent routes)
# --------------------------------------------------------------------------
def test_P9_golden_oblate_and_geometry_values():
    for rp, f, eta, xi, x0, y0, u1, u2, flux in _golden("oblate"):
        d = oblate_outline(rp, f, np.deg2rad(eta), np.deg2rad(xi))
        assert abs(orc.flux_outline(x0, y0, *d, u1, u2) - flux) < 2e-13
    for rp, f, eta, xi, x0, y0, a0, a1, a2 in _golden("areas"):
        d = oblate_outline(rp, f, np.deg2rad(eta), np.deg2rad(xi))
        A, _ = orc.areas(x0, y0, *d)
        assert np.all(np.abs(A - [a0, a1, a2]) < 1e-8)
    for d_, rp, fp, pa, u1, u2, flux, ncross in _golden("geom"):
        got = orc.flux_geometry([[d_, rp, fp, pa, u1, u2]])[0]
        assert abs(got - flux) < 2e-15
        a, b = rp, rp * (1 - fp)
        cxx = a * a * np.cos(pa) ** 2 + b * b * np.sin(pa) ** 2
        dxx = np.sqrt(cxx)
        _, n = orc.areas(d_, 0.0, dxx, (a * a - b * b) * np.cos(pa) * np.sin(pa) / dxx, a * b / dxx)
        assert n == int(ncross)
    for d_, rp, fp, pa, a0, a1, a2 in _golden("geomareas"):
        a, b = rp, rp * (1 - fp)
        dxx = np.sqrt(a * a * np.cos(pa) ** 2 + b * b * np.sin(pa) ** 2)
        A, n = orc.areas(d_, 0.0, dxx, (a * a - b * b) * np.cos(pa) * np.sin(pa) / dxx, a * b / dxx)
        assert n == 4 and np.all(np.abs(A - [a0, a1, a2]) < 5e-16)


def test_geometry_row_convention_major_axis_along_PA():
    """PA = 0 puts the MAJOR axis along the star->planet direction: at d = 1 + Rp(1-f)
    + margin only a PA = 0 planet (reach Rp) touches the disc, a PA = pi/2 one (reach
    Rp(1-f)) does not."""
    rp, fp = 0.2, 0.5
    d = 1 + rp * (1 - fp) + 0.02
    assert orc.flux_geometry([[d, rp, fp, 0.0, 0.3, 0.2]])[0] < 1.0
    assert orc.flux_geometry([[d, rp, fp, PI / 2, 0.3, 0.2]])[0] == 1.0


# --------------------------------------------------------------------------
# orbit (reading R7): Kepler residual, conjunction, e -> 0, and two-body dynamics
# --------------------------------------------------------------------------
def test_kepler_residual_and_limits():
    rng = np.random.default_rng(9)
    for _ in range(200):
        M, e = rng.uniform(-10, 10), rng.uniform(0, 0.95)
        E = orc.kepler(M, e)
        assert abs(E - e * np.sin(E) - M) < 4e-15 * max(1, abs(M))
    assert orc.kepler(1.234, 0.0) == 1.234


@pytest.mark.parametrize("e,om", [(0.0, 0.0), (0.1, 0.3), (0.3, 2.0), (0.6, -1.0), (0.5, PI / 2)])
def test_conjunction_is_at_impact_parameter(e, om):
    row = np.array([1.7, 30.0, 40.0, 0.35, e, om, 0.1, 0.2, 0.3, 0.2, 0.4, 0.25])
    x0, y0, front = orc.position(row, 1.7)
    assert front and abs(x0 - 0.35) < 1e-13 and abs(y0) < 1e-13
    x1, y1, _ = orc.position(row, 1.7 + 0.01)
    assert y1 > 0            # the planet moves toward +y (alpha increasing, eq. 10)


def test_circular_orbit_is_eqs_9_10():
    row = np.array([0.2, 10.0, 20.0, 0.3, 0.0, 1.3, 0.1, 0.2, 0.3, 0.2, 0.4, 0.25])
    for t in np.linspace(-4, 6, 41):
        al = 2 * PI * (t - 0.2) / 10.0
        x0, y0, front = orc.position(row, t)
        assert abs(x0 - 20.0 * np.cos(al) * (0.3 / 20.0)) < 1e-12       # eq. 9, sin(beta) = b/d
        assert abs(y0 - 20.0 * np.sin(al)) < 1e-12                      # eq. 10
        assert front == (np.cos(al) > 0)
    ecc = row.copy()
    ecc[4] = 1e-9
    for t in np.linspace(-1, 1, 9):
        assert np.allclose(orc.position(ecc, t)[:2], orc.position(row, t)[:2], atol=1e-6)


@pytest.mark.parametrize("e,om", [(0.3, 0.7), (0.6, 2.5), (0.15, -2.0)])
def test_eccentric_orbit_obeys_two_body_dynamics(e, om):
    """Integrate r'' = -mu r/|r|^3 in the sky frame from the periapsis state and compare
    with the oracle's Kepler-solver positions (pins e>0 beyond self-consistency)."""
    P, aR, b, t0 = 20.0, 15.0, 0.4, 0.3
    row = np.array([t0, P, aR, b, e, om, 0.1, 0.2, 0.3, 0.2, 0.4, 0.25])
    n = 2 * PI / P
    mu_g = n * n * aR ** 3
    cosi = (b / aR) * (1 + e * np.sin(om)) / (1 - e * e)
    sini = np.sqrt(1 - cosi * cosi)
    # orbital-plane basis in (x, y, z): conjunction direction (phi = 0) and quadrature (phi = pi/2)
    e_conj = np.array([cosi, 0.0, -sini])     # in front of the star (z < 0), x0 = r cos i
    e_quad = np.array([0.0, 1.0, 0.0])        # +y, direction of motion at conjunction
    phi_p = om - PI / 2                       # periapsis: nu = 0  =>  phi = omega - pi/2
    rhat = np.cos(phi_p) * e_conj + np.sin(phi_p) * e_quad
    that = -np.sin(phi_p) * e_conj + np.cos(phi_p) * e_quad
    r_p = aR * (1 - e)
    v_p = np.sqrt(mu_g * (1 + e) / (aR * (1 - e)))
    # time of periapsis from the closed-form forward Kepler relation at conjunction
    nuc = PI / 2 - om
    Ec = 2 * np.arctan2(np.sqrt(1 - e) * np.sin(nuc / 2), np.sqrt(1 + e) * np.cos(nuc / 2))
    t_peri = t0 - (Ec - e * np.sin(Ec)) / n
    ts = t_peri + np.linspace(0.0, 1.3 * P, 14)[1:]
    sol = integrate.solve_ivp(lambda t, s: np.concatenate([s[3:], -mu_g * s[:3] / np.linalg.norm(s[:3]) ** 3]),
                              (t_peri, ts[-1]), np.concatenate([r_p * rhat, v_p * that]),
                              t_eval=ts, method="DOP853", rtol=1e-13, atol=1e-13)
    for t, s in zip(ts, sol.y.T):
        x0, y0, front = orc.position(row, t)
        assert abs(x0 - s[0]) < 2e-8 and abs(y0 - s[1]) < 2e-8
        assert front == (s[2] < 0)


# --------------------------------------------------------------------------
# supersampling (reading R18) and chi^2 (reading R19): self-consistency only
# --------------------------------------------------------------------------
def test_supersampling_is_midpoint_mean_and_converges_to_time_average():
    row = np.array([0.0, 10.0, 20.0, 0.3, 0.0, 0.0, 0.1, 0.3, 0.5, 0.3, 0.4, 0.25])
    t, texp = 0.075, 0.02
    for S in (1, 3, 4, 15):
        offs = ((np.arange(S) + 0.5) / S - 0.5) * texp
        manual = np.mean([orc.flux_time(row, t + o) for o in offs])
        assert abs(orc.flux_time(row, t, texp, S) - manual) < 2e-16
    avg, _ = integrate.quad(lambda s: orc.flux_time(row, s), t - texp / 2, t + texp / 2,
                            epsabs=1e-13, limit=200)
    assert abs(orc.flux_time(row, t, texp, 200) - avg / texp) < 2e-8


def test_chi2_definition_and_invalid_walkers():
    rng = np.random.default_rng(10)
    rows = np.array([[0.0, 10.0, 20.0, 0.3, 0.0, 0.0, 0.1, 0.3, 0.5, 0.3, 0.4, 0.25],
                     [0.01, 10.0, 21.0, 0.1, 0.0, 0.0, 0.08, 0.0, 0.0, 0.0, 0.3, 0.1],
                     [0.0, 10.0, 20.0, 0.3, 0.0, 0.0, 0.6, 0.3, 0.5, 0.3, 0.4, 0.25]])  # Rp >= 0.5
    times = np.linspace(-0.2, 0.2, 81)
    sigma = rng.uniform(1e-4, 3e-4, times.size)
    flux = orc.lightcurve(rows, times, 0.01, 3)
    obs = flux[0] + rng.normal(0, 1, times.size) * sigma
    chi2, flux2 = orc.loglike(rows, times, 0.01, 3, obs, sigma)
    assert np.array_equal(flux[:2], flux2[:2])
    import math
    for b in range(2):
        ref = math.fsum(((obs - flux[b]) / sigma) ** 2)
        assert abs(chi2[b] - ref) <= 1e-13 * ref
    assert np.all(np.isnan(flux[2])) and np.isinf(chi2[2])
    chi_self, _ = orc.loglike(rows[:1], times, 0.01, 3, flux[0], sigma)
    assert chi_self[0] == 0.0
    assert not orc.params_valid(rows[2]) and orc.params_valid(rows[0])


# ---------------------------------------------------------------------------------------------
# NEXT-2: extended rows (triaxial / tidally locked), oracle.lightcurve_ex.  The outline functions
# (eqs. 11-13, B14-B16) are pinned above by brute-force projection; these pins fix how the light
# curve USES them: which alpha and beta go into B14-B16 (reading R23), the axis columns, and the
# reductions that must hold exactly.
# ---------------------------------------------------------------------------------------------
def _short_period_row(**kw):
    row = dict(t0=0.0, P=3.0, aR=6.0, b=0.3, e=0.0, om=0.0, Rp=0.1, f=0.4, xi=0.5, eta=0.3,
               u1=0.0, u2=0.0, zeta=0.0, rb=1.0, rc=1.0, locked=0.0)
    row.update(kw)
    return np.array([[row[k] for k in ("t0", "P", "aR", "b", "e", "om", "Rp", "f", "xi", "eta",
                                       "u1", "u2", "zeta", "rb", "rc", "locked")]])


def test_ex_rows_reduce_to_the_oblate_model():
    t = np.linspace(-0.12, 0.12, 41)
    p = _short_period_row(u1=0.4, u2=0.25)
    assert np.array_equal(orc.lightcurve_ex(p, t, 0.01, 3), orc.lightcurve(p[:, :12], t, 0.01, 3))
    # a sphere does not care about locking, zeta, or which way it turns
    s0 = orc.lightcurve(_short_period_row(f=0.0, u1=0.4, u2=0.25)[:, :12], t)
    s1 = orc.lightcurve_ex(_short_period_row(f=0.0, u1=0.4, u2=0.25, locked=1.0, zeta=0.7), t)
    assert np.abs(s1 - s0).max() < 1e-14
    # zeta spins an oblate spheroid (b = c) about its own symmetry axis: nothing changes
    z = orc.lightcurve_ex(_short_period_row(u1=0.4, u2=0.25, zeta=1.1), t)
    assert np.abs(z - orc.lightcurve(p[:, :12], t)).max() < 1e-13
    # invalid extended columns
    assert not orc.params_ex_valid(_short_period_row(rb=0.0)[0])
    assert not orc.params_ex_valid(_short_period_row(locked=0.5)[0])
    assert not orc.params_ex_valid(_short_period_row(rc=6.0)[0])
    assert np.all(np.isnan(orc.lightcurve_ex(_short_period_row(rb=-1.0), t)))


def test_ex_uniform_depth_is_the_projected_area():
    """Uniform limb darkening, outline wholly inside the disc: 1 - F = dx * dy2 (pin P2), with the
    outline of eqs. 11-13 (free) or of eqs. B14-B16 at alpha = 2 pi (t - t0)/P, sin(beta) = b/(a/R*)
    (locked) -- computed here from the outline functions alone."""
    for kw in (dict(rb=0.8, rc=0.6, zeta=0.4), dict(rb=1.3, rc=0.7, zeta=-0.9, xi=-0.4)):
        free = _short_period_row(**kw)
        lock = _short_period_row(locked=1.0, **kw)
        a, b, c = 0.1 * 0.6, 0.1 * kw["rb"], 0.1 * kw["rc"]
        ts = np.array([-0.05, -0.03, 0.0, 0.02, 0.045])
        Ff = orc.lightcurve_ex(free, ts)[0]
        Fl = orc.lightcurve_ex(lock, ts)[0]
        d0 = orc.outline(a, b, c, kw["zeta"], 0.3, kw.get("xi", 0.5))
        assert np.abs((1 - Ff) - d0[0] * d0[2]).max() < 1e-13
        beta = np.arcsin(0.3 / 6.0)
        for t, F in zip(ts, Fl):
            dl = orc.outline_locked(a, b, c, kw["zeta"], 0.3, kw.get("xi", 0.5), 2 * np.pi * t / 3.0, beta)
            assert abs((1 - F) - dl[0] * dl[2]) < 1e-13
        # a locked triaxial body does change its projected area along the chord
        assert np.ptp(1 - Fl) > 1e-5 and np.ptp(1 - Ff) < 1e-13


def test_ex_locked_brute_force_pixels():
    """One locked, limb-darkened, limb-crossing sample against a pixel sum over the outline
    obtained by PROJECTING the rotated ellipsoid point by point (eq. B13), not from B14-B16."""
    kw = dict(rb=0.7, rc=1.2, zeta=0.3, u1=0.4, u2=0.25, b=0.5, locked=1.0)
    p = _short_period_row(**kw)
    t = 0.069                                  # ingress: the outline straddles the limb
    F = orc.lightcurve_ex(p, np.array([t]))[0, 0]
    al, be = 2 * np.pi * t / 3.0, np.arcsin(0.5 / 6.0)
    x0, y0, front = orc.position(p[0, :12], t)
    assert front and 0.9 < np.hypot(x0, y0) < 1.1
    # eq. B13: x' = R [Rx(-al) Ry(be) x + (0,0,d)] takes OBSERVER coordinates x to BODY coordinates
    # x' (the ellipsoid's axes are the primed ones), so the body seen by the observer is x = M^T x' 
    R = np.array(orc.rotation(0.3, 0.3, 0.5)).reshape(3, 3)
    ca, sa, cb, sb = np.cos(al), np.sin(al), np.cos(be), np.sin(be)
    Rx = np.array([[1, 0, 0], [0, ca, sa], [0, -sa, ca]])          # Rx(-alpha), eq. 3
    Ry = np.array([[cb, 0, sb], [0, 1, 0], [-sb, 0, cb]])          # Ry(beta), eq. 4
    M = R @ Rx @ Ry
    S = np.diag([0.06, 0.07, 0.12]) ** 2
    C = (M.T @ S @ M)[:2, :2]                  # covariance of the projected outline
    Ci = np.linalg.inv(C)
    n = 3000
    h = 0.14
    gx = x0 + (np.arange(n) + 0.5) * (2 * h / n) - h
    gy = y0 + (np.arange(n) + 0.5) * (2 * h / n) - h
    X, Y = np.meshgrid(gx, gy, indexing="ij")
    dxp, dyp = X - x0, Y - y0
    inside = (Ci[0, 0] * dxp * dxp + 2 * Ci[0, 1] * dxp * dyp + Ci[1, 1] * dyp * dyp <= 1.0)
    r2 = X * X + Y * Y
    mu = np.sqrt(np.clip(1 - r2, 0, None))
    inten = np.where(r2 <= 1, 1 - 0.4 * (1 - mu) - 0.25 * (1 - mu) ** 2, 0.0)
    blocked = (inten * inside).sum() * (2 * h / n) ** 2 / (np.pi * (1 - 0.4 / 3 - 0.25 / 6))
    assert abs((1 - F) - blocked) < 3e-6


# ---------------------------------------------------------------------------------------------
# NEXT-3: the sampling parameters of App. A.  Pins: the forward map (A1, A4)
# against the defining relations A2-A3; the Jacobian A5 by finite differences; A6 |det J| = cos(eta)
# (eq. A7, with its normalisation); the sampler A10/A12 by a Monte-Carlo test of what it is FOR
# (f uniform, eta cosine-distributed), which goes through the inverse map as well; and App. A's
# physical claim (equal mu, equal R_eq => identical light curves) through the whole front end.
# ---------------------------------------------------------------------------------------------
def test_munu_forward_inverse_and_jacobian():
    rng = np.random.default_rng(21)
    for _ in range(200):
        f, eta = rng.uniform(0.01, 0.97), rng.uniform(0.02, PI / 2 - 0.02)
        mu, nu = orc.munu_of(f, eta)
        # A1 by its own definition and A3 through A2
        assert abs(mu - ((f - 1) ** 2 + f * (f - 2) * np.cos(2 * eta))) < 1e-15
        fmin = 1 - np.sqrt((mu + 1) / 2)
        assert abs(f - (fmin + (1 - fmin) * nu)) < 1e-13
        assert -1 < mu < 1 and 0 < nu <= 1
        f2, eta2 = orc.feta_of(mu, nu)
        assert abs(f2 - f) < 1e-13 and abs(eta2 - eta) < 1e-9 / max(np.sin(2 * eta), 1e-3)
        # eq. A5 by central differences of the forward map
        h = 1e-6
        J = np.array([(orc.munu_of(f + h, eta) - orc.munu_of(f - h, eta)) / (2 * h),
                      (orc.munu_of(f, eta + h) - orc.munu_of(f, eta - h)) / (2 * h)]).T
        detJ = np.linalg.det(J)
        A5 = 2 ** 1.5 * f * (f - 2) * np.sin(2 * eta) / np.sqrt(2 + f * (f - 2) * (1 + np.cos(2 * eta)))
        assert abs(detJ - A5) < 1e-6 * max(1.0, abs(A5))
        # eq. A6 |det J| = cos(eta): eq. A7 including the constant (uniform f on [0,1], cos eta on [0, pi/2])
        assert abs(np.exp(orc.log_prior_munu(mu, nu)) * abs(A5) - np.cos(eta)) < 1e-9
    assert orc.log_prior_munu(1.2, 0.5) == -np.inf and orc.log_prior_munu(0.2, 0.0) == -np.inf


def test_munu_sampler_gives_uniform_f_and_cosine_eta():
    from scipy import stats
    rng = np.random.default_rng(22)
    n = 40_000
    f, eta = np.empty(n), np.empty(n)
    for k, (u, w) in enumerate(rng.random((n, 2))):
        mu, nu = orc.munu_from_uniform(u, w)
        f[k], eta[k] = orc.feta_of(mu, nu)
    assert stats.kstest(f, "uniform").pvalue > 1e-3                 # p(f) = 1 on [0, 1]
    assert stats.kstest(np.sin(eta), "uniform").pvalue > 1e-3       # p(eta) = cos(eta): CDF sin(eta)
    assert abs(np.corrcoef(f, np.sin(eta))[0, 1]) < 0.02            # and independent (eq. A7)


def test_params_from_munu_front_end():
    # two (f, eta) pairs on one mu contour, same equatorial radius: identical curves (App. A, R22)
    f1, eta1 = 0.5, 0.9
    mu, _ = orc.munu_of(f1, eta1)
    f2 = 0.3
    eta2 = 0.5 * np.arccos((mu - (f2 - 1) ** 2) / (f2 * (f2 - 2)))
    rows = []
    for f, eta in ((f1, eta1), (f2, eta2)):
        m, n = orc.munu_of(f, eta)
        assert abs(m - mu) < 1e-14
        rows.append([0.0, 10.0, 20.0, 0.3, 0.0, 0.0, 0.1 * (1 - f) ** (1 / 3), m, n, 0.5, 0.36, 0.3])
    p, lp = orc.params_from_munu(rows)
    assert np.allclose(p[:, 6], 0.1, rtol=1e-14) and np.allclose(p[:, 7], [f1, f2], atol=1e-13)
    assert np.allclose(p[:, 9], [eta1, eta2], atol=1e-12)
    # Kipping: u1 = 2 sqrt(q1) q2, u2 = sqrt(q1)(1 - 2 q2)  <=>  q1 = (u1 + u2)^2, q2 = u1 / (2 (u1 + u2))
    assert np.allclose((p[:, 10] + p[:, 11]) ** 2, 0.36) and np.allclose(p[:, 10] / (2 * (p[:, 10] + p[:, 11])), 0.3)
    t = np.linspace(-0.15, 0.15, 61)
    a, b = orc.lightcurve(p[:1], t), orc.lightcurve(p[1:], t)
    assert np.abs(a - b).max() < 1e-13 and a.min() < 0.995
    assert np.all(np.isfinite(lp))
    bad, lpb = orc.params_from_munu([[0, 10, 20, 0.3, 0, 0, 0.1, 1.5, 0.5, 0.5, 0.3, 0.3]])
    assert np.all(np.isnan(bad)) and lpb[0] == -np.inf


# ---------------------------------------------------------------------------------------------
# NEXT-4: Gaussian-process likelihood (Matern-3/2 + jitter), dense definition.
# ---------------------------------------------------------------------------------------------
def test_gp_dense_definition():
    from scipy import stats
    rng = np.random.default_rng(33)
    t = np.sort(rng.uniform(0, 3, 60))
    sig = rng.uniform(0.5e-4, 2e-4, 60)
    r = 1e-4 * rng.standard_normal(60)
    s, rho, jit = 3e-4, 0.2, 1e-4
    # kernel values: variance at zero lag, textbook value at one timescale, decay
    assert abs(orc.matern32(0.0, s, rho) - s * s) < 1e-20
    assert abs(orc.matern32(rho, s, rho) - s * s * (1 + np.sqrt(3)) * np.exp(-np.sqrt(3))) < 1e-20
    assert orc.matern32(10 * rho, s, rho) < 1e-6 * s * s
    # against a library routine on the same covariance
    K = orc.matern32(t[:, None] - t[None, :], s, rho) + np.diag(sig ** 2 + jit ** 2)
    want = stats.multivariate_normal(mean=np.zeros(60), cov=K, allow_singular=False).logpdf(r)
    assert abs(orc.gp_loglike_dense(r, t, sig, s, rho, jit) - want) < 1e-8 * abs(want)
    # white-noise limit: s -> 0 gives -chi^2/2 - sum ln sqrt(sigma^2 + jit^2) - T/2 ln 2 pi
    v = sig ** 2 + jit ** 2
    white = -0.5 * (r * r / v).sum() - 0.5 * np.log(v).sum() - 30 * np.log(2 * np.pi)
    assert abs(orc.gp_loglike_dense(r, t, sig, 0.0, rho, jit) - white) < 1e-9 * abs(white)
    # a draw from the process is more likely under its own hyper-parameters than under wrong ones
    L = np.linalg.cholesky(K)
    y = L @ rng.standard_normal(60)
    assert orc.gp_loglike_dense(y, t, sig, s, rho, jit) > orc.gp_loglike_dense(y, t, sig, 30 * s, rho, jit)
