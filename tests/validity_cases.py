"""Rows that walk every per-walker validity rule across its boundary.

The expected verdicts are written out BY HAND from the rule list in include/greenlantern_b200.h
(lines 41-44) / SURVEY.md 8(b): a walker is invalid iff any entry is non-finite, P <= 0, e outside
[0, 1), Rp_eq outside (0, 0.5), f outside [0, 1), a/R* (1 - e) <= 1, |b| (1 + e sin omega) >
a/R* (1 - e^2), or 1 - u1/3 - u2/6 <= 0; for the extended rows also: zeta, rb, rc, locked non-finite,
rb <= 0, rc <= 0, Rp rb >= 0.5, Rp rc >= 0.5, locked not in {0, 1}.  Neither the oracle nor the
CUDA path is asked: tests/test_validity_rules.py checks the oracle against this table (CPU), and
tests/test_gpu_parity.py feeds the same rows to the library (GPU).
No transit-model arithmetic lives here.
"""
import numpy as np

COLS = {"t0": 0, "P": 1, "aR": 2, "b": 3, "e": 4, "om": 5, "Rp": 6, "f": 7, "xi": 8, "eta": 9,
        "u1": 10, "u2": 11, "zeta": 12, "rb": 13, "rc": 14, "locked": 15}
BASE = dict(t0=0.0, P=10.0, aR=20.0, b=0.3, e=0.0, om=0.0, Rp=0.1, f=0.3, xi=0.5, eta=0.3,
            u1=0.4, u2=0.25, zeta=0.0, rb=1.0, rc=1.0, locked=0.0)
HALF_PI = float(np.pi / 2)

# (name, {column: value}, valid?)   -- 12-column rules
CASES12 = [
    ("base", {}, True),
    ("P zero", {"P": 0.0}, False),
    ("P negative", {"P": -10.0}, False),
    ("P tiny positive", {"P": 1e-3, "aR": 20.0}, True),
    ("e slightly negative", {"e": -1e-9}, False),
    ("e zero with omega set", {"e": 0.0, "om": 1.0}, True),
    ("e = 0.6", {"e": 0.6, "om": 0.7}, True),
    ("e = 1", {"e": 1.0, "aR": 2000.0}, False),
    ("e > 1", {"e": 1.5, "aR": 2000.0}, False),
    ("Rp zero", {"Rp": 0.0}, False),
    ("Rp negative", {"Rp": -0.1}, False),
    ("Rp just below 0.5", {"Rp": 0.4999}, True),
    ("Rp = 0.5", {"Rp": 0.5}, False),
    ("f slightly negative", {"f": -1e-9}, False),
    ("f zero", {"f": 0.0}, True),
    ("f = 0.95", {"f": 0.95}, True),
    ("f = 1", {"f": 1.0}, False),
    ("aR = 1 (periastron on the surface)", {"aR": 1.0}, False),
    ("aR = 1.5", {"aR": 1.5}, True),
    ("aR(1-e) = 1", {"aR": 2.0, "e": 0.5, "om": 0.3, "b": 0.1}, False),
    ("aR(1-e) just above 1", {"aR": 2.2, "e": 0.5, "om": 0.3, "b": 0.1}, True),
    ("|b| = aR, e = 0 (face-on, allowed)", {"b": 20.0}, True),
    ("b = -aR, e = 0", {"b": -20.0}, True),
    ("|b| > aR, e = 0", {"b": 20.001}, False),
    ("b < -aR, e = 0", {"b": -20.001}, False),
    ("|b|(1+e) just inside aR(1-e^2), omega = pi/2", {"e": 0.5, "om": HALF_PI, "b": 9.99}, True),
    ("|b|(1+e) beyond aR(1-e^2), omega = pi/2", {"e": 0.5, "om": HALF_PI, "b": 10.01}, False),
    ("same, b negative", {"e": 0.5, "om": HALF_PI, "b": -10.01}, False),
    ("|b|(1-e) just inside, omega = -pi/2", {"e": 0.5, "om": -HALF_PI, "b": 29.9}, True),
    ("|b|(1-e) beyond, omega = -pi/2", {"e": 0.5, "om": -HALF_PI, "b": 30.1}, False),
    ("LD norm zero (u1 = 3)", {"u1": 3.0, "u2": 0.0}, False),
    ("LD norm negative", {"u1": 3.5, "u2": 0.0}, False),
    ("LD norm small positive", {"u1": 2.0, "u2": 0.0}, True),
    ("LD norm zero (u2 = 6)", {"u1": 0.0, "u2": 6.0}, False),
    ("never transits, b > 1 + Rp", {"b": 1.2}, True),
    ("never transits, b < -(1 + Rp)", {"b": -1.2}, True),
    ("grazing, b = 1.05", {"b": 1.05}, True),
    ("grazing, b = -1.05", {"b": -1.05}, True),
    ("negative angles", {"xi": -1.1, "eta": -0.7, "b": -0.4}, True),
]
for _c in ("t0", "P", "aR", "b", "e", "om", "Rp", "f", "xi", "eta", "u1", "u2"):
    CASES12.append((f"{_c} NaN", {_c: float("nan")}, False))
    CASES12.append((f"{_c} +inf", {_c: float("inf")}, False))
    CASES12.append((f"{_c} -inf", {_c: float("-inf")}, False))

# extended-row rules (columns 12-15); every 12-column case carries over with rb = rc = 1, locked = 0
CASES_EX = [
    ("ex base triaxial", {"zeta": 0.3, "rb": 0.9, "rc": 1.1}, True),
    ("ex locked", {"zeta": 0.3, "rb": 0.9, "rc": 1.1, "locked": 1.0}, True),
    ("zeta NaN", {"zeta": float("nan")}, False),
    ("zeta inf", {"zeta": float("inf")}, False),
    ("rb zero", {"rb": 0.0}, False),
    ("rb negative", {"rb": -1.0}, False),
    ("rb NaN", {"rb": float("nan")}, False),
    ("rc zero", {"rc": 0.0}, False),
    ("rc inf", {"rc": float("inf")}, False),
    ("Rp rb = 0.5", {"rb": 5.0}, False),
    ("Rp rb just below 0.5", {"rb": 4.99}, True),
    ("Rp rc = 0.5", {"rc": 5.0}, False),
    ("Rp rc just below 0.5", {"rc": 4.99}, True),
    ("locked = 0.5", {"locked": 0.5}, False),
    ("locked = 2", {"locked": 2.0}, False),
    ("locked = -1", {"locked": -1.0}, False),
    ("locked NaN", {"locked": float("nan")}, False),
]


def row16(mods):
    r = dict(BASE)
    r.update(mods)
    out = np.empty(16)
    for k, v in r.items():
        out[COLS[k]] = v
    return out


def rows12():
    """([n, 12] rows, [n] expected validity, names)."""
    rows = np.array([row16(m)[:12] for _, m, _ in CASES12])
    return rows, np.array([v for _, _, v in CASES12]), [n for n, _, _ in CASES12]


def rows16():
    cases = [(n, m, v) for n, m, v in CASES12] + CASES_EX
    rows = np.array([row16(m) for _, m, _ in cases])
    return rows, np.array([v for _, _, v in cases]), [n for n, _, _ in cases]


# bare-geometry rows (d, Rp, f_proj, PA, u1, u2) of gl_flux_geometry: invalid iff any entry non-finite,
# d < 0, Rp outside (0, 0.5), f_proj outside [0, 1), 1 - u1/3 - u2/6 <= 0 (include/greenlantern_b200.h)
GEOM_BASE = [0.6, 0.1, 0.3, 0.7, 0.4, 0.25]
GEOM_CASES = [
    ({}, True), ({0: 0.0}, True), ({0: -0.1}, False), ({0: 5.0}, True), ({1: 0.0}, False), ({1: -0.1}, False),
    ({1: 0.4999}, True), ({1: 0.5}, False), ({2: -1e-9}, False), ({2: 0.0}, True), ({2: 0.95}, True),
    ({2: 1.0}, False), ({3: -2.0}, True), ({3: 40.0}, True), ({4: 3.0, 5: 0.0}, False), ({4: 2.0, 5: 0.0}, True),
    ({4: 0.0, 5: 6.0}, False),
] + [({k: v}, False) for k in range(6) for v in (float("nan"), float("inf"), float("-inf"))]


def geom_rows():
    rows = []
    for mods, _ in GEOM_CASES:
        r = list(GEOM_BASE)
        for k, v in mods.items():
            r[k] = v
        rows.append(r)
    return np.array(rows), np.array([v for _, v in GEOM_CASES])
