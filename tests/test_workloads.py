"""Host-side checks of the seeded input recipes."""
import numpy as np

import oracle as orc
from paper_2410_05408_b200 import workloads as wl


def test_shapes_and_determinism():
    c1, c2, c3, c4 = wl.config1(), wl.config2(), wl.config3(), wl.config4(B=8, T=2000)
    assert c1.params.shape == (1, 12) and c1.times.shape == (1000,) and c1.n_ss == 1
    assert abs(c1.meta["T14"] - 0.16853143995258) < 1e-12          # SURVEY.md 8(c) reading 17
    assert c2.times.shape == (3900,) and c2.n_ss == 15 and abs(c2.t_exp - 29.4 / 1440) < 1e-15
    assert abs(c2.times[0] + 39.80) < 0.01 and abs(c2.times[-1] - 39.80) < 0.01
    assert c3.params.shape == (256, 12) and np.array_equal(c3.obs, c2.obs)
    assert c4.params.shape == (8, 12) and c4.n_ss == 3
    again = wl.config3()
    assert np.array_equal(again.params, c3.params) and np.array_equal(again.obs, c3.obs)
    p = c3.params
    assert np.all((p[:, 7] >= 0) & (p[:, 7] < 0.9)) and np.all((p[:, 6] >= 0.06) & (p[:, 6] <= 0.072))
    assert np.all(p[:, 4] == 0) and np.all(p[:, 1] == 542.0)
    assert all(orc.params_valid(r) for r in p)
    # noise level of the stand-in data
    assert 0.8e-4 < np.std(c2.obs[:1500] - 1.0) < 1.2e-4


def test_config4_window_is_self_inconsistent_as_documented():
    """reading R20: 20000 x 5 s = 1.157 d, i.e. +-0.737 T14, not +-1.2 T14."""
    c4 = wl.config4(B=1)
    T14 = wl.transit_duration(542.0, 230.0, 0.2, 0.066)
    assert abs(T14 - 0.7854147) < 1e-6
    assert abs((c4.times[-1] - c4.times[0]) / T14 / 2 - 0.737) < 0.01


def test_config5_mix_and_forced_classes():
    geom, cls = wl.config5(N=40_000)
    assert geom.shape == (40_000, 6) and np.all(geom[:36_000:1000, 2] == 0.0)
    assert [(cls == k).sum() for k in range(5)] == [36_000, 1000, 1000, 1000, 1000]
    assert np.all(geom[:, 0] >= 0) and np.all((geom[:, 3] >= 0) & (geom[:, 3] <= np.pi))
    # tangent constructions really are (near-)tangent: nudging the planet radially in or
    # out by 1e-3 changes whether the outline touches the limb
    def ncross(row):
        d, rp, fp, pa = row[:4]
        a, b = rp, rp * (1 - fp)
        dx = np.sqrt(a * a * np.cos(pa) ** 2 + b * b * np.sin(pa) ** 2)
        return orc.areas(d, 0.0, dx, (a * a - b * b) * np.cos(pa) * np.sin(pa) / dx, a * b / dx)[1]
    ext = geom[cls == 1][:60]
    for row in ext:
        far, near = row.copy(), row.copy()
        far[0] += 1e-3
        near[0] -= 1e-3
        assert ncross(far) == -1 and ncross(near) >= 2
    four = sum(ncross(r) == 4 for r in geom[cls == 4][:200])
    assert four > 120
    on_limb = geom[cls == 3]
    assert np.all(np.abs(on_limb[:, 0] - 1.0) <= 1e-4)
