"""gl_gp_loglike_static: the GP likelihood with its scratch in a file-scope device array (no
cudaMalloc on the path) against gl_gp_loglike, the existing path with a caller-allocated scratch.
Collected LAST by pytest (file name), so a failure here hides no other test under `pytest -x`.

The two entry points run the same launches (the static one only substitutes the scratch pointer), so
the results must agree bit for bit; the assertion uses the tolerance the GP tests use for fp32 (1e-4
relative of |ln L|, tests/test_gpu_parity.py::test_gp_likelihood) AND reports exact equality.
Two calls in a row: the second one finds the first one's contents in the shared array, for a batch of
another shape (smaller B, shorter T: stale elements beyond the new [B, T] must not matter, and the
rows land at other offsets).
"""
import numpy as np
import pytest

from paper_2410_05408_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gl():
    import torch
    assert torch.cuda.is_available()
    import paper_2410_05408_b200 as g
    g.load_library()
    return g


def dev(x):
    import torch
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device="cuda:0")


def _case(B, lo, hi, seed):
    """Config-3-shaped walkers on a slice of the K2-shaped series around the transit, one invalid walker,
    one walker without a correlated term."""
    rng = np.random.default_rng(seed)
    w = wl.config3(B=B)
    p = w.params.copy()
    p[B // 2, 6] = 0.7                                   # invalid walker: ln L = -inf on both paths
    gp = np.column_stack([rng.uniform(0.3e-4, 5e-4, B), rng.uniform(0.01, 1.0, B), rng.uniform(0.0, 2e-4, B)])
    gp[1, 0] = 0.0
    s = slice(lo, hi)
    return p, w.times[s], w.t_exp, w.n_ss, w.obs[s], w.sigma[s], gp


def _agree(a, b):
    a, b = a.cpu().numpy(), b.cpu().numpy()
    assert a.shape == b.shape
    inf = np.isinf(b)
    assert np.array_equal(np.isinf(a), inf) and np.array_equal(a[inf], b[inf])
    assert inf.sum() == 1 and np.all(np.isfinite(b[~inf]))
    rel = np.abs(a[~inf] - b[~inf]) / np.maximum(np.abs(b[~inf]), 1.0)
    assert rel.max() <= 1e-4, rel.max()
    return bool(np.array_equal(a, b))


def test_gp_loglike_static_scratch_matches_allocating_path(gl):
    import torch
    cap = gl.gl_gp_static_capacity()
    assert cap == 1 << 20
    exact = []
    # first call: 48 walkers x 1500 exposures; second call right behind it: other shape, stale scratch
    for B, lo, hi, seed in ((48, 1200, 2700, 7), (20, 1700, 2200, 8)):
        p, t, t_exp, n_ss, obs, sig, gp = _case(B, lo, hi, seed)
        args = (dev(p), dev(t), t_exp, n_ss, dev(obs), dev(sig), dev(gp))
        ref = gl.gl_gp_loglike(*args, dtype="f32")
        out = torch.full((B,), 123.0, dtype=torch.float64, device="cuda:0")
        got = gl.gl_gp_loglike_static(*args, out=out)
        torch.cuda.synchronize()
        assert got is out
        exact.append(_agree(got, ref))
    assert all(exact), exact                               # same launches, same bits
    # the same inputs again through the static path: the array's earlier contents do not leak in
    again = gl.gl_gp_loglike_static(*args)
    torch.cuda.synchronize()
    assert torch.equal(again, got)
    # the whole of config 3 fits (256 x 3900 <= capacity) ...
    w = wl.config3()
    assert w.B * w.T <= cap
    gp3 = np.tile([2e-4, 0.5, 1e-4], (w.B, 1))
    a3 = (dev(w.params), dev(w.times), w.t_exp, w.n_ss, dev(w.obs), dev(w.sigma), dev(gp3))
    full = gl.gl_gp_loglike_static(*a3)
    ref3 = gl.gl_gp_loglike(*a3, dtype="f32")
    torch.cuda.synchronize()
    assert torch.equal(full, ref3)
    # ... and one row more than the capacity is refused with the library's own message, nothing enqueued
    Tbig = cap // 4 + 1
    tb = np.linspace(-1.0, 1.0, Tbig)
    with pytest.raises(gl.GreenlanternError, match="capacity"):
        gl.gl_gp_loglike_static(dev(w.params[:4]), dev(tb), w.t_exp, 1, dev(np.ones(Tbig)),
                                dev(np.full(Tbig, 1e-4)), dev(gp3[:4]))
    ok = gl.gl_gp_loglike_static(dev(w.params[:4]), dev(tb[:-1]), w.t_exp, 1, dev(np.ones(Tbig - 1)),
                                 dev(np.full(Tbig - 1, 1e-4)), dev(gp3[:4]))
    torch.cuda.synchronize()
    assert torch.isfinite(ok).all()
