"""Small launches that reach every synchronisation pattern of the library, for compute-sanitizer:

    compute-sanitizer --tool memcheck  python tests/sanitizer_shapes.py
    compute-sanitizer --tool racecheck python tests/sanitizer_shapes.py        (shared memory only)

(one tool per GPU call; results are recorded in profiles/r02_sanitizer.md).  `--lib <.so>` runs the
same launches through another build of the library (the CHECKED build: index assertions + random
per-CTA delays), `--dump <.npz>` writes every fp32 output for a bitwise comparison between builds.  Every output is also
compared with the fp64 path of the library itself, so a run that "passes" the tool on garbage shows.
Patterns: hot_kernel sparse mode (compaction of the near-limb pairs, two lanes per pair, fill by idle
warps) and dense mode; hot_kernel as a cluster (barrier_arrive at entry / wait before the first DSMEM
push); flux-only calls cut into segments; units looping over grid rows; walkers off the common path
(eccentric, flat, close-in, short-period: generic_unit inside hot_kernel) alone and mixed with common
and invalid ones; the full transit_kernel (fp64, extended/locked rows) with several walkers per
cluster and multi-round series (T > C * tile: lists reused under a cluster barrier); the fp32
baseline + hot PDL chain; the GP scan behind it; the resident-series host and device calls (graph
replay); the bare-geometry kernels.  Not collected by pytest (run under the tool).
"""
import sys
from pathlib import Path

import numpy as np
import torch

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))
import paper_2410_05408_b200 as gl  # noqa: E402
from paper_2410_05408_b200 import workloads as wl  # noqa: E402

QUICK = "--quick" in sys.argv          # racecheck is ~100x slower than memcheck: smaller batches
RESULTS = {}                           # name -> fp32 outputs, written to `--dump file.npz` when asked for


def _opt(name):
    return sys.argv[sys.argv.index(name) + 1] if name in sys.argv else None


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device="cuda:0")


def check(name, a32, a64, tol):
    a32, a64 = a32.double().cpu().numpy(), a64.cpu().numpy()
    both_nan = np.isnan(a32) & np.isnan(a64)
    both_inf = np.isinf(a32) & np.isinf(a64)
    err = np.abs(np.where(both_nan | both_inf, 0.0, a32 - a64))
    rel = err / np.maximum(np.abs(np.where(both_nan | both_inf, 1.0, a64)), 1.0)
    print(f"  {name}: max |f32 - f64| = {err.max():.2e} (relative to max(|x|,1): {rel.max():.2e})")
    assert rel.max() <= tol, name
    RESULTS[f"{len(RESULTS):02d} {name}"] = a32


def loglike_both(p, t, t_exp, n_ss, obs, sig, ex=False):
    f = gl.gl_loglike_ex if ex else gl.gl_loglike
    c32, f32 = f(dev(p), dev(t), t_exp, n_ss, dev(obs), dev(sig), dtype="f32", want_flux=True)
    c64, f64 = f(dev(p), dev(t), t_exp, n_ss, dev(obs), dev(sig), dtype="f64", want_flux=True)
    torch.cuda.synchronize()
    return c32, f32, c64, f64


def main():
    if _opt("--lib"):      # a CHECKED build of the library (tests/test_gpu_parity.py) instead of the product
        from paper_2410_05408_b200 import binding
        binding._LIBPATH = Path(_opt("--lib"))
    gl.load_library()
    w = wl.config3(B=6 if QUICK else 24)
    rng = np.random.default_rng(1)

    print("hot_kernel, sparse mode (K2-shaped series), chi2 + flux / chi2 only / flux only")
    c32, f32, c64, f64 = loglike_both(w.params, w.times, w.t_exp, w.n_ss, w.obs, w.sigma)
    check("flux", f32, f64, 5e-7)
    check("chi2", c32, c64, 1e-4)
    c_only = gl.gl_loglike(dev(w.params), dev(w.times), w.t_exp, w.n_ss, dev(w.obs), dev(w.sigma), dtype="f32")
    lc = gl.gl_lightcurve(dev(w.params), dev(w.times), w.t_exp, w.n_ss, dtype="f32")
    torch.cuda.synchronize()
    assert torch.equal(c_only, c32)                      # same launch shape: same bits
    assert (lc - f32).abs().max().item() <= 1.2e-7       # other launch shape (segments): 1-2 ulp at most

    print("hot_kernel as a cluster, dense mode (long in-window range), and flux-only segments")
    T = 20_000
    t = (np.arange(T) - (T - 1) / 2) * (30.0 / 86400.0)
    obs = 1.0 + 3e-5 * rng.standard_normal(T)
    sig = np.full(T, 3e-5)
    p = w.params[:2 if QUICK else 4]
    c32, f32, c64, f64 = loglike_both(p, t, 30.0 / 86400.0, 3, obs, sig)
    check("flux", f32, f64, 5e-7)
    check("chi2", c32, c64, 1e-4)
    lc = gl.gl_lightcurve(dev(p[:1]), dev(t), 30.0 / 86400.0, 3, dtype="f32")
    torch.cuda.synchronize()
    assert (lc[0] - f32[0]).abs().max().item() <= 1.2e-7

    print("mixed batch: walkers off the common path (eccentric, flat, close-in, short period) + invalid ones")
    q = wl.config3(B=16 if QUICK else 40).params.copy()
    q[1::8, 4], q[1::8, 5] = 0.3, 1.0
    q[2::8, 7], q[2::8, 9] = 0.97, 0.02
    q[3::8, 6] = 0.7
    q[4::8, 2] = 2.5
    q[5::8, 1] = 3.0
    c32, f32, c64, f64 = loglike_both(q, w.times, w.t_exp, w.n_ss, w.obs, w.sigma)
    check("flux", f32, f64, 5e-7)
    check("chi2", c32, c64, 1e-4)

    print("all walkers eccentric (generic_unit; fp64: several walkers per cluster), and a multi-round two-transit series")
    B = 200 if QUICK else 600
    e = wl.draw_walkers(B, 5)
    e[:, 4], e[:, 5] = 0.2, rng.uniform(0, 6, B)
    sel = slice(1900, 2000)
    c32, f32, c64, f64 = loglike_both(e, w.times[sel], w.t_exp, 3, w.obs[sel], w.sigma[sel])
    check("flux", f32, f64, 5e-7)
    check("chi2", c32, c64, 1e-4)
    T2 = 40_000
    t2 = np.linspace(-1.2, 1.2, T2) + 542.0 * np.repeat([0.0, 3.0], T2 // 2)
    o2, s2 = 1.0 + 1e-4 * rng.standard_normal(T2), np.full(T2, 1e-4)
    c32, f32, c64, f64 = loglike_both(e[:2], t2, w.t_exp, 2, o2, s2)
    check("flux", f32, f64, 5e-7)
    check("chi2", c32, c64, 1e-4)

    print("more units than grid rows (a CTA loops over walkers)")
    Bm = 66_000
    pw = wl.draw_walkers(Bm, 99)
    ts = w.times[1946:1954]
    c32, f32, c64, f64 = loglike_both(pw, ts, w.t_exp, 1, w.obs[1946:1954], w.sigma[1946:1954])
    check("flux", f32, f64, 5e-7)
    # (eight in-transit points, some walkers fit them to a few sigma: chi^2 ~ 100 moves by 2 r dF/sigma
    # per point, 2e-2 for the 3e-8 of the fp32 flux -- 2e-4 of such a chi^2; config-sized series: 1e-6)
    check("chi2", c32, c64, 1e-3)

    print("extended rows (triaxial, tidally locked): transit_kernel<EX>")
    ext = np.tile([0.3, 0.9, 1.1, 1.0], (6, 1))
    pe = np.concatenate([w.params[:6], ext], axis=1)
    pe[::2, 15] = 0.0
    c32, f32, c64, f64 = loglike_both(pe, w.times[sel], w.t_exp, 3, w.obs[sel], w.sigma[sel], ex=True)
    check("flux", f32, f64, 5e-7)
    check("chi2", c32, c64, 1e-4)

    print("GP likelihood (flux kernels + parallel-in-time scan, PDL chain)")
    gp = np.tile([2e-4, 0.5, 1e-4], (6, 1))
    tt = w.times[1800:2100]
    l32 = gl.gl_gp_loglike(dev(w.params[:6]), dev(tt), w.t_exp, 3, dev(w.obs[1800:2100]), dev(w.sigma[1800:2100]),
                           dev(gp), dtype="f32")
    l64 = gl.gl_gp_loglike(dev(w.params[:6]), dev(tt), w.t_exp, 3, dev(w.obs[1800:2100]), dev(w.sigma[1800:2100]),
                           dev(gp), dtype="f64")
    torch.cuda.synchronize()
    check("lnL", l32, l64, 1e-4)

    print("resident series: host call (mapped params / chi2), device call (graph capture + replay)")
    ser = gl.GlSeries(w.times, w.obs, w.sigma, w.t_exp, w.n_ss, B_max=64)
    _, _, c64, f64 = loglike_both(q, w.times, w.t_exp, w.n_ss, w.obs, w.sigma)
    for _ in range(2):
        ch, fh = ser.loglike(q, want_flux=True)
        check("host flux", torch.as_tensor(fh), f64, 5e-7)
        check("host chi2", torch.as_tensor(ch), c64, 1e-4)
    for _ in range(3):
        cd, fd = ser.loglike_dev(dev(q), want_flux=True)
        torch.cuda.synchronize()
    check("dev flux", fd, f64, 5e-7)
    check("dev chi2", cd, c64, 1e-4)
    ser.close()

    print("bare geometries: binned fp32 kernel, fp64 kernel, the paper's snap + Simpson kernel")
    geom, _ = wl.config5(N=4_000 if QUICK else 40_000)
    g32 = gl.gl_flux_geometry(dev(geom), dtype="f32")
    g64 = gl.gl_flux_geometry(dev(geom), dtype="f64")
    s32 = gl.gl_flux_geometry_simpson(dev(geom[:500]), 512, dtype="f32")
    torch.cuda.synchronize()
    check("geometry", g32, g64, 5e-7)
    assert torch.isfinite(s32).all()
    if _opt("--dump"):
        np.savez(_opt("--dump"), **RESULTS)
    print("sanitizer_shapes: all launches done and consistent")


if __name__ == "__main__":
    main()
