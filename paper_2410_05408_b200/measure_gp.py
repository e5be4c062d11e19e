"""NEXT-4 measurement: time of gl_gp_loglike (transit kernel + Kalman-filter likelihood kernel) beside
gl_loglike (chi^2) on the K2- and JWST-shaped batches.

    python -m paper_2410_05408_b200.measure_gp

CUDA events, L2 flushed between steps, inputs resident in HBM.  Needs a CUDA device."""
from __future__ import annotations

import numpy as np


def main():
    import torch
    from . import binding as gl
    from . import workloads as wl

    gl.load_library()
    dev = torch.device("cuda:0")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    print("| workload | call | us per step | flux evals/s |")
    print("|---|---|---|---|")
    for w in (wl.config3(), wl.config4()):
        d = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device=dev)  # noqa: E731
        P, Tm, O, S = d(w.params), d(w.times), d(w.obs), d(w.sigma)
        rng = np.random.default_rng(3)
        gp = d(np.column_stack([rng.uniform(0.5, 2.0, w.B) * w.sigma[0],
                                rng.uniform(0.05, 0.5, w.B), np.full(w.B, 0.3 * w.sigma[0])]))
        calls = {
            "gl_loglike (chi^2 + flux)": lambda: gl.gl_loglike(P, Tm, w.t_exp, w.n_ss, O, S, "f32", True),
            "gl_gp_loglike (GP + flux)": lambda: gl.gl_gp_loglike(P, Tm, w.t_exp, w.n_ss, O, S, gp, "f32", True),
        }
        for name, fn in calls.items():
            for _ in range(3):
                fn()
            torch.cuda.synchronize()
            ts = []
            for _ in range(20):
                flush.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fn()
                b.record()
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b) * 1e3)
            us = float(np.mean(ts))
            print(f"| {w.name} | {name} | {us:.1f} | {w.B * w.T / (us * 1e-6):.3g} |")


if __name__ == "__main__":
    main()
