"""NEXT-1 measurement: the paper's snap + Simpson kernel beside the production crossings + closed-form
kernel, on config 5's geometry mix.

    python -m paper_2410_05408_b200.compare_simpson [--rows 1000000] [--sample 50000]

Prints a markdown report: (1) max |dflux| of the Simpson kernel against the fp64 production kernel
(itself within 1e-11 of the CPU oracle, tests/test_gpu_parity.py) as a function of the number of
Simpson intervals, per geometry class; (2) time per geometry of both kernels in fp32 (CUDA events,
whole config-5 batch resident in HBM).  Needs a CUDA device; no CPU fallback.
"""
from __future__ import annotations

import argparse

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--rows", type=int, default=1_000_000)
    ap.add_argument("--sample", type=int, default=50_000)
    args = ap.parse_args()
    import torch
    from . import binding as gl
    from . import workloads as wl

    gl.load_library()
    dev = torch.device("cuda:0")
    geom, cls = wl.config5(N=args.rows)
    names = ["random draw", "external tangency", "internal tangency", "centre on the limb",
             "four crossings"]

    def timed(fn, reps=5):
        fn()
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            torch.cuda.synchronize()
            best = min(best, a.elapsed_time(b))
        return best

    # ---- accuracy versus node count, on a sample that keeps the class mix
    idx = np.sort(np.random.default_rng(1).choice(args.rows, min(args.sample, args.rows), replace=False))
    gs = torch.as_tensor(geom[idx], device=dev)
    cs = cls[idx]
    exact = gl.gl_flux_geometry(gs, "f64").cpu().numpy()
    prod32 = gl.gl_flux_geometry(gs, "f32").double().cpu().numpy()
    print("## Accuracy: max |flux - exact| on %d config-5 rows (exact = fp64 production kernel)\n" % len(idx))
    print("| kernel | " + " | ".join(names) + " |")
    print("|---|" + "---|" * len(names))
    row = ["%.1e" % np.abs(prod32 - exact)[cs == c].max() for c in range(5)]
    print("| production fp32 (6-32 nodes) | " + " | ".join(row) + " |")
    for n in (64, 256, 1024, 4096, 16384, 65536):
        for dt in ("f32", "f64"):
            out = gl.gl_flux_geometry_simpson(gs, n, dt).double().cpu().numpy()
            row = ["%.1e" % np.abs(out - exact)[cs == c].max() for c in range(5)]
            print("| snap + Simpson, %d intervals, %s | " % (n, dt) + " | ".join(row) + " |")

    # ---- time per geometry, whole batch
    g = torch.as_tensor(geom, device=dev)
    print("\n## Time: %d config-5 rows, fp32, best of 5 (CUDA events)\n" % args.rows)
    print("| kernel | ms | ns per geometry | geometries/s |")
    print("|---|---|---|---|")
    ms = timed(lambda: gl.gl_flux_geometry(g, "f32"))
    print("| production (crossings + closed forms + fixed-node rules) | %.3f | %.2f | %.3g |"
          % (ms, 1e6 * ms / args.rows, args.rows / (ms * 1e-3)))
    for n in (256, 1024, 4096, 16384):
        ms = timed(lambda: gl.gl_flux_geometry_simpson(g, n, "f32"), reps=3)
        print("| snap + Simpson, %d intervals, one warp per geometry | %.3f | %.2f | %.3g |"
              % (n, ms, 1e6 * ms / args.rows, args.rows / (ms * 1e-3)))


if __name__ == "__main__":
    main()
