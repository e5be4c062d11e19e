"""Per-CTA phase timeline of one fused launch (development aid cited by profiles/r01_v*.md).

    python -m paper_2410_05408_b200.timeline [cfg3|cfg4] [--no-flush] [--chi2-only]

Builds csrc/greenlantern_b200.cu with -DGL_TIMELINE into a temporary directory (the product library
is untouched): every CTA of transit_kernel then records %globaltimer at its phase boundaries
(start, prelude done, list built, first cluster barrier passed, evaluation done, CTA sum done,
second barrier passed, exit) into a device array, maximum over its warps.  Prints, over all CTAs,
the distribution of each time stamp and of each phase length in microseconds.
"""
from __future__ import annotations

import argparse
import ctypes
import subprocess
import tempfile
from pathlib import Path

import numpy as np

NAMES = ["start", "prelude_done", "list_built", "barrier1_passed", "eval_done", "cta_sum_done",
         "barrier2_passed", "exit"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("workload", nargs="?", default="cfg3", choices=["cfg3", "cfg4"])
    ap.add_argument("--no-flush", action="store_true", help="leave the L2 warm before the measured launch")
    ap.add_argument("--chi2-only", action="store_true", help="no flux output")
    args = ap.parse_args()
    import torch
    from . import binding, build, workloads as wl

    tmp = Path(tempfile.mkdtemp(prefix="gl_timeline_")) / "libgreenlantern_timeline.so"
    subprocess.run([build._nvcc(), *build.NVCC_FLAGS, "-DGL_TIMELINE", "-o", str(tmp),
                    *map(str, build.SOURCES)], check=True)
    binding._LIBPATH = tmp
    lib = binding.load_library()
    lib.gl_debug_timeline.argtypes = [ctypes.c_void_p, ctypes.c_int]
    w = wl.config3() if args.workload == "cfg3" else wl.config4()
    dev = torch.device("cuda:0")
    P, Tm, O, S = (torch.as_tensor(np.ascontiguousarray(x), device=dev)
                   for x in (w.params, w.times, w.obs, w.sigma))

    def call():
        return binding.gl_loglike(P, Tm, w.t_exp, w.n_ss, O, S, dtype="f32", want_flux=not args.chi2_only)

    for _ in range(3):
        call()
    torch.cuda.synchronize()
    lib.gl_debug_timeline(None, 1)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    if not args.no_flush:
        flush.zero_()
    torch.cuda.synchronize()
    call()
    torch.cuda.synchronize()
    buf = np.zeros(8192 * 8, dtype=np.int64)
    lib.gl_debug_timeline(buf.ctypes.data, 0)
    tl = buf.reshape(8192, 8)
    tl = tl[tl[:, 0] > 0]
    rel = (tl - tl[:, 0].min()) / 1000.0
    print(f"{w.name}: {len(tl)} CTAs, L2 {'warm' if args.no_flush else 'flushed'}, "
          f"{'chi2 only' if args.chi2_only else 'chi2 + flux'}  (microseconds since the first CTA started)")
    for k, n in enumerate(NAMES):
        v = rel[:, k]
        print(f"  {n:16s} min {v.min():7.2f}  median {np.median(v):7.2f}  p90 {np.quantile(v, 0.9):7.2f}  max {v.max():7.2f}")
    d = np.diff(rel, axis=1)
    for k in range(7):
        v = d[:, k]
        print(f"  phase {NAMES[k]} -> {NAMES[k + 1]}: median {np.median(v):6.2f}  p90 {np.quantile(v, 0.9):6.2f}  max {v.max():6.2f}")


if __name__ == "__main__":
    main()
