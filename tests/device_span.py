"""On-device span of one hot_kernel launch (first CTA's first stamp -> last chi^2 write), by %globaltimer:

    python tests/device_span.py --lib <library built with -include tests/span_hooks.cuh> [cfg3 cfg2 cfg4]

Run by tests/test_gpu_parity.py::test_device_span_of_one_step (which builds that library); prints one JSON
object: per workload and mode (chi2+flux / chi2 only; L2 flushed / warm) the mean, min and max span in
microseconds over 20 launches and the CUDA-event time of the same launches.  Test infrastructure: not
collected by pytest, not used by the product.
"""
import ctypes
import json
import sys
from pathlib import Path

import numpy as np
import torch

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))
from paper_2410_05408_b200 import binding  # noqa: E402

binding._LIBPATH = Path(sys.argv[sys.argv.index("--lib") + 1])
import paper_2410_05408_b200 as gl  # noqa: E402
from paper_2410_05408_b200 import workloads as wl  # noqa: E402


def main():
    lib = gl.load_library()
    dev = torch.device("cuda:0")
    d = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device=dev)  # noqa: E731
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    out = (ctypes.c_ulonglong * 2)()
    names = [a for a in sys.argv[1:] if a.startswith("cfg")] or ["cfg3", "cfg2", "cfg4"]
    res = {}
    for name in names:
        w = wl.get(name)
        P = d(w.params)
        ser = gl.GlSeries(w.times, w.obs, w.sigma, w.t_exp, w.n_ss, w.B)
        chi2 = torch.empty(w.B, dtype=torch.float32, device=dev)
        flux = torch.empty((w.B, w.T), dtype=torch.float32, device=dev)
        calls = {"chi2+flux": lambda: ser.loglike_dev(P, want_flux=True, chi2_out=chi2, flux_out=flux),
                 "chi2": lambda: ser.loglike_dev(P, chi2_out=chi2)}
        for mode, fn in calls.items():
            for cold in (True, False):
                spans, evs = [], []
                for it in range(25):
                    spacer = flush.zero_ if cold else (lambda: torch.cuda._sleep(100_000))
                    spacer()
                    torch.cuda.synchronize()
                    assert lib.gl_debug_span(out, 1) == 0
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    spacer()
                    a.record()
                    fn()
                    b.record()
                    torch.cuda.synchronize()
                    assert lib.gl_debug_span(out, 0) == 0
                    if it >= 5:
                        spans.append((out[1] - out[0]) * 1e-3)
                        evs.append(a.elapsed_time(b) * 1e3)
                res[f"{name} {mode} {'L2 flushed' if cold else 'L2 warm'}"] = {
                    "span_us_mean": round(float(np.mean(spans)), 2), "span_us_min": round(float(np.min(spans)), 2),
                    "span_us_max": round(float(np.max(spans)), 2), "event_us_mean": round(float(np.mean(evs)), 2)}
        ser.close()
    print(json.dumps(res))


if __name__ == "__main__":
    main()
