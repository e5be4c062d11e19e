#!/usr/bin/env python
"""bench.py -- throughput of the fused oblate-transit kernel on BASELINE.json's headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg4] [--impl reference]

One step = one pass of the whole hot path (prelude, Kepler/position, crossings, boundary integrals,
exposure mean, chi^2) over one batch: gl_loglike with flux output, i.e. chi2[B] and flux[B,T].
Default workload: config 3 of BASELINE.json (B=256 walkers x T=3900 x 15 sub-exposures, fp32), the
configuration the metric's ">= 40 % of FP32 SIMT peak" is quoted on.  Prints ONE JSON line.
See DESIGN.md "Measurement" for what every key means and how the roofline numbers are formed.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from paper_2410_05408_b200 import workloads as wl  # noqa: E402

METRIC = "oblate-transit flux evals/sec (fp32, quad LD)"
UNIT = "flux evals/s"
# FP32 SIMT peak of a B200: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x SM clock.
N_SM, LANES = 148, 128
# Algorithmic fp32 flop per in-transit sub-exposure (operation count of the scheme with the whole
# outline inside the disc); limb-crossing samples need ~1050, so this undercounts.
ALG_FLOP_PER_SUBSAMPLE = 750.0
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of transit_kernel<float>, from the
# `ncu --set full` captures summarised in profiles/r01_v5.md (not measured live: ncu is not run here)
NCU_DRAM_BYTES = {"cfg3": 232_704 + 0, "cfg4": 606_464 + 15_872}


def make_workload(name, rank):
    if name == "cfg3":
        w = wl.config3()
        if rank:
            w.params = wl.draw_walkers(w.B, wl.SEED_CFG3_WALKERS + 1000 * rank)
    elif name == "cfg4":
        w = wl.config4()
        if rank:
            w.params = wl.draw_walkers(w.B, wl.SEED_CFG4_WALKERS + 1000 * rank)
    elif name in ("cfg4ex_free", "cfg4ex_locked"):
        # NEXT-2 context lines: config 4's batch with the extended rows of gl_loglike_ex (triaxial
        # axes 1 : 0.9 : 1.1 x (1-f), zeta = 0.3 rad), orientation free or tidally locked
        w = wl.config4()
        if rank:
            w.params = wl.draw_walkers(w.B, wl.SEED_CFG4_WALKERS + 1000 * rank)
        ext = np.tile([0.3, 0.9, 1.1, 1.0 if name.endswith("locked") else 0.0], (w.B, 1))
        w.params = np.concatenate([w.params, ext], axis=1)
        w.name = w.name.replace("cfg4", name)
    else:
        raise SystemExit(f"unknown workload {name}")
    return w


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


def oracle_timed(w, repeat=1):
    """The CPU oracle as it stands, all host cores, on the whole workload."""
    import oracle as orc
    orc.build()
    t0 = time.perf_counter()
    used = 0
    for _ in range(repeat):
        _, _, used = orc.loglike(w.params, w.times, w.t_exp, w.n_ss, w.obs, w.sigma,
                                 return_threads=True)
    dt = (time.perf_counter() - t0) / repeat
    return w.B * w.T / dt, used, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload, 0)
    for _ in range(min(args.warmup, 1)):
        oracle_timed(w)
    times = []
    used = 0
    for _ in range(args.steps):
        v, used, dt = oracle_timed(w)
        times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = w.B * w.T / (ms * 1e-3)
    sample = f"whole workload {w.name} (B={w.B}, T={w.T}, S={w.n_ss}) per step, OpenMP over (walker,time)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": w.name, "B": w.B, "T": w.T, "n_ss": w.n_ss},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg3",
                    choices=["cfg3", "cfg4", "cfg4ex_free", "cfg4ex_locked"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2410_05408_b200 as gl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    gl.load_library()
    W = max(args.warmup, 3)
    K = args.steps

    w = make_workload(args.workload, rank)
    d = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device=dev)  # noqa: E731
    P, Tm, O, S = d(w.params), d(w.times), d(w.obs), d(w.sigma)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    extended = w.params.shape[1] == 16
    loglike = gl.gl_loglike_ex if extended else gl.gl_loglike

    def step():
        return loglike(P, Tm, w.t_exp, w.n_ss, O, S, dtype="f32", want_flux=True)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        chi2, flux = step()
    torch.cuda.synchronize()
    n_in_exposures = int((flux < 1.0).sum().item())
    launches0 = gl.gl_launch_count()

    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(K)]
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    barrier()
    wall0 = time.perf_counter()
    for a, b in ev:
        flush.zero_()                 # L2 flush between timed iterations (outside the event pair)
        a.record()
        step()
        b.record()
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    launches = gl.gl_launch_count() - launches0
    # the same K steps with the L2 left warm (context only: a spinning spacer kernel, no memory
    # traffic, lets the host run ahead so that the event pair sees GPU time, not submission gaps)
    ev_w = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
            for _ in range(K)]
    for a, b in ev_w:
        torch.cuda._sleep(200_000)
        a.record()
        step()
        b.record()
    torch.cuda.synchronize()
    warm_ms = float(np.mean([a.elapsed_time(b) for a, b in ev_w]))
    dev_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(np.sum(dev_ms))
    tmax = torch.tensor([total_ms], device=dev, dtype=torch.float64)
    if dist is not None:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    total_ms_max = float(tmax.item())
    ms_per_step = total_ms_max / K
    evals_per_step = w.B * w.T * world
    value = evals_per_step / (ms_per_step * 1e-3)

    # ---- end to end through the HOST-buffer C ABI call, pinned host memory, copies timed
    pin = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64)).pin_memory().numpy()  # noqa: E731
    hp, ht, ho, hs = pin(w.params), pin(w.times), pin(w.obs), pin(w.sigma)
    c_h = torch.empty(w.B, dtype=torch.float32).pin_memory().numpy()          # pinned outputs too
    f_h = torch.empty((w.B, w.T), dtype=torch.float32).pin_memory().numpy()
    if extended:
        # no host-pointer variant of the _ex entry points: the same copies, issued from here
        pins = [torch.from_numpy(x) for x in (hp, ht, ho, hs)]
        c_t, f_t = torch.from_numpy(c_h), torch.from_numpy(f_h)

        def e2e_call():
            for dst, src in zip((P, Tm, O, S), pins):
                dst.copy_(src, non_blocking=True)
            chi2_d, flux_d = step()
            c_t.copy_(chi2_d, non_blocking=True)
            f_t.copy_(flux_d, non_blocking=True)
            torch.cuda.synchronize()
        api = "gl_loglike_ex + pinned H2D/D2H copies issued by bench.py (wall clock over K calls)"
    else:
        def e2e_call():
            gl.gl_loglike_host(hp, ht, w.t_exp, w.n_ss, ho, hs, dtype="f32", want_flux=True,
                               chi2_out=c_h, flux_out=f_h)
        api = "gl_loglike_host (pinned host inputs and outputs, wall clock over K calls)"
    for _ in range(3):
        e2e_call()
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        e2e_call()
    e2e_s = time.perf_counter() - t0
    te = torch.tensor([e2e_s], device=dev, dtype=torch.float64)
    if dist is not None:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_value = evals_per_step * K / float(te.item())
    h2d = int(hp.nbytes + ht.nbytes + ho.nbytes + hs.nbytes)
    d2h = int(c_h.nbytes + f_h.nbytes)
    # what an MCMC caller needs back is chi2[B] alone (flux never leaves the GPU): same call, no flux
    e2e_chi2_only = None
    if not extended:
        for _ in range(3):
            gl.gl_loglike_host(hp, ht, w.t_exp, w.n_ss, ho, hs, dtype="f32", chi2_out=c_h)
        barrier()
        t0 = time.perf_counter()
        for _ in range(K):
            gl.gl_loglike_host(hp, ht, w.t_exp, w.n_ss, ho, hs, dtype="f32", chi2_out=c_h)
        tc = torch.tensor([time.perf_counter() - t0], device=dev, dtype=torch.float64)
        if dist is not None:
            dist.all_reduce(tc, op=dist.ReduceOp.MAX)
        e2e_chi2_only = evals_per_step * K / float(tc.item())

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the (only) kernel: plain FP32 ALU work
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak_tflops = N_SM * LANES * 2 * sm_max * 1e6 / 1e12
    probe = gl.gl_probe_peaks()      # FFMA / DFMA / MUFU chain kernels, measured now, on this GPU
    k_ms = float(np.mean(dev_ms))
    n_sub_in = n_in_exposures * w.n_ss
    alg_flop = ALG_FLOP_PER_SUBSAMPLE * n_sub_in
    achieved = alg_flop / (k_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops, "traffic": NCU_DRAM_BYTES.get(args.workload),
                "traffic_unit": "bytes per launch (ncu --set full, profiles/r01_v5.md); the path is "
                                "ALU-bound, algorithmic HBM bytes are B*96 + T*24 in, B*T*4 + B*4 out",
                "kernel": "transit_kernel<float> (+ one-CTA baseline_kernel, overlapped by "
                          "programmatic dependent launch)", "kernel_ms": k_ms,
                "kernel_ms_warm_l2": warm_ms,
                "peak_source": f"derived: {N_SM} SMs x {LANES} FP32 lanes x 2 x {sm_max:.0f} MHz "
                               "(MEASURED_PEAKS.json has no FP32 SIMT figure)",
                "peak_measured_ffma_chain": probe["fp32_tflops"],
                "frac_of_measured_peak": achieved / probe["fp32_tflops"],
                "fp64_dfma_chain_tflops": probe["fp64_tflops"], "mufu_chain_tops": probe["mufu_tops"],
                "alg_flop_per_in_transit_subsample": ALG_FLOP_PER_SUBSAMPLE,
                "in_transit_subsamples_per_launch": n_sub_in,
                "in_transit_fraction": n_sub_in / (w.B * w.T * w.n_ss),
                "in_transit_subsamples_per_s": n_sub_in / (k_ms * 1e-3)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "B": w.B, "T": w.T, "n_ss": w.n_ss, "outputs": "chi2[B]+flux[B,T]",
                   "l2": "256 MiB flush between timed iterations", "parallelism": f"dp{world} over walkers"},
        "subsample_evals_per_s": value * w.n_ss,
        "wall_ms_per_step_incl_flush": 1e3 * wall / K,
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "api": api,
                "chi2_only_value": e2e_chi2_only, "chi2_only_d2h_bytes_per_step": int(c_h.nbytes)},
        "roofline": roofline,
    }
    if world == 1 and not args.no_cpu_baseline and not extended:
        v, used, dt = oracle_timed(w, repeat=1)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": used, "kind": "oracle",
                               "sample": f"whole workload {w.name} once ({dt:.2f} s), OpenMP over (walker,time)"}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
