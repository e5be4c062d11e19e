#!/usr/bin/env python
"""bench.py -- throughput of the fused oblate-transit path on BASELINE.json's headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg4] [--impl reference]
                    [--no-extra] [--no-cpu-baseline] [--dry]

One step = one pass of the whole hot path (prelude, position, crossings, boundary integrals,
exposure mean, chi^2) over one batch: chi2[B] AND flux[B,T] for B walkers against a resident series
(gl_series_loglike_dev: the series was uploaded once, the parameter rows are resident in HBM).
Default workload: config 3 of BASELINE.json (B=256 walkers x T=3900 x 15 sub-exposures, fp32), the
configuration the metric's ">= 40 % of FP32 SIMT peak" is quoted on.  Prints ONE JSON line.
`extra` carries the other workloads (cfg4, cfg5, cfg3 in fp64, cfg3 with every walker eccentric, cfg3's series
with 4096 walkers, the GP
likelihood, the paper's snap + Simpson kernel, one light curve of 1e5 exposures, the stateless
gl_loglike call) timed the same way in the same run; `roofline.event_time_vs_kernel_time` shows how the
event timer of this hardware quantises a kernel's duration.
`--gpus N` without a torchrun environment starts N ranks itself (torch.distributed.run on
127.0.0.1); `--dry` exercises that plumbing on a CPU box with the gloo backend and no kernels.
See DESIGN.md section 6 for what every key means and how the roofline numbers are formed.
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
# Algorithmic fp32 flop per in-transit sub-exposure: 1.0-1.1 kflop with the outline
# inside the disc (16 f_lin nodes x 60-70 flop + ~100), 1.4-1.6 kflop when it crosses the limb (root
# isolation + polishing + atan2).  Mid-points; the mix is counted per workload from the sky distance.
ALG_FLOP_INSIDE, ALG_FLOP_LIMB = 1050.0, 1500.0
NCU_FILE = ROOT / "profiles" / "r02_ncu_constants.json.txt"


def ncu_constants():
    """Counters of the SHIPPED kernels from the committed ncu captures (profiles/r02_kernels.md), keyed
    by the commit they were captured at; bench.py cannot run ncu itself."""
    try:
        return json.loads(NCU_FILE.read_text())
    except (OSError, ValueError):
        return {}


def make_workload(name, rank):
    if name == "cfg3":
        w = wl.config3()
        if rank:
            w.params = wl.draw_walkers(w.B, wl.SEED_CFG3_WALKERS + 1000 * rank)
    elif name == "cfg4":
        w = wl.config4()
        if rank:
            w.params = wl.draw_walkers(w.B, wl.SEED_CFG4_WALKERS + 1000 * rank)
    else:
        raise SystemExit(f"unknown workload {name}")
    return w


def in_transit_mix(w):
    """(in-transit sub-exposures, of which the outline crosses the limb) for circular walkers, from the
    sky distance of the planet centre alone (eqs. 9-10): bookkeeping for the
    algorithmic flop count, not part of any timed path."""
    p = w.params
    offs = ((np.arange(w.n_ss) + 0.5) / w.n_ss - 0.5) * w.t_exp
    n_in = n_limb = 0
    for row in p:
        t0, P, aR, b, rp = row[0], row[1], row[2], row[3], row[6]
        ph = (w.times[:, None] + offs[None, :] - t0) / P
        ph -= np.rint(ph)
        near = np.abs(ph) < 0.25
        phi = 2.0 * np.pi * ph[near]
        r0 = np.hypot(b * np.cos(phi), aR * np.sin(phi))
        n_in += int((r0 < 1.0 + rp).sum())
        n_limb += int(((r0 < 1.0 + rp) & (r0 > 1.0 - rp)).sum())
    return n_in, n_limb


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
                 "--format=csv,noheader,nounits", "-lms", "100"],
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


# ---------------------------------------------------------------------------------------------
# reference arm = the oracle (tier rules): timed as it stands on the host cores
# ---------------------------------------------------------------------------------------------
def oracle_timed(w, nthreads=0, rows=None):
    """The CPU oracle as it stands on `rows` walkers of the workload (all if None)."""
    import oracle as orc
    orc.build()
    p = w.params if rows is None else w.params[:rows]
    t0 = time.perf_counter()
    _, _, used = orc.loglike(p, w.times, w.t_exp, w.n_ss, w.obs, w.sigma, nthreads=nthreads,
                             return_threads=True)
    dt = time.perf_counter() - t0
    return p.shape[0] * w.T / dt, used, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload, 0)
    W = min(args.warmup, 1)
    for _ in range(W):
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
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
        "n_gpus": int(os.environ.get("WORLD_SIZE", args.gpus)),
        "steps": args.steps, "warmup": W, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": w.name, "B": w.B, "T": w.T, "n_ss": w.n_ss},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------
# multi-rank plumbing
# ---------------------------------------------------------------------------------------------
def spawn_ranks(args):
    """--gpus N outside torchrun: start N ranks on this node (one process per GPU) and relay rank 0's
    JSON line."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve()),
           *sys.argv[1:]]
    return subprocess.call(cmd)


def run_dry(args, world, rank):
    """The multi-rank code path without a GPU (tests/test_multirank_host.py): sharded walker draw,
    barrier, max-over-ranks of a per-rank time, one JSON line from rank 0."""
    import torch
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("gloo")
    w = make_workload(args.workload, rank)
    t = torch.tensor([1.0 + rank], dtype=torch.float64)     # stand-in for the per-rank device time [ms]
    shard = torch.tensor([float(w.params[:, 0].sum())], dtype=torch.float64)
    gathered = [torch.zeros_like(shard) for _ in range(world)]
    if world > 1:
        dist.barrier()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_gather(gathered, shard)
    else:
        gathered = [shard]
    if rank == 0:
        print(json.dumps({"metric": METRIC, "dry": True, "n_gpus": world, "steps": args.steps,
                          "ms_per_step": float(t.item()), "value": w.B * w.T * world / (float(t.item()) * 1e-3),
                          "unit": UNIT, "scaling": "weak",
                          "distinct_shards": len({round(float(g.item()), 9) for g in gathered}),
                          "config": {"workload": w.name, "parallelism": f"dp{world} over walkers"}}))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg3", choices=["cfg3", "cfg4"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true")
    ap.add_argument("--dry", action="store_true", help="multi-rank plumbing only (gloo, no GPU)")
    ap.add_argument("--profile", default=None, help="run one named call five times and exit (for ncu)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.profile:
        return run_profile(args)
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        raise SystemExit(spawn_ranks(args))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.dry:
        return run_dry(args, world, rank)

    import torch
    import paper_2410_05408_b200 as gl

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

    d = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device=dev)  # noqa: E731
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, k=K, warm=W, cold=True):
        """CUDA events around each of k calls on torch's current stream (the launching stream); L2
        flushed before each call (cold) or a spinning spacer kernel instead (warm L2, context)."""
        for _ in range(warm):
            if cold:
                flush.zero_()
            fn()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
        for a, b in ev:
            if cold:
                flush.zero_()
            else:
                torch.cuda._sleep(200_000)
            a.record()
            fn()
            b.record()
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    w = make_workload(args.workload, rank)
    P = d(w.params)
    ser = gl.GlSeries(w.times, w.obs, w.sigma, w.t_exp, w.n_ss, w.B, device=dev)
    chi2_d = torch.empty(w.B, dtype=torch.float32, device=dev)
    flux_d = torch.empty((w.B, w.T), dtype=torch.float32, device=dev)

    def step():
        ser.loglike_dev(P, want_flux=True, chi2_out=chi2_d, flux_out=flux_d)

    step()
    torch.cuda.synchronize()
    n_in_exposures = int((flux_d < 1.0).sum().item())
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.5)                # nvidia-smi is up and sampling before anything is timed
    for _ in range(W):             # W untimed warm-up steps, in the timed loop's own rhythm (flush, step)
        flush.zero_()
        step()
    torch.cuda.synchronize()
    launches0 = gl.gl_launch_count()
    barrier()
    wall0 = time.perf_counter()
    dev_ms = timed(step, warm=0)
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    launches = gl.gl_launch_count() - launches0
    warm_ms = float(np.mean(timed(step, warm=0, cold=False)))
    total_ms = float(np.sum(dev_ms))
    tmax = torch.tensor([total_ms], device=dev, dtype=torch.float64)
    if dist is not None:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    ms_per_step = float(tmax.item()) / K
    evals_per_step = w.B * w.T * world
    value = evals_per_step / (ms_per_step * 1e-3)

    # ---- end to end: HOST parameter rows in, HOST chi^2 (and flux) out, through gl_series_loglike
    hp = torch.as_tensor(np.ascontiguousarray(w.params)).pin_memory().numpy()
    c_h = torch.empty(w.B, dtype=torch.float32).pin_memory().numpy()
    f_h = torch.empty((w.B, w.T), dtype=torch.float32).pin_memory().numpy()

    def wall_per_call(fn):
        for _ in range(3):
            fn()
        barrier()
        t0 = time.perf_counter()
        for _ in range(K):
            fn()
        t = torch.tensor([time.perf_counter() - t0], device=dev, dtype=torch.float64)
        if dist is not None:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item()) / K

    e2e_s = wall_per_call(lambda: ser.loglike(hp, want_flux=True, chi2_out=c_h, flux_out=f_h))
    e2e_chi2_s = wall_per_call(lambda: ser.loglike(hp, chi2_out=c_h))
    h2d = int(hp.nbytes)
    d2h = int(c_h.nbytes + f_h.nbytes)

    if rank != 0:
        ser.close()
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (hot_kernel): plain FP32 ALU work
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak_tflops = N_SM * LANES * 2 * sm_max * 1e6 / 1e12
    probe = gl.gl_probe_peaks()      # FFMA / DFMA / MUFU chain kernels, measured now, on this GPU
    ncu = ncu_constants()

    def fractions(workload_key, n_in, n_limb, ms):
        alg = ALG_FLOP_INSIDE * (n_in - n_limb) + ALG_FLOP_LIMB * n_limb
        out = {"alg_flop": alg, "alg_tflops": alg / (ms * 1e-3) / 1e12,
               "frac_alg": alg / (ms * 1e-3) / 1e12 / peak_tflops}
        ex = ncu.get("executed_fp32_flop", {}).get(workload_key)
        if ex:
            out["executed_flop_ncu"] = ex
            out["frac_executed"] = ex / (ms * 1e-3) / 1e12 / peak_tflops
        return out

    k_ms = float(np.mean(dev_ms))
    n_in, n_limb = in_transit_mix(w)
    fr = fractions(args.workload, n_in, n_limb, k_ms)
    hs = (1, w.B, 512)               # hot_kernel's launch shape for this batch: (cluster, rows, threads)
    floor_graph = float(np.mean(timed(lambda: gl.gl_probe_empty_graph(hs[0], hs[1], hs[2]), k=max(K, 20))))
    floor_stream = float(np.mean(timed(lambda: gl.gl_probe_empty_launch(hs[0], hs[1], hs[2]), k=max(K, 20))))
    # How the event-timed duration answers to the kernel's real duration on this box: a one-thread kernel
    # that spins for a known number of SM cycles (torch.cuda._sleep), timed exactly like a step.
    sm_hz = (clocks.get("sm_mhz") or sm_max) * 1e6
    stair_spin_us = [0.0, 2.0, 4.0, 6.0, 8.0, 9.0, 10.0, 11.0, 12.0, 13.0, 14.0]
    stair_event_us = [1e3 * float(np.mean(timed(lambda c=int(us * 1e-6 * sm_hz): torch.cuda._sleep(c), k=12, warm=2)))
                      for us in stair_spin_us]
    roofline = {
        "bound": "alu", "achieved": fr["alg_tflops"], "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": fr["frac_alg"],
        "frac_label": "ALGORITHMIC flop (SURVEY.md 8(d): 1050 per in-transit sub-exposure inside the disc, "
                      "1500 on the limb) / CUDA-event step time / derived peak",
        "frac_executed": fr.get("frac_executed"),
        "frac_executed_label": "fp32 flop the kernel EXECUTES (ncu: FADD + FMUL + 2 FFMA thread instructions, "
                               f"capture of commit {ncu.get('commit')}) / step time / derived peak",
        "traffic": ncu.get("dram_bytes", {}).get(args.workload),
        "traffic_source": f"dram__bytes_read.sum + dram__bytes_write.sum of one hot_kernel launch, ncu --set full "
                          f"at commit {ncu.get('commit')} (profiles/r02_kernels.md); the path is ALU/latency-bound, "
                          "algorithmic HBM bytes are B*96 in, B*T*4 + B*4 out",
        "kernel": "glh::hot_kernel<true> (one launch per step, replayed as a CUDA graph)",
        "kernel_ms": k_ms, "kernel_ms_warm_l2": warm_ms,
        "launch_floor_ms": floor_graph, "launch_floor_stream_launch_ms": floor_stream,
        "launch_floor_note": "an EMPTY kernel of hot_kernel's grid/block shape, replayed as a CUDA graph the way "
                             "a step is (and launched on the stream, for comparison), timed exactly like a step, "
                             "L2 flushed",
        "event_time_vs_kernel_time": {
            "spin_kernel_us": stair_spin_us, "event_timed_us": stair_event_us,
            "note": "CUDA-event time of a one-thread kernel that spins for the given time (torch.cuda._sleep), "
                    "measured like a step.  On the B200s of this pool it is a staircase, about 6.1 us + 2.05 us "
                    "x floor(kernel time / 2.04 us): the end of a kernel is observed on a 2.048-us grid, so "
                    "ms_per_step moves in 2-us treads (14.3, 16.4, 18.4 us) while the kernel changes by tenths "
                    "(profiles/r02_kernels.md, 'Event-time staircase'; on-device span of a step: "
                    "profiles/r02_device_span.md)"},
        "peak_source": f"derived: {N_SM} SMs x {LANES} FP32 lanes x 2 x {sm_max:.0f} MHz "
                       "(MEASURED_PEAKS.json has no FP32 SIMT figure)",
        "peak_measured_ffma_chain": probe["fp32_tflops"],
        "frac_of_measured_peak": fr["alg_tflops"] / probe["fp32_tflops"],
        "fp64_dfma_chain_tflops": probe["fp64_tflops"], "mufu_chain_tops": probe["mufu_tops"],
        "alg_flop_per_in_transit_subsample": {"inside": ALG_FLOP_INSIDE, "limb": ALG_FLOP_LIMB},
        "in_transit_subsamples_per_launch": n_in, "of_which_limb_crossing": n_limb,
        "in_window_exposures_with_flux_below_1": n_in_exposures,
        "in_transit_fraction": n_in / (w.B * w.T * w.n_ss),
        "in_transit_subsamples_per_s": n_in / (k_ms * 1e-3)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "B": w.B, "T": w.T, "n_ss": w.n_ss, "outputs": "chi2[B]+flux[B,T]",
                   "api": "gl_series_loglike_dev (series resident, parameter rows resident)",
                   "l2": "256 MiB flush between timed iterations", "parallelism": f"dp{world} over walkers"},
        "subsample_evals_per_s": value * w.n_ss,
        "ms_per_step_median": float(np.median(dev_ms)), "ms_per_step_min": float(np.min(dev_ms)),
        "ms_per_step_max": float(np.max(dev_ms)),
        "wall_ms_per_step_incl_flush": 1e3 * wall / K,
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": evals_per_step / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h,
                "api": "gl_series_loglike: host parameter rows in, host chi2 + flux out (wall clock over K calls)",
                "ms_per_call": 1e3 * e2e_s,
                "chi2_only_value": evals_per_step / e2e_chi2_s, "chi2_only_ms_per_call": 1e3 * e2e_chi2_s,
                "chi2_only_d2h_bytes_per_step": int(c_h.nbytes)},
        "roofline": roofline,
    }
    if world == 1 and not args.no_extra:
        out["extra"] = extra_workloads(gl, dev, d, timed, fractions, peak_tflops, probe, ncu, w, ser, P)
    ser.close()
    if world == 1 and not args.no_cpu_baseline:
        v, used, dt = oracle_timed(w)
        v1, _, dt1 = oracle_timed(w, nthreads=1, rows=16)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": used, "kind": "oracle",
                               "sample": f"whole workload {w.name} once ({dt:.2f} s), OpenMP over (walker,time)",
                               "single_thread_value": v1,
                               "single_thread_sample": f"first 16 walkers of {w.name}, 1 thread ({dt1:.2f} s)"}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def secondary_calls(gl, dev, d, w3, ser3, P3):
    """name -> (callable that enqueues one call, units per call, unit name, keep-alive objects) for the
    workloads beside the headline: used by `extra` (timed) and by --profile (run a few times under ncu)."""
    import torch
    calls = {}
    T3, O3, S3 = d(w3.times), d(w3.obs), d(w3.sigma)
    chi2_only = torch.empty(w3.B, dtype=torch.float32, device=dev)
    calls["cfg3_gl_loglike_stateless"] = (
        lambda: gl.gl_loglike(P3, T3, w3.t_exp, w3.n_ss, O3, S3, dtype="f32", want_flux=True), w3.B * w3.T, "flux_evals")
    calls["cfg3_chi2_only"] = (lambda: ser3.loglike_dev(P3, chi2_out=chi2_only), w3.B * w3.T, "flux_evals")
    # the same batch with every walker on an eccentric orbit (e = 0.2, omega uniform): off hot_kernel's common
    # path, same single launch (generic_unit: Kepler's equation per sub-exposure)
    pe = w3.params.copy()
    pe[:, 4] = 0.2
    pe[:, 5] = np.random.default_rng(wl.SEED_CFG3_WALKERS + 7).uniform(0.0, 2.0 * np.pi, w3.B)
    P3e = d(pe)
    chi2_e = torch.empty(w3.B, dtype=torch.float32, device=dev)
    flux_e = torch.empty((w3.B, w3.T), dtype=torch.float32, device=dev)
    calls["cfg3_all_walkers_eccentric_e0.2"] = (
        lambda: ser3.loglike_dev(P3e, want_flux=True, chi2_out=chi2_e, flux_out=flux_e), w3.B * w3.T, "flux_evals")
    calls["cfg3_fp64"] = (
        lambda: gl.gl_loglike(P3, T3, w3.t_exp, w3.n_ss, O3, S3, dtype="f64", want_flux=True), w3.B * w3.T, "flux_evals")
    # the same series with 16x the walkers (sixteen waves of CTAs): what the kernel sustains once the launch is
    # not one walker's dependent chain any more (context for roofline.frac; not BASELINE.json's configuration)
    Bbig = 16 * w3.B
    serb = gl.GlSeries(w3.times, w3.obs, w3.sigma, w3.t_exp, w3.n_ss, Bbig, device=dev)
    Pb = d(wl.draw_walkers(Bbig, wl.SEED_CFG3_WALKERS + 99))
    chi2_b = torch.empty(Bbig, dtype=torch.float32, device=dev)
    flux_b = torch.empty((Bbig, w3.T), dtype=torch.float32, device=dev)
    calls["cfg3_shape_B4096"] = (
        lambda: serb.loglike_dev(Pb, want_flux=True, chi2_out=chi2_b, flux_out=flux_b), Bbig * w3.T, "flux_evals")
    gp3 = d(np.tile([2e-4, 0.5, 1e-4], (w3.B, 1)))
    calls["cfg3_gp_loglike"] = (
        lambda: gl.gl_gp_loglike(P3, T3, w3.t_exp, w3.n_ss, O3, S3, gp3, dtype="f32"), w3.B * w3.T, "flux_evals")
    w4 = wl.config4()
    ser4 = gl.GlSeries(w4.times, w4.obs, w4.sigma, w4.t_exp, w4.n_ss, w4.B, device=dev)
    P4 = d(w4.params)
    c4 = torch.empty(w4.B, dtype=torch.float32, device=dev)
    f4 = torch.empty((w4.B, w4.T), dtype=torch.float32, device=dev)
    calls["cfg4"] = (lambda: ser4.loglike_dev(P4, want_flux=True, chi2_out=c4, flux_out=f4), w4.B * w4.T, "flux_evals")
    geom, _ = wl.config5()
    G = d(geom)
    calls["cfg5"] = (lambda: gl.gl_flux_geometry(G, dtype="f32"), geom.shape[0], "geometries")
    G1 = d(geom[-200_000:])          # (the last 10^5 of these are the forced rows)
    calls["cfg5_fp64_200k"] = (lambda: gl.gl_flux_geometry(G1, dtype="f64"), 200_000, "geometries")
    G2 = d(geom[:20_000])
    calls["simpson_fp32_20k_x4096"] = (lambda: gl.gl_flux_geometry_simpson(G2, 4096, dtype="f32"), 20_000, "geometries")
    T1 = 100_000
    t1 = d(np.linspace(-0.6, 0.6, T1))
    p1 = d(wl.CFG2_ROW[None, :])
    f1 = torch.empty((1, T1), dtype=torch.float32, device=dev)
    calls["single_lightcurve_T1e5"] = (lambda: gl.gl_lightcurve(p1, t1, 0.0, 1, dtype="f32", out=f1), T1, "flux_evals")
    return calls, {"w4": w4, "ser4": ser4, "serb": serb, "Pb_rows": Bbig}


def extra_workloads(gl, dev, d, timed, fractions, peak_tflops, probe, ncu, w3, ser3, P3):
    """The secondary numbers, timed like the headline (CUDA events, L2 flushed, inputs resident), so that
    the driver's run carries them: each with ms, units/s and both roofline fractions where they apply."""
    calls, keep = secondary_calls(gl, dev, d, w3, ser3, P3)
    ex = {}
    for name, (fn, units, unit) in calls.items():
        slow = name in ("cfg3_fp64", "cfg5_fp64_200k", "simpson_fp32_20k_x4096")
        ms = float(np.mean(timed(fn, k=5 if slow else 20, warm=2 if slow else 3)))
        ex[name] = {"ms": ms, f"{unit}_per_s": units / (ms * 1e-3)}
    ex["cfg3_gl_loglike_stateless"]["launches_per_step"] = 2
    ex["cfg3_fp64"].update({"dtype": "f64", "dfma_chain_tflops": probe["fp64_tflops"]})
    exf = ncu.get("executed_fp64_flop", {}).get("cfg3_fp64")
    if exf:
        ex["cfg3_fp64"]["executed_fp64_flop_ncu"] = exf
        ex["cfg3_fp64"]["frac_executed_of_dfma_chain"] = exf / (ex["cfg3_fp64"]["ms"] * 1e-3) / 1e12 / probe["fp64_tflops"]
    w4 = keep["w4"]
    n_in, n_limb = in_transit_mix(w4)
    ex["cfg4"].update({"B": w4.B, "T": w4.T, "n_ss": w4.n_ss, "in_transit_subsamples": n_in,
                       "of_which_limb_crossing": n_limb, **fractions("cfg4", n_in, n_limb, ex["cfg4"]["ms"])})
    # (the walkers of the large batch are drawn like config 3's: the in-transit mix per walker is the same)
    n_in3, n_limb3 = in_transit_mix(w3)
    scale = keep["Pb_rows"] / w3.B
    ex["cfg3_shape_B4096"].update({"B": keep["Pb_rows"], "note": "in-transit counts scaled from config 3's walkers",
                                   **fractions("cfg3", int(n_in3 * scale), int(n_limb3 * scale),
                                               ex["cfg3_shape_B4096"]["ms"])})
    if "executed_flop_ncu" in ex["cfg3_shape_B4096"]:      # the capture is of the 256-walker launch: scale it
        exf3 = ex["cfg3_shape_B4096"]["executed_flop_ncu"] * scale
        ex["cfg3_shape_B4096"]["executed_flop_ncu"] = exf3
        ex["cfg3_shape_B4096"]["frac_executed"] = exf3 / (ex["cfg3_shape_B4096"]["ms"] * 1e-3) / 1e12 / peak_tflops
    keep["serb"].close()
    ex["cfg5"]["active_lanes_per_instruction_ncu"] = ncu.get("active_lanes", {}).get("cfg5")
    ex["single_lightcurve_T1e5"].update({
        "us_per_flux_sample": ex["single_lightcurve_T1e5"]["ms"] * 1e3 / 100_000,
        "paper": "about 0.5 us per sample at 1e4-1e5 samples on a Quadro RTX 5000 (PAPER.md:171; another "
                 "machine: context)"})
    keep["ser4"].close()
    return ex


def run_profile(args):
    """--profile NAME: the named call five times and nothing else (a short command for ncu)."""
    import torch
    import paper_2410_05408_b200 as gl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    gl.load_library()
    d = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64), device=dev)  # noqa: E731
    w = make_workload("cfg3", 0)
    P = d(w.params)
    ser = gl.GlSeries(w.times, w.obs, w.sigma, w.t_exp, w.n_ss, w.B, device=dev)
    chi2_d = torch.empty(w.B, dtype=torch.float32, device=dev)
    flux_d = torch.empty((w.B, w.T), dtype=torch.float32, device=dev)
    calls, keep = secondary_calls(gl, dev, d, w, ser, P)
    calls["cfg3"] = (lambda: ser.loglike_dev(P, want_flux=True, chi2_out=chi2_d, flux_out=flux_d), w.B * w.T, "flux_evals")
    if args.profile not in calls:
        raise SystemExit(f"--profile: one of {sorted(calls)}")
    for _ in range(5):
        calls[args.profile][0]()
    torch.cuda.synchronize()
    print(json.dumps({"profile": args.profile, "calls": 5}))


if __name__ == "__main__":
    main()
