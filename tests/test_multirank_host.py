"""N > 1 host logic of bench.py on CPU: world_size-2 gloo run.

Walkers shard over ranks with no data-path collective: every rank draws its own walkers on the
same series, the only exchanges are the barrier and the MAX over ranks of the timings.  The ranks'
chi^2 (here from the oracle: no GPU in this test) must equal the rows a single process computes
for the same draws, and the job-level value must be (units of all ranks) / (slowest rank's time)."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    import bench
    import oracle as orc
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = bench.make_workload("cfg3", rank)
    w.params = w.params[:4]
    sel = slice(1930, 1975)
    chi2, _ = orc.loglike(w.params, w.times[sel], w.t_exp, w.n_ss, w.obs[sel], w.sigma[sel])
    # the max-over-ranks timing rule of bench.py, with fake per-rank times
    t = torch.tensor([1.0 + rank], dtype=torch.float64)
    dist.barrier()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    np.save(Path(out_dir) / f"r{rank}.npy", np.concatenate([chi2, [t.item()]]))
    dist.destroy_process_group()


def test_two_ranks_shard_walkers(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    sys.path.insert(0, str(ROOT))
    import bench
    import oracle as orc
    from paper_2410_05408_b200 import workloads as wl
    got = [np.load(tmp_path / f"r{r}.npy") for r in range(world)]
    base = wl.config3()
    sel = slice(1930, 1975)
    for r in range(world):
        p = base.params if r == 0 else wl.draw_walkers(base.B, wl.SEED_CFG3_WALKERS + 1000 * r)
        ref, _ = orc.loglike(p[:4], base.times[sel], base.t_exp, base.n_ss, base.obs[sel],
                             base.sigma[sel])
        assert np.array_equal(got[r][:-1], ref)
        assert got[r][-1] == float(world)          # every rank sees the slowest rank's time
    # ranks get DIFFERENT walkers (weak scaling: per-rank work fixed, total grows)
    assert not np.array_equal(got[0][:-1], got[1][:-1])
    assert np.array_equal(bench.make_workload("cfg3", 0).params, base.params)


def test_bench_gpus_flag_starts_the_ranks():
    """`python bench.py --gpus 2 --dry` outside torchrun: bench.py must START two ranks (gloo on this
    CPU box), shard the walkers and print one JSON line with n_gpus = 2 and the slowest rank's time."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--gpus", "2", "--dry", "--steps", "2"],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout
    rec = json.loads(lines[0])
    assert rec["n_gpus"] == 2 and rec["dry"] is True
    assert rec["ms_per_step"] == 2.0            # max over ranks of (1 + rank)
    assert rec["distinct_shards"] == 2          # the two ranks drew different walkers
    # one process, no flag: one rank
    out1 = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--dry"], capture_output=True, text=True,
                          timeout=300, env=env)
    rec1 = json.loads([ln for ln in out1.stdout.splitlines() if ln.startswith("{")][0])
    assert rec1["n_gpus"] == 1
