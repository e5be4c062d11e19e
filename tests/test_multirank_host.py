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
