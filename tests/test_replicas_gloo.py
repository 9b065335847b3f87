"""The N > 1 path of bench.py on CPU: world_size-2 gloo.  The path does not shard (replicas
only), so the only multi-rank logic is: each rank draws its own batch, the job's time is the max over
ranks and its work the sum.  No data-path collective exists to test."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from workloads import CONFIGS, DEFAULT_SEED, make_workload
    w = make_workload(CONFIGS["tiny_local"], seed=bench.rank_seed(DEFAULT_SEED, rank), with_codes=False)
    ms = 10.0 + 5.0 * rank                                    # rank 1 is the slow one
    units, inputs = 1000.0 * (rank + 1), float(w.cand_ids.numel())
    t, u, c = bench.aggregate_over_ranks(ms, units, inputs)
    dist.barrier()
    torch.save({"t": t, "u": u, "c": c, "inputs": inputs, "head": w.cand_ids[:64].clone(),
                "queries": w.queries[:2].clone()}, os.path.join(out, f"r{rank}.pt"))
    dist.destroy_process_group()


def test_two_replicas_aggregate_max_time_and_summed_work(tmp_path):
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = (torch.load(os.path.join(tmp_path, f"r{r}.pt")) for r in (0, 1))
    for r in (r0, r1):                                        # every rank sees the same aggregate
        assert r["t"] == 15.0                                 # max over ranks, not mean or sum
        assert r["u"] == 3000.0                               # work is summed
        assert r["c"] == r0["inputs"] + r1["inputs"]
    # replicas score different batches (different seeds), not copies of one batch
    assert not torch.equal(r0["queries"], r1["queries"])
    assert not torch.equal(r0["head"], r1["head"])


def test_single_process_passes_through():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.5, 7, 9) == (3.5, 7.0, 9.0)
    assert bench.rank_seed(100, 3) == 103 and np.isfinite(bench.L2_BYTES)
