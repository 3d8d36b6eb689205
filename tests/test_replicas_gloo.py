"""N > 1 is "replicas only": no data-path collective, only the max-over-ranks timing and
per-rank token streams.  This runs that host-side logic of bench.py with world_size 2 on the gloo backend (CPU)."""
import os
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]
sys.path.insert(0, str(ROOT))


def _worker(rank: int, world: int, port: int, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import dfssm_synth as ds
    s = ds.shape_for_config(0)
    toks = ds.token_batch(s.vocab, 4, seed=bench.replica_seed(rank, 0), batch=1)
    # rank r "measures" (r + 1) ms on the device leg and (2 - r) s end to end
    ms, e2e = bench.max_over_ranks([float(rank + 1), float(2 - rank)], dist, "cpu")
    dist.barrier()
    q.put((rank, toks.tolist(), ms, e2e))
    dist.destroy_process_group()


def test_two_replicas_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, t0, ms0, e0), (_, t1, ms1, e1) = res
    assert t0 != t1, "replicas must decode different token streams"
    assert ms0 == ms1 == 2.0 and e0 == e1 == 2.0, "every rank reports the max over ranks"
    import bench
    assert bench.whole_job_rate(world, 1, 10, 2.0e-3) == 2 * 10 / 2.0e-3
    assert bench.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]          # single process: identity


def test_reference_arm_other_ranks_do_no_work(monkeypatch, capsys):
    """--impl reference under torchrun: only rank 0 runs; the others exit without output."""
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setattr(sys, "argv", ["bench.py", "--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "1"])
    bench.main()
    assert capsys.readouterr().out == ""
