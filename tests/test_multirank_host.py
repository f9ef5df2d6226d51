"""N > 1 host logic of bench.py (replicas only) on CPU: two gloo processes.
Distinct replica seeds per rank, max-over-ranks timing, whole-job value; the reference arm runs on
rank 0 only."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2604_06309_b200 import inputs
    seed = bench.replica_seed(rank)
    theta = np.linspace(0.0, 1.0, 16)
    t, mu, hist = inputs.synthetic_history(theta, 1.0 - theta, 8, -2.0, 2.0, seed=seed)
    ms_local = 10.0 + 5.0 * rank                 # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world)
    seeds = [None] * world
    dist.all_gather_object(seeds, seed)
    sums = [None] * world
    dist.all_gather_object(sums, float(hist.sum()))
    out[rank] = dict(ms=ms, seeds=seeds, sums=sums, value=bench.job_value(1000, 3, world, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    world = 2
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        assert res[r]["ms"] == 15.0                       # max over ranks, same on every rank
        assert res[r]["seeds"][0] != res[r]["seeds"][1]   # distinct replicas
        assert res[r]["sums"][0] != res[r]["sums"][1]
        assert abs(res[r]["value"] - 1000 * 3 * 2 / 15e-3) < 1e-6


def test_reference_arm_runs_on_rank0_only(monkeypatch):
    import bench
    monkeypatch.setenv("RANK", "1")
    args = type("A", (), dict(workload="config2", L=64, stencil=4, ref_targets=4, warmup=0, steps=1, gpus=2))()
    assert bench.run_reference(args) == 0                 # returns before touching the oracle
