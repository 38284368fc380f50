"""N > 1 path (replicas only, no data-path collective), covered on CPU with gloo,
world_size 2: the replica shard of every rank, the max-over-ranks timing reduction of bench.py, and
that the shards together reproduce the single-process run of the ORACLE (replica independence:
a batch of R equals R single-replica calls with first_replica = r)."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_1807_10750_b200 import workloads as W
    from oracle import ising_oracle as O
    wl = W.config2(n=300, p=0.03, sweeps=30, replicas=4)
    first, R = bench.replica_shard(rank, world, wl.n_replicas)
    assert (first, R) == (rank * 4, 4)
    o = O.anneal_workload(wl, n_replicas=R, first_replica=first, n_threads=1)
    t = bench.max_over_ranks(1.0 + rank, dist, "cpu")
    assert t == float(world)
    cuts = torch.from_numpy(o["best_cut"].astype(np.int64))
    gathered = [torch.zeros_like(cuts) for _ in range(world)]
    dist.all_gather(gathered, cuts)           # test-side only: the product path has no collective
    if rank == 0:
        out.put(torch.cat(gathered).numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_replicas_and_reduce_time():
    sys.path.insert(0, ROOT)
    from paper_1807_10750_b200 import workloads as W
    from oracle import ising_oracle as O
    O.lib()
    W._load_native()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = out.get(timeout=240)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    wl = W.config2(n=300, p=0.03, sweeps=30, replicas=8)
    whole = O.anneal_workload(wl, n_threads=2)
    np.testing.assert_array_equal(got, whole["best_cut"])
