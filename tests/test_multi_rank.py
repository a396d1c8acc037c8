"""Host logic of the N > 1 path (bench.py): every rank evaluates its own replica, no data-path
collective; the reported time is the max over ranks and the units are summed.  Covered here with
world_size-2 gloo processes on the CPU (the kernels themselves are rank-local and unchanged)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r "took" (r + 1) seconds for 1000 * (r + 1) atoms
    t, u = bench.reduce_times(float(rank + 1), 1000 * (rank + 1))
    seeds = [bench.rank_seed(4, r) for r in range(world)]
    out[rank] = (t, u, seeds)
    dist.barrier()
    dist.destroy_process_group()


def test_reduce_times_world_size_2_gloo():
    world = 2
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    for r in range(world):
        t, u, seeds = out[r]
        assert t == 2.0            # max over ranks
        assert u == 3000.0         # sum over ranks
        assert seeds[0] == 4 and len(set(seeds)) == world   # rank 0 keeps the config's seed; replicas differ


def test_reduce_times_single_process_is_identity():
    import bench
    assert bench.reduce_times(1.5, 10) == (1.5, 10)


def test_reference_arm_nonzero_ranks_do_no_work(monkeypatch):
    import bench
    monkeypatch.setenv("RANK", "1")
    monkeypatch.setenv("WORLD_SIZE", "2")

    class A:
        pass
    assert bench.run_reference(A()) == 0
