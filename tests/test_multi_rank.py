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


# ---- channel-sharded evaluation: replicated positions, channels a mod G, one exchange ----

def _sharded_system():
    import numpy as np
    rng = np.random.default_rng(44)
    box, grid, w, c = [9.0, 10.0, 8.5], [16, 18, 16], 6, 12.024
    N = 40
    pos = rng.uniform(0, 1, (N, 3)) * box
    q = rng.normal(0, 0.6, (5, N))
    ex = [1, 1, 3, 6, 6]          # five channels on two ranks: ranks own 3 and 2 of them
    return pos, q, ex, box, grid, w, c


def _sharded_worker(rank, world, port, out):
    import numpy as np
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import gridded as G
    from paper_2606_06617_b200 import sharding
    pos, q, ex, box, grid, w, c = _sharded_system()
    r_c, c_w = G.default_r_c(box, grid, c), G.default_c_w(w)
    own = sharding.channel_partition(len(ex), world, rank)
    # this rank's evaluation: oracle B on its channels only (on a GPU box: the C library, same contract)
    E_l, Ech_l, phi_l, F_l = G.gridded(pos, q[own], [ex[a] for a in own], box, grid, w, c, r_c, c_w)
    E = torch.tensor([E_l], dtype=torch.float64)
    F = torch.tensor(F_l, dtype=torch.float64)
    sharding.reduce_results(E, F)
    phi = sharding.gather_potentials(torch.tensor(phi_l, dtype=torch.float64), len(ex), world, rank)
    out[rank] = (own, float(E.item()), F.numpy().copy(), phi.numpy().copy())
    dist.barrier()
    dist.destroy_process_group()


def test_channel_sharded_evaluation_world_size_2_gloo():
    """Two ranks evaluate disjoint channel subsets with oracle B; after the exchange step (all-reduce of
    F and E, all-gather of phi) every rank holds the single-rank result of all five channels."""
    import numpy as np
    from oracle import gridded as G
    world = 2
    port = _free_port()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_sharded_worker, args=(world, port, out), nprocs=world, join=True)
    pos, q, ex, box, grid, w, c = _sharded_system()
    E, Ech, phi, F = G.gridded(pos, q, ex, box, grid, w, c, G.default_r_c(box, grid, c), G.default_c_w(w))
    assert sorted(out[0][0] + out[1][0]) == list(range(5)) and out[0][0] == [0, 2, 4] and out[1][0] == [1, 3]
    for r in range(world):
        own, E_r, F_r, phi_r = out[r]
        assert abs(E_r - E) < 1e-12 * abs(E)
        assert np.allclose(F_r, F, rtol=0, atol=1e-12 * np.abs(F).max())
        assert np.allclose(phi_r, phi, rtol=0, atol=1e-12 * np.abs(phi).max())


def test_channel_partition_properties():
    from paper_2606_06617_b200 import sharding
    for C in (1, 4, 5, 8, 11):
        for world in (1, 2, 3, 8):
            parts = [sharding.channel_partition(C, world, r) for r in range(world)]
            assert sorted(sum(parts, [])) == list(range(C))                    # a partition
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1   # balanced
    # single process: the exchange step is the identity
    E, F = torch.ones(1, dtype=torch.float64), torch.ones((3, 3))
    assert sharding.reduce_results(E, F)[0].item() == 1.0
    phi = sharding.gather_potentials(torch.arange(6.0).reshape(2, 3), 2, 1, 0)
    assert phi.tolist() == [[0.0, 1.0, 2.0], [3.0, 4.0, 5.0]]
