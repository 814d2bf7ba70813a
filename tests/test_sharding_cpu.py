"""world_size-2 gloo test of the multi-GPU host logic on CPU: sharded walkers reproduce the
unsharded trajectories (Philox is keyed by the global walker index), timings reduce by max,
the energy estimate reduces by (sum, sum^2, count)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2506_09743_b200 import workloads as wl
from paper_2506_09743_b200.sharding import global_energy, max_over_ranks, shard_range


def test_shard_range_partitions():
    for n, w in [(10, 3), (131072, 8), (5, 8), (7, 1)]:
        rs = [shard_range(n, r, w) for r in range(w)]
        assert rs[0][0] == 0 and rs[-1][1] == n
        assert all(rs[i][1] == rs[i + 1][0] for i in range(w - 1))
        sizes = [b - a for a, b in rs]
        assert max(sizes) - min(sizes) <= 1


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import binding as ob
    d, r = wl.lih(M=96)
    o = ob.OracleSystem(d)
    w0, w1 = shard_range(96, rank, world)
    # a rank holds only its walkers and passes its global offset, as bench.py does with walker_offset
    full = ob.metropolis(o, r, 0.3, 4, seed=123)                      # reference: unsharded
    L = ob.lib()
    rr = np.array(r, order="C", copy=True)
    lp = np.zeros(96); sg = np.zeros(96)
    acc = np.zeros((4, 96), np.uint8)
    assert L.oracle_metropolis(o.ref, rr.ctypes.data, 96, w0, w1, 0.3, 4, 123, 0, lp.ctypes.data, sg.ctypes.data,
                               acc.ctypes.data, None, None) == 0
    assert np.array_equal(rr[:, :, w0:w1], full["r"][:, :, w0:w1])
    assert np.array_equal(acc[:, w0:w1], full["accept"][:, w0:w1])
    el = ob.local_energy(o, np.ascontiguousarray(rr[:, :, w0:w1]))[2]
    mean, err = global_energy(float(el.sum()), float((el * el).sum()), len(el))
    el_full = ob.local_energy(o, full["r"])[2]
    assert abs(mean - el_full.mean()) < 1e-12 * abs(el_full.mean())
    assert abs(err - el_full.std(ddof=1) / np.sqrt(96)) < 1e-9 * abs(err)
    t = max_over_ranks([1.0 + rank, 5.0 - rank])
    assert t == [float(world), 5.0]
    np.save(os.path.join(out_dir, f"ok{rank}.npy"), np.array([1]))
    dist.destroy_process_group()


def test_two_rank_sharding_gloo(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert all(os.path.exists(tmp_path / f"ok{r}.npy") for r in range(2))
