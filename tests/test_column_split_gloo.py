"""N>1 path on CPU (gloo, world_size 2): the column split needs no exchange.  Each rank applies the ORACLE operator
and filter to its own column slice; the gathered slices equal the single-process result bit for bit, and the timing
reduction is the max over ranks.  (The CUDA path shards the same way: bench.py --gpus N gives every rank its own
B-column block, 'scaling': 'weak'.)"""
import os
import socket

import numpy as np
import pytest

import workloads
from paper_2510_10529_b200.colsplit import column_slice, job_throughput, max_over_ranks

torch = pytest.importorskip("torch")


def test_column_slice_partitions():
    for B in (0, 1, 7, 64, 129):
        for world in (1, 2, 3, 8):
            s = [column_slice(B, r, world) for r in range(world)]
            assert s[0][0] == 0 and s[-1][1] == B
            assert all(s[i][1] == s[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in s]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        column_slice(8, 2, 2)
    assert job_throughput(10.0, 4, 2.0) == 20.0


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist

    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = workloads.config(1)
    om = oracle.OracleMesh(w.xe, w.ye, w.ze, w.p)
    om.set_potential(w.V(om.quad_coords()))
    om.assemble()
    X = w.X(om.mask())
    eps = workloads.shifts(2001, w.B)
    lo, hi = column_slice(w.B, rank, world)
    Xr = np.ascontiguousarray(X[:, lo:hi])
    Y = om.apply(Xr, eps[lo:hi])
    F = om.filter(Xr, 6, 3.0, 25.0, 1.0)
    np.save(os.path.join(out_dir, "Y%d.npy" % rank), Y)
    np.save(os.path.join(out_dir, "F%d.npy" % rank), F)
    t = max_over_ranks([1.0 + rank, 5.0 - rank], dist)
    dist.barrier()
    assert t == [float(world), 5.0]
    dist.destroy_process_group()


def test_column_split_world2(tmp_path):
    import torch.multiprocessing as mp

    import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = workloads.config(1)
    om = oracle.OracleMesh(w.xe, w.ye, w.ze, w.p)
    om.set_potential(w.V(om.quad_coords()))
    om.assemble()
    X = w.X(om.mask())
    eps = workloads.shifts(2001, w.B)
    Y = np.concatenate([np.load(tmp_path / ("Y%d.npy" % r)) for r in range(world)], axis=1)
    F = np.concatenate([np.load(tmp_path / ("F%d.npy" % r)) for r in range(world)], axis=1)
    assert np.array_equal(Y, om.apply(X, eps))
    assert np.array_equal(F, om.filter(X, 6, 3.0, 25.0, 1.0))
