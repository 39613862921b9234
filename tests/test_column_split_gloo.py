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


def _bench_stub(*flags):
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--stub", "--workload", "2", "--steps", "2",
                          *flags], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout  # rank 0 alone prints
    return json.loads(lines[0])


def test_bench_rank_logic_world2_gloo():
    """bench.py's own N > 1 path on CPU: `python bench.py --gpus 2` with no torchrun environment must start two ranks
    itself; the step time of the line is the MAX over ranks, the value the units of ALL ranks over that time (weak
    scaling: every rank its own B columns; strong: the B columns dealt out).  --stub replaces the GPU step by a fixed fake
    time per rank (10 ms x (rank + 1)); everything else is the code path the driver runs."""
    w = workloads.config(2)
    one = _bench_stub("--gpus", "1")
    assert one["n_gpus"] == 1 and one["data"] == "stub" and one["ms_per_step"] == 10.0
    assert one["value"] == pytest.approx(w.N_free * w.B * w.m / 0.010 / 1e9)
    two = _bench_stub("--gpus", "2")
    assert two["n_gpus"] == 2 and two["scaling"] == "weak" and two["ms_per_step"] == 20.0  # the slower rank
    assert two["config"]["columns_per_gpu"] == w.B and two["config"]["columns_total"] == 2 * w.B
    assert two["value"] == pytest.approx(2 * w.N_free * w.B * w.m / 0.020 / 1e9)
    assert two["e2e"]["value"] == pytest.approx(2 * w.N_free * w.B * w.m / 0.040 / 1e9)
    strong = _bench_stub("--gpus", "2", "--scaling", "strong")
    assert strong["config"]["columns_per_gpu"] == w.B // 2 and strong["config"]["columns_total"] == w.B
    assert strong["value"] == pytest.approx(w.N_free * w.B * w.m / 0.020 / 1e9)
