"""N > 1 host logic on CPU (gloo, world_size 2): k-point sharding of bench.py and the max-over-ranks timing reduction.
The data path itself has no collective."""
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, os.environ["BS_ROOT"])
import bench, workloads as wl
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
w = wl.get("C1")
mine = bench.dense_kpath(w, world, rank)
assert mine.shape == (w.nk, 2)
parts = [torch.zeros(w.nk, 2, dtype=torch.float64) for _ in range(world)]
dist.all_gather(parts, torch.from_numpy(mine))
dense = wl.kpath(w.cells[0].lattice, wl.SQUARE_PATH, w.nk * world)
merged = np.zeros_like(dense)
for r in range(world):
    merged[r::world] = parts[r].numpy()
assert np.array_equal(merged, dense), "shards do not tile the dense k-path"
t = torch.tensor([10.0 + rank, 5.0 - rank], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert t.tolist() == [10.0 + world - 1, 5.0]
dist.barrier()
if rank == 0:
    print("OK", world)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_kpoint_sharding_and_timing_reduction_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, BS_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "OK 2" in r.stdout


def test_reference_arm_other_ranks_exit_silently():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=120, env=env)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_single_rank_share_is_the_workload_path():
    sys.path.insert(0, ROOT)
    import bench
    import workloads as wl
    w = wl.get("C3")
    assert np.array_equal(bench.dense_kpath(w, 1, 0), w.kpts)
    a, b = bench.dense_kpath(w, 2, 0), bench.dense_kpath(w, 2, 1)
    assert a.shape == b.shape == w.kpts.shape and np.allclose(a[0], 0) and np.allclose(b[-1], 0)


GATHER_WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, os.environ["BS_ROOT"])
from paper_1310_6380_b200 import sharded
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# the full result a single rank would produce: value encodes (cell, k, band)
for ncells, nk, nb in [(1, 30, 6), (5, 7, 3), (1, 2, 4), (7, 1, 2)]:
    full = (np.arange(ncells)[:, None, None] * 1e6 + np.arange(nk)[None, :, None] * 1e3 + np.arange(nb)[None, None, :]).astype(np.float64)
    for axis_name in ("kpoints", "cells"):
        n = nk if axis_name == "kpoints" else ncells
        ax = 1 if axis_name == "kpoints" else 0
        lo, hi = sharded.shard_range(n, world, rank)
        counts = sharded.shard_counts(n, world)
        assert sum(counts) == n and counts[rank] == hi - lo
        local = torch.from_numpy(np.ascontiguousarray(full[:, lo:hi] if ax == 1 else full[lo:hi]))
        got = sharded.gather_shards(local, counts, ax).numpy()
        assert np.array_equal(got, full), (ncells, nk, nb, axis_name)    # the gathered index map is the 1-rank order
assert sharded.choose_axis(256, 40, world) == "cells" and sharded.choose_axis(1, 120, world) == "kpoints"
dist.barrier()
if rank == 0:
    print("GATHER OK", world)
dist.destroy_process_group()
"""


def _run_workers(tmp_path, text, nproc, marker):
    script = tmp_path / "worker.py"
    script.write_text(text)
    env = dict(os.environ, BS_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc), "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert marker in r.stdout


def test_result_gather_reproduces_single_rank_order_world2(tmp_path):
    _run_workers(tmp_path, GATHER_WORKER, 2, "GATHER OK 2")


def test_result_gather_ragged_world3(tmp_path):
    _run_workers(tmp_path, GATHER_WORKER, 3, "GATHER OK 3")


def test_shard_ranges_tile_the_units():
    sys.path.insert(0, ROOT)
    from paper_1310_6380_b200 import sharded
    for n in (0, 1, 5, 120, 256, 10240):
        for world in (1, 2, 3, 8, 16):
            ranges = [sharded.shard_range(n, world, r) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
            sizes = [b - a for a, b in ranges]
            assert max(sizes) - min(sizes) <= 1
