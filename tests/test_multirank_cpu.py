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
