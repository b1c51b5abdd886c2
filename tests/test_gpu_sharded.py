"""The sharded driver (paper_1310_6380_b200/sharded.py) on the GPU: two ranks (two processes sharing cuda:0, gloo for the
result gather, no kernel of one rank waits for the other) must reproduce the single-rank eigenvalues BIT FOR BIT, for the
k-point split (config 1) and for the cell split (a small config-4 batch).  SURVEY 8(e)."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu

WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, os.environ["BS_ROOT"])
import paper_1310_6380_b200 as bs
from paper_1310_6380_b200 import sharded
import workloads as wl
torch.cuda.set_device(0)
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
out = {}
for name, w in (("C1", wl.get("C1")), ("C4", wl.get("C4", ncells=5))):
    inputs = [(c.lattice, c.vert_offset, c.verts, bs.bs_isotropic_plane_strain(c.E, c.nu), c.rho) for c in w.cells]
    lam = sharded.bands_sharded(inputs, w.Mt, w.kpts, w.nbands)
    assert lam.shape == (len(w.cells), w.nk, w.nbands)
    out[name] = lam.cpu().numpy()
    for forced in ("kpoints", "cells"):
        again = sharded.bands_sharded(inputs, w.Mt, w.kpts, w.nbands, axis=forced).cpu().numpy()
        assert np.array_equal(again, out[name]), (name, forced)      # both splits give the same bits
if rank == 0:
    np.savez(os.environ["BS_OUT"], **out)
dist.barrier()
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_ranks_reproduce_the_single_rank_result_bitwise(tmp_path):
    import paper_1310_6380_b200 as bs
    from paper_1310_6380_b200 import sharded
    import workloads as wl
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    outp = str(tmp_path / "sharded.npz")
    env = dict(os.environ, BS_ROOT=ROOT, BS_OUT=outp, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    got = np.load(outp)
    for name, w in (("C1", wl.get("C1")), ("C4", wl.get("C4", ncells=5))):
        inputs = [(c.lattice, c.vert_offset, c.verts, bs.bs_isotropic_plane_strain(c.E, c.nu), c.rho) for c in w.cells]
        one = sharded.bands_sharded(inputs, w.Mt, w.kpts, w.nbands).cpu().numpy()      # no process group: one rank
        assert np.array_equal(got[name], one), name
