"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol include/bs.h declares, the header
and the binding agree, pure-host entry points work, and compute calls fail loudly (no CPU fallback) without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1310_6380_b200 import build
    return build.build()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "bs.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bs_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    names = header_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/bs.h but not exported by libbs.so"


def test_binding_lists_the_header_symbols(libpath):
    from paper_1310_6380_b200 import binding
    assert sorted(binding.SYMBOLS) == header_symbols()
    for n in binding.SYMBOLS:
        assert hasattr(binding, n), f"binding lacks a wrapper named {n}"


def test_host_only_entry_point_matches_oracle(libpath):
    from paper_1310_6380_b200 import binding
    E = np.array([1e9, 70e9, 3.5e9, 200e9])
    nu = np.array([0.15, 0.33, 0.35, 0.45])
    got = binding.bs_isotropic_plane_strain(E, nu)
    assert np.allclose(got, oracle.isotropic_plane_strain_compliance(E, nu), rtol=1e-15, atol=0)
    with pytest.raises(binding.BsError) as ei:
        binding.bs_isotropic_plane_strain([1.0], [0.5])
    assert ei.value.status == binding.BS_ERR_ARG


def test_no_cpu_fallback(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1310_6380_b200 import binding
    c = wl.random_small_cell(1, 2)
    comp = binding.bs_isotropic_plane_strain(c.E, c.nu)
    with pytest.raises(binding.BsError) as ei:
        binding.bs_create_cell(c.lattice, c.vert_offset, c.verts, comp, c.rho)
    assert ei.value.status == binding.BS_ERR_CUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1310_6380_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_1310_6380_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_1310_6380_b200/``", "")


def test_workloads_shapes():
    # the five configs have the sizes BASELINE.json names
    expect = {"C1": (16, 3, 30, 6), "C2": (400, 7, 60, 10), "C3": (1132, 10, 90, 18), "C5": (1132, 15, 120, 18)}
    for name, (P, Mt, nk, b) in expect.items():
        w = wl.get(name)
        assert (w.cells[0].nphase, w.Mt, w.nk, w.nbands) == (P, Mt, nk, b)
        assert np.allclose(w.kpts[0], 0) and np.allclose(w.kpts[-1], 0)
    w = wl.get("C4", ncells=3)
    assert (len(w.cells), w.cells[0].nphase, w.Mt, w.nk, w.nbands) == (3, 64, 5, 40, 8)
    a = wl.get("C4", ncells=2).cells[1]
    assert np.array_equal(a.E, w.cells[1].E)       # seeded per cell, independent of the batch size
