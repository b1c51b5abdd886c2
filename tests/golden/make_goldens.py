#!/usr/bin/env python
"""Writes the stored oracle results the full-size GPU parity tests compare against.

    python tests/golden/make_goldens.py [C2 C3 C4 C5]

Imports ONLY ``oracle`` and ``workloads`` (never the CUDA package): every stored value is the CPU oracle's
(``oracle.band_structure`` = assemble + LAPACK zhegv at every k-point).  Output, per config:
``tests/golden/<name>_lambda.npz`` with ``lam`` (lowest nbands eigenvalues lambda = omega^2 at EVERY k-point of the
workload), ``lam_max`` (largest eigenvalue per k-point, needed by the backward-error clause of reading R8) and, for C4,
``cells`` (the 16 cell indices, spread over the 256-cell batch, whose 40 k-points each are stored).
C5 is about five minutes of zhegv on eight cores; the others take seconds to a minute.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import workloads as wl  # noqa: E402

C4_CELLS = [0, 17, 34, 51, 68, 85, 102, 119, 131, 136, 153, 170, 187, 204, 221, 255]


def one_cell(cell, Mt, kpts, nbands):
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
    return oracle.band_structure(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, Mt, kpts, nbands)


def main(names):
    for name in names:
        t0 = time.time()
        w = wl.get(name)
        if name == "C4":
            lam = np.zeros((len(C4_CELLS), w.nk, w.nbands))
            lmax = np.zeros((len(C4_CELLS), w.nk))
            for j, ci in enumerate(C4_CELLS):
                lam[j], lmax[j] = one_cell(w.cells[ci], w.Mt, w.kpts, w.nbands)
            np.savez(os.path.join(HERE, f"{name}_lambda.npz"), lam=lam, lam_max=lmax, cells=np.array(C4_CELLS),
                     kpts=w.kpts)
        else:
            lam, lmax = one_cell(w.cells[0], w.Mt, w.kpts, w.nbands)
            np.savez(os.path.join(HERE, f"{name}_lambda.npz"), lam=lam, lam_max=lmax, kpts=w.kpts)
        print(f"{name}: {lam.shape} in {time.time() - t0:.1f} s", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:] or ["C2", "C3", "C4", "C5"])
