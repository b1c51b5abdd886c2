"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_1310_6380_b200``).  It holds no arithmetic of the method itself: it only
emits plain NumPy arrays (lattice, polygons, E/nu/rho, k-points in reduced
coordinates).  Turning E/nu into a compliance tensor (eq. 14), shape
integrals, matrices and eigenvalues are implemented independently on each side.

The paper's own workloads are unpublished Gmsh meshes of one steel/epoxy cell
(PAPER.md:108, 177-186, 275-291); they are not available, so these inputs take their
shapes (hexagonal cell, ~10^3 triangular phases, 18 bands, tens of k-points; simple
square cells, few bands) and stand in for them.

Recipe: ``numpy.random.default_rng(seed)`` (PCG64); config c uses
``seed = 13106380 + c``; config 4 cell j uses ``default_rng([13106384, j])``.  Draw
order per cell: E[P], nu[P], rho[P], then geometry jitter, then split choices.
"""
from __future__ import annotations

import dataclasses
from typing import List

import numpy as np

SEED_BASE = 13106380

STIFF = (70.0e9, 0.33, 2700.0)   # E [Pa], nu, rho [kg/m^3]  (configs 2 and 4)
SOFT = (3.5e9, 0.35, 1180.0)

SQUARE = np.array([[1.0, 0.0], [0.0, 1.0]])
HEXAGONAL = np.array([[1.0, 0.0], [0.5, np.sqrt(3.0) / 2.0]])


@dataclasses.dataclass
class Cell:
    """One unit cell: lattice rows h1,h2; CSR polygons (CCW, Cartesian); per-phase E, nu, rho."""
    lattice: np.ndarray       # (2,2) float64, rows = h1, h2   ([A] of PAPER.md:138)
    vert_offset: np.ndarray   # (P+1,) int32
    verts: np.ndarray         # (sum E_p, 2) float64 Cartesian
    E: np.ndarray             # (P,) Pa
    nu: np.ndarray            # (P,)
    rho: np.ndarray           # (P,) kg/m^3

    @property
    def nphase(self) -> int:
        return int(self.vert_offset.shape[0] - 1)

    def polygon(self, p: int) -> np.ndarray:
        return self.verts[self.vert_offset[p]:self.vert_offset[p + 1]]


@dataclasses.dataclass
class Workload:
    name: str
    cells: List[Cell]
    Mt: int                   # plane-wave truncation, indices in [-Mt, Mt]  (paper's M)
    kpts: np.ndarray          # (nk,2) reduced coordinates (Q1,Q2), k = Q1 q1 + Q2 q2
    nbands: int
    description: str

    @property
    def N(self) -> int:
        return (2 * self.Mt + 1) ** 2

    @property
    def nk(self) -> int:
        return int(self.kpts.shape[0])


# ----------------------------------------------------------------------------- geometry helpers
def _signed_area(poly: np.ndarray) -> float:
    x, y = poly[:, 0], poly[:, 1]
    return 0.5 * float(np.sum(x * np.roll(y, -1) - np.roll(x, -1) * y))


def _csr(polys: List[np.ndarray]):
    off = np.zeros(len(polys) + 1, dtype=np.int32)
    off[1:] = np.cumsum([len(p) for p in polys])
    return off, np.ascontiguousarray(np.concatenate(polys, axis=0), dtype=np.float64)


def pixel_polygons(n: int, lattice: np.ndarray = SQUARE) -> List[np.ndarray]:
    """n x n pixel grid; pixel (i,j) = [i/n,(i+1)/n] x [j/n,(j+1)/n] in fractional coords, CCW, p = n*i + j."""
    polys = []
    for i in range(n):
        for j in range(n):
            frac = np.array([[i / n, j / n], [(i + 1) / n, j / n],
                             [(i + 1) / n, (j + 1) / n], [i / n, (j + 1) / n]])
            polys.append(frac @ lattice)
    return polys


def jittered_triangle_mesh(rng: np.random.Generator, lattice: np.ndarray,
                           nx: int = 24, ny: int = 23, nsplit: int = 14) -> List[np.ndarray]:
    """SURVEY.md §8(d) C3/C5 mesh: nx x ny structured grid in fractional coordinates, interior
    vertices jittered by U[-1/4,1/4] of the grid spacing per coordinate (boundary vertices fixed,
    so the tiling of the cell is exact), every quad split along its (i,j)-(i+1,j+1) diagonal, then
    the first ``nsplit`` triangles of ``rng.permutation(ntri)`` are split at the centroid into 3."""
    gx = np.arange(nx + 1) / nx
    gy = np.arange(ny + 1) / ny
    F = np.stack(np.meshgrid(gx, gy, indexing="ij"), axis=-1)          # (nx+1, ny+1, 2) fractional
    jit = rng.uniform(-0.25, 0.25, size=(nx - 1, ny - 1, 2))
    F[1:-1, 1:-1, 0] += jit[:, :, 0] / nx
    F[1:-1, 1:-1, 1] += jit[:, :, 1] / ny
    tris = []
    for i in range(nx):
        for j in range(ny):
            a, b, c, d = F[i, j], F[i + 1, j], F[i + 1, j + 1], F[i, j + 1]
            tris.append(np.array([a, b, c]))
            tris.append(np.array([a, c, d]))
    ntri = len(tris)
    chosen = set(int(t) for t in rng.permutation(ntri)[:nsplit])
    out = []
    for t, tri in enumerate(tris):
        if t in chosen:
            g = tri.mean(axis=0)
            out.extend([np.array([tri[0], tri[1], g]), np.array([tri[1], tri[2], g]),
                        np.array([tri[2], tri[0], g])])
        else:
            out.append(tri)
    polys = [p @ lattice for p in out]
    total = 0.0
    for p in polys:
        a = _signed_area(p)
        assert a > 0.0, "jittered mesh produced a non-positive triangle"
        total += a
    assert abs(total - abs(np.linalg.det(lattice))) < 1e-12
    return polys


def kpath(lattice: np.ndarray, corners_reduced: np.ndarray, nk: int) -> np.ndarray:
    """Closed polyline through ``corners_reduced`` (reduced coords), sampled uniformly in CARTESIAN
    arclength, t_j = j L/(nk-1), j = 0..nk-1, both end points included."""
    Tinv = np.linalg.inv(lattice)
    Qm = 2.0 * np.pi * Tinv.T                      # rows = q1, q2  (q^i . h^j = 2 pi delta_ij)
    cart = corners_reduced @ Qm
    seg = np.linalg.norm(np.diff(cart, axis=0), axis=1)
    cum = np.concatenate([[0.0], np.cumsum(seg)])
    L = cum[-1]
    out = np.zeros((nk, 2))
    for j in range(nk):
        t = L * j / (nk - 1) if nk > 1 else 0.0
        s = min(int(np.searchsorted(cum, t, side="right") - 1), len(seg) - 1)
        f = (t - cum[s]) / seg[s]
        out[j] = corners_reduced[s] + f * (corners_reduced[s + 1] - corners_reduced[s])
    return out


SQUARE_PATH = np.array([[0.0, 0.0], [0.5, 0.0], [0.5, 0.5], [0.0, 0.0]])              # Gamma-X-M-Gamma
HEX_PATH = np.array([[0.0, 0.0], [0.5, 0.0], [2.0 / 3.0, 1.0 / 3.0], [0.0, 0.0]])     # Gamma-M-K-Gamma


# ----------------------------------------------------------------------------- the five configs
def config1() -> Workload:
    rng = np.random.default_rng(SEED_BASE + 1)
    P = 16
    E = rng.uniform(1.0, 70.0, P) * 1e9
    nu = rng.uniform(0.2, 0.4, P)
    rho = rng.uniform(1000.0, 3000.0, P)
    off, verts = _csr(pixel_polygons(4))
    cell = Cell(SQUARE.copy(), off, verts, E, nu, rho)
    return Workload("C1", [cell], 3, kpath(SQUARE, SQUARE_PATH, 30), 6,
                    "square a=1, 4x4 random pixels (P=16), Mt=3 (N=49, K 98x98), 30 k, 6 bands")


def config2() -> Workload:
    n = 20
    E, nu, rho = np.zeros(n * n), np.zeros(n * n), np.zeros(n * n)
    for i in range(n):
        for j in range(n):
            c = np.array([(i + 0.5) / n, (j + 0.5) / n])
            m = STIFF if np.hypot(c[0] - 0.5, c[1] - 0.5) <= 0.35 else SOFT
            E[n * i + j], nu[n * i + j], rho[n * i + j] = m
    off, verts = _csr(pixel_polygons(n))
    cell = Cell(SQUARE.copy(), off, verts, E, nu, rho)
    return Workload("C2", [cell], 7, kpath(SQUARE, SQUARE_PATH, 60), 10,
                    "square a=1, 20x20 pixels, stiff disc r=0.35 in soft matrix (P=400), Mt=7 (N=225), 60 k, 10 bands")


def _hex_cell(seed: int) -> Cell:
    rng = np.random.default_rng(seed)
    P = 1132
    E = rng.uniform(1.0, 200.0, P) * 1e9
    nu = rng.uniform(0.15, 0.45, P)
    rho = rng.uniform(800.0, 8000.0, P)
    polys = jittered_triangle_mesh(rng, HEXAGONAL)
    assert len(polys) == P
    off, verts = _csr(polys)
    return Cell(HEXAGONAL.copy(), off, verts, E, nu, rho)


def config3() -> Workload:
    return Workload("C3", [_hex_cell(SEED_BASE + 3)], 10, kpath(HEXAGONAL, HEX_PATH, 90), 18,
                    "hexagonal a=1, 1132 seeded triangular phases, Mt=10 (N=441, Phi 1323, K 882), 90 k, 18 bands")


def config4(ncells: int = 256) -> Workload:
    cells = []
    polys = pixel_polygons(8)
    off, verts = _csr(polys)
    for j in range(ncells):
        rng = np.random.default_rng([SEED_BASE + 4, j])
        u = rng.uniform(0.0, 1.0, 64)
        stiff = u < 0.5
        E = np.where(stiff, STIFF[0], SOFT[0])
        nu = np.where(stiff, STIFF[1], SOFT[1])
        rho = np.where(stiff, STIFF[2], SOFT[2])
        cells.append(Cell(SQUARE.copy(), off.copy(), verts.copy(), E, nu, rho))
    return Workload("C4", cells, 5, kpath(SQUARE, SQUARE_PATH, 40), 8,
                    f"batch of {ncells} square cells, 8x8 two-material random pixels (P=64), Mt=5 (N=121), 40 k each, 8 bands")


def config5() -> Workload:
    return Workload("C5", [_hex_cell(SEED_BASE + 5)], 15, kpath(HEXAGONAL, HEX_PATH, 120), 18,
                    "hexagonal a=1, 1132 seeded triangular phases, Mt=15 (N=961, Phi 2883, K 1922), 120 k, 18 bands")


CONFIGS = {"C1": config1, "C2": config2, "C3": config3, "C4": config4, "C5": config5}


def get(name: str, **kw) -> Workload:
    return CONFIGS[name](**kw)


def homogeneous_cell(lattice: np.ndarray, E: float, nu: float, rho: float, n: int = 2) -> Cell:
    """A homogeneous cell tiled by n x n parallelogram pixels (test helper: analytic dispersion pin)."""
    off, verts = _csr(pixel_polygons(n, lattice))
    P = n * n
    return Cell(np.array(lattice, dtype=np.float64), off, verts,
                np.full(P, E), np.full(P, nu), np.full(P, rho))


def random_small_cell(seed: int, n: int = 3, lattice: np.ndarray = SQUARE) -> Cell:
    """Small random-property pixel cell for quick parity cases."""
    rng = np.random.default_rng(seed)
    P = n * n
    E = rng.uniform(1.0, 70.0, P) * 1e9
    nu = rng.uniform(0.2, 0.4, P)
    rho = rng.uniform(1000.0, 3000.0, P)
    off, verts = _csr(pixel_polygons(n, lattice))
    return Cell(np.array(lattice, dtype=np.float64), off, verts, E, nu, rho)
