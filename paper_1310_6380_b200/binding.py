"""ctypes binding of ``libbs.so`` (C-ABI in ``include/bs.h``): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C calls.  PyTorch supplies device memory (the workspace
tensor lent to the handle) and the stream.  There is no CPU fallback: importing this module compiles ``libbs.so``
with nvcc when it is missing and raises if that fails, and every compute call fails with ``BsError`` when there is no
CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libbs.so")

BS_OK, BS_ERR_ARG, BS_ERR_GEOMETRY, BS_ERR_NOT_PD, BS_ERR_STATE, BS_ERR_CUDA, BS_ERR_NOMEM = 0, -1, -2, -3, -4, -5, -6
BS_OPT_PENCIL_MODE, BS_OPT_PANEL, BS_OPT_TIMING, BS_OPT_TRIDIAG = 0, 1, 2, 3
BS_TRIDIAG_TWO_STAGE, BS_TRIDIAG_ONE_STAGE, BS_TRIDIAG_TWO_STAGE_STREAMED = 0, 1, 2
BS_OPT_ASSEMBLY = 4
BS_OPT_PHI_INVERSE = 5
BS_OPT_OUTPUT = 6
BS_OPT_MODES = 7
BS_OPT_REFINE = 8
BS_OUTPUT_OMEGA2, BS_OUTPUT_OMEGA = 0, 1
BS_ASSEMBLY_EXACT, BS_ASSEMBLY_CENTROID = 0, 1
BS_PENCIL_POLY, BS_PENCIL_DIRECT = 0, 1
BS_T_TABLE, BS_T_EXPAND, BS_T_FACTOR, BS_T_COEF, BS_T_PENCIL, BS_T_TRIDIAG, BS_T_BISECT, BS_T_COUNT = 0, 1, 2, 3, 4, 5, 6, 8
BS_GEMM_LOWER_ONLY, BS_GEMM_KLO_ROW, BS_GEMM_KHI_ROW, BS_GEMM_KLO_COL, BS_GEMM_KHI_COL, BS_GEMM_A_HERM_LOWER = 1, 2, 4, 8, 16, 32

# every symbol include/bs.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "bs_isotropic_plane_strain", "bs_create_cell", "bs_create_cells_shared", "bs_set_properties", "bs_destroy_cell", "bs_set_option", "bs_workspace_bytes",
    "bs_set_workspace", "bs_assemble", "bs_assemble_batch", "bs_get_matrices", "bs_get_table", "bs_get_pencil",
    "bs_bands", "bs_bands_batch", "bs_modes", "bs_modes_batch", "bs_get_tridiagonal", "bs_get_timings", "bs_get_kernel_timings", "bs_launch_count",
    "bs_last_error",
    "bs_fp64_peak", "bs_zgemm", "bs_zpotrf_trtri", "bs_zhetrd_scratch_elems", "bs_zhetrd", "bs_sturm",
    "bs_zhetrd_static_bytes", "bs_zhetrd_static",
]


class BsError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"bs status {status}: {message}")
        self.status = status


if not os.path.exists(LIB_PATH):
    # not built yet (fresh checkout: the .so is git-ignored): compile it now with nvcc; there is no CPU fallback, so a
    # failed build is fatal
    try:
        from . import build as _build
        _build.build()
    except Exception as exc:  # pragma: no cover
        raise ImportError(f"{LIB_PATH} is missing and could not be built ({exc}); run "
                          "`python -m paper_1310_6380_b200.build` (there is no CPU fallback)") from exc
lib = C.CDLL(LIB_PATH)

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_vp = C.c_void_p
lib.bs_last_error.restype = C.c_char_p
lib.bs_launch_count.restype = C.c_int64
lib.bs_launch_count.argtypes = [_vp]
lib.bs_zhetrd_scratch_elems.restype = C.c_size_t
lib.bs_zhetrd_scratch_elems.argtypes = [C.c_int32, C.c_int32]
lib.bs_destroy_cell.restype = None
lib.bs_destroy_cell.argtypes = [_vp]
lib.bs_isotropic_plane_strain.argtypes = [C.c_int32, _dp, _dp, _dp]
lib.bs_create_cell.argtypes = [_dp, C.c_int32, _ip, _dp, _dp, _dp, C.POINTER(_vp)]
lib.bs_create_cells_shared.argtypes = [_dp, C.c_int32, _ip, _dp, C.c_int32, _dp, _dp, C.POINTER(_vp)]
lib.bs_set_properties.argtypes = [_vp, _dp, _dp]
lib.bs_set_option.argtypes = [_vp, C.c_int32, C.c_int32]
lib.bs_workspace_bytes.argtypes = [_vp, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]
lib.bs_set_workspace.argtypes = [_vp, _vp, C.c_size_t]
lib.bs_assemble.argtypes = [_vp, C.c_int32, _vp]
lib.bs_assemble_batch.argtypes = [C.POINTER(_vp), C.c_int32, C.c_int32, _vp]
lib.bs_get_matrices.argtypes = [_vp, _vp, _vp]
lib.bs_get_table.argtypes = [_vp, _vp]
lib.bs_get_pencil.argtypes = [_vp, _dp, _vp, _vp]
lib.bs_bands.argtypes = [_vp, C.c_int32, _dp, C.c_int32, _vp, _vp]
lib.bs_bands_batch.argtypes = [C.POINTER(_vp), C.c_int32, C.c_int32, _dp, C.c_int32, _vp, _vp]
lib.bs_modes.argtypes = [_vp, C.c_int32, _dp, C.c_int32, _vp, _vp, _vp, _vp]
lib.bs_modes_batch.argtypes = [C.POINTER(_vp), C.c_int32, C.c_int32, _dp, C.c_int32, _vp, _vp, _vp, _vp]
lib.bs_get_tridiagonal.argtypes = [_vp, _dp, _dp]
lib.bs_get_timings.argtypes = [_vp, _dp]
lib.bs_get_kernel_timings.argtypes = [_vp, _dp, _dp, C.POINTER(C.c_int64)]
lib.bs_fp64_peak.argtypes = [_dp, _dp, _vp]
lib.bs_zgemm.argtypes = [C.c_int32] * 5 + [_dp, _vp, C.c_int32, C.c_int64, _vp, C.c_int32, C.c_int64, _dp, _vp, C.c_int32,
                                           C.c_int64, C.c_int32, C.c_int32, _vp]
lib.bs_zpotrf_trtri.argtypes = [C.c_int32, _vp, C.c_int32, C.c_int64, _vp, _vp, _vp, _vp, C.c_int32, _vp]
lib.bs_zhetrd.argtypes = [C.c_int32, _vp, C.c_int32, C.c_int64, _vp, _vp, _vp, C.c_int32, C.c_int32, C.c_int32, _vp]
lib.bs_sturm.argtypes = [C.c_int32, _vp, _vp, C.c_int32, _vp, C.c_int32, _vp]
lib.bs_zhetrd_static_bytes.restype = C.c_size_t
lib.bs_zhetrd_static_bytes.argtypes = [C.c_int32, C.c_int32]
lib.bs_zhetrd_static.argtypes = [C.c_int32, _vp, C.c_int32, C.c_int64, _vp, _vp, C.c_int32, _vp]
for _name in SYMBOLS:
    if _name not in ("bs_last_error", "bs_launch_count", "bs_zhetrd_scratch_elems", "bs_zhetrd_static_bytes", "bs_destroy_cell"):
        getattr(lib, _name).restype = C.c_int


def _check(status: int) -> None:
    if status != BS_OK:
        raise BsError(status, (lib.bs_last_error() or b"").decode())


def bs_last_error() -> str:
    return (lib.bs_last_error() or b"").decode()


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a: np.ndarray, typ=_dp):
    return a.ctypes.data_as(typ)


def _stream(stream) -> Optional[int]:
    """cudaStream_t of a torch stream (None -> torch's current stream)."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def bs_isotropic_plane_strain(E, nu) -> np.ndarray:
    """PAPER.md:121 (eq. 14).  Returns (n,6) [D1111 D2222 D1122 D1112 D2212 D1212]."""
    E, nu = _f64(E).ravel(), _f64(nu).ravel()
    out = np.empty((E.shape[0], 6))
    _check(lib.bs_isotropic_plane_strain(E.shape[0], _ptr(E), _ptr(nu), _ptr(out)))
    return out


class Cell:
    """Owner of one ``bs_cell`` handle and of the torch workspace tensor lent to it."""

    def __init__(self, lattice=None, vert_offset=None, verts=None, compliance=None, density=None, _adopt=None):
        if _adopt is not None:      # a handle created by bs_create_cells_shared
            self.handle, self.nphase = _adopt
            self.workspace = None
            self.Mt = None
            return
        lattice = _f64(lattice).reshape(4)
        off = np.ascontiguousarray(np.asarray(vert_offset, dtype=np.int32))
        verts = _f64(verts).reshape(-1)
        compliance = _f64(compliance).reshape(-1)
        density = _f64(density).reshape(-1)
        self.nphase = int(off.shape[0] - 1)
        if compliance.shape[0] != 6 * self.nphase or density.shape[0] != self.nphase or verts.shape[0] != 2 * int(off[-1]):
            raise BsError(BS_ERR_ARG, "array sizes do not match nphase / vert_offset")
        h = _vp()
        _check(lib.bs_create_cell(_ptr(lattice), self.nphase, _ptr(off, _ip), _ptr(verts), _ptr(compliance),
                                  _ptr(density), C.byref(h)))
        self.handle = h
        self.workspace = None
        self.Mt = None

    def close(self):
        if getattr(self, "handle", None) and lib is not None:   # lib is None during interpreter shutdown
            lib.bs_destroy_cell(self.handle)
            self.handle = None
            self.workspace = None

    def __del__(self):
        self.close()

    @property
    def N(self) -> int:
        return (2 * self.Mt + 1) ** 2


def bs_create_cell(lattice, vert_offset, verts, compliance, density) -> Cell:
    return Cell(lattice, vert_offset, verts, compliance, density)


def bs_create_cells_shared(lattice, vert_offset, verts, compliances, densities):
    """ncells handles that share ONE geometry: ``compliances`` (ncells, P, 6), ``densities``
    (ncells, P).  Returns a list of Cell."""
    lattice = _f64(lattice).reshape(4)
    off = np.ascontiguousarray(np.asarray(vert_offset, dtype=np.int32))
    verts = _f64(verts).reshape(-1)
    P = int(off.shape[0] - 1)
    comp = _f64(compliances).reshape(-1, P, 6)
    rho = _f64(densities).reshape(-1, P)
    ncells = comp.shape[0]
    if rho.shape[0] != ncells or verts.shape[0] != 2 * int(off[-1]):
        raise BsError(BS_ERR_ARG, "array sizes do not match nphase / vert_offset / ncells")
    hs = (_vp * ncells)()
    _check(lib.bs_create_cells_shared(_ptr(lattice), P, _ptr(off, _ip), _ptr(verts), ncells, _ptr(comp), _ptr(rho), hs))
    return [Cell(_adopt=(_vp(h), P)) for h in hs]


def bs_set_properties(cell: Cell, compliance, density) -> None:
    comp, rho = _f64(compliance).reshape(-1), _f64(density).reshape(-1)
    if comp.shape[0] != 6 * cell.nphase or rho.shape[0] != cell.nphase:
        raise BsError(BS_ERR_ARG, "array sizes do not match nphase")
    _check(lib.bs_set_properties(cell.handle, _ptr(comp), _ptr(rho)))


def bs_destroy_cell(cell: Cell) -> None:
    cell.close()


def bs_set_option(cell: Cell, option: int, value: int) -> None:
    _check(lib.bs_set_option(cell.handle, option, value))


def bs_workspace_bytes(cell: Cell, truncation: int, nk: int) -> int:
    b = C.c_size_t(0)
    _check(lib.bs_workspace_bytes(cell.handle, truncation, nk, C.byref(b)))
    return int(b.value)


def bs_set_workspace(cell: Cell, tensor) -> None:
    """Lend a torch uint8 CUDA tensor (kept alive by the Cell)."""
    _check(lib.bs_set_workspace(cell.handle, C.c_void_p(tensor.data_ptr()), tensor.numel() * tensor.element_size()))
    cell.workspace = tensor


def allocate_workspace(cell: Cell, truncation: int, nk: int, device="cuda:0") -> None:
    import torch
    nbytes = bs_workspace_bytes(cell, truncation, nk)
    bs_set_workspace(cell, torch.empty(nbytes, dtype=torch.uint8, device=device))


def bs_assemble(cell: Cell, truncation: int, stream=None) -> None:
    _check(lib.bs_assemble(cell.handle, truncation, _stream(stream)))
    cell.Mt = truncation


def _handles(cells: Sequence[Cell]):
    arr = (_vp * len(cells))(*[c.handle for c in cells])
    return arr


def bs_assemble_batch(cells: Sequence[Cell], truncation: int, stream=None) -> None:
    _check(lib.bs_assemble_batch(_handles(cells), len(cells), truncation, _stream(stream)))
    for c in cells:
        c.Mt = truncation


def bs_get_matrices(cell: Cell):
    """Phi (3N,3N) and Psi (2N,2N) as NumPy complex128 arrays (row index = test function)."""
    N = cell.N
    phi = np.empty((3 * N, 3 * N), dtype=np.complex128, order="F")
    psi = np.empty((2 * N, 2 * N), dtype=np.complex128, order="F")
    _check(lib.bs_get_matrices(cell.handle, phi.ctypes.data_as(_vp), psi.ctypes.data_as(_vp)))
    return phi, psi


def bs_get_table(cell: Cell) -> np.ndarray:
    L = 4 * cell.Mt + 1
    tab = np.empty((7, L, L), dtype=np.complex128)
    _check(lib.bs_get_table(cell.handle, tab.ctypes.data_as(_vp)))
    return tab


def bs_get_pencil(cell: Cell, kred, stream=None) -> np.ndarray:
    n = 2 * cell.N
    K = np.empty((n, n), dtype=np.complex128, order="F")
    k = _f64(kred).reshape(2)
    _check(lib.bs_get_pencil(cell.handle, _ptr(k), K.ctypes.data_as(_vp), _stream(stream)))
    return K


def _out_pointer(out, shape):
    """Validates a caller-supplied result buffer (float64, C-contiguous, exactly `shape`) and returns its address: a
    wrong buffer would otherwise be a host or device overflow inside the library."""
    n = int(np.prod(shape))
    if isinstance(out, np.ndarray):
        if out.dtype != np.float64 or not out.flags["C_CONTIGUOUS"] or out.size != n or not out.flags["WRITEABLE"]:
            raise BsError(BS_ERR_ARG, f"out must be a writable C-contiguous float64 array of {n} elements")
        return C.c_void_p(out.ctypes.data)
    import torch
    if not isinstance(out, torch.Tensor) or out.dtype != torch.float64 or not out.is_contiguous() or out.numel() != n:
        raise BsError(BS_ERR_ARG, f"out must be a contiguous float64 NumPy array or torch tensor of {n} elements")
    return C.c_void_p(out.data_ptr())


def bs_bands(cell: Cell, kpts, nbands: int, out=None, stream=None):
    """omega^2 (nk, nbands), ascending.  ``out``: None -> new host NumPy array; a NumPy array (host) or a torch CUDA
    float64 tensor (device) is filled in place and returned."""
    k = _f64(kpts).reshape(-1, 2)
    nk = k.shape[0]
    if out is None:
        out = np.empty((nk, nbands))
    p = _out_pointer(out, (nk, nbands))
    _check(lib.bs_bands(cell.handle, nk, _ptr(k), nbands, p, _stream(stream)))
    cell.last_nmat = nk
    return out


def bs_bands_batch(cells: Sequence[Cell], kpts, nbands: int, out=None, stream=None):
    k = _f64(kpts).reshape(-1, 2)
    nk = k.shape[0]
    if out is None:
        out = np.empty((len(cells), nk, nbands))
    p = _out_pointer(out, (len(cells), nk, nbands))
    _check(lib.bs_bands_batch(_handles(cells), len(cells), nk, _ptr(k), nbands, p, _stream(stream)))
    cells[0].last_nmat = len(cells) * nk
    return out


def bs_modes(cell: Cell, kpts, nbands: int, stress: bool = True, stream=None):
    """Mode shapes: returns (omega2 (nk, nbands), U (nk, 2N, nbands), S (nk, 3N, nbands) or None) as host
    NumPy arrays; U[k][:, j] is the Psi-orthonormal displacement coefficient vector of band j."""
    k = _f64(kpts).reshape(-1, 2)
    nk, N = k.shape[0], cell.N
    lam = np.empty((nk, nbands))
    U = np.empty((nk, nbands, 2 * N), dtype=np.complex128)          # block k is column-major 2N x nbands
    S = np.empty((nk, nbands, 3 * N), dtype=np.complex128) if stress else None
    _check(lib.bs_modes(cell.handle, nk, _ptr(k), nbands, C.c_void_p(lam.ctypes.data), C.c_void_p(U.ctypes.data),
                        C.c_void_p(S.ctypes.data) if stress else None, _stream(stream)))
    cell.last_nmat = nk
    return lam, U.transpose(0, 2, 1), (S.transpose(0, 2, 1) if stress else None)


def bs_modes_batch(cells: Sequence[Cell], kpts, nbands: int, stress: bool = True, stream=None):
    """bs_modes for a batch of handles: (omega2 (ncells, nk, nbands), U (ncells, nk, 2N, nbands), S (ncells, nk, 3N, nbands)
    or None) as host NumPy arrays."""
    k = _f64(kpts).reshape(-1, 2)
    nc, nk, N = len(cells), k.shape[0], cells[0].N
    lam = np.empty((nc, nk, nbands))
    U = np.empty((nc, nk, nbands, 2 * N), dtype=np.complex128)
    S = np.empty((nc, nk, nbands, 3 * N), dtype=np.complex128) if stress else None
    _check(lib.bs_modes_batch(_handles(cells), nc, nk, _ptr(k), nbands, C.c_void_p(lam.ctypes.data), C.c_void_p(U.ctypes.data),
                              C.c_void_p(S.ctypes.data) if stress else None, _stream(stream)))
    cells[0].last_nmat = nc * nk
    return lam, U.transpose(0, 1, 3, 2), (S.transpose(0, 1, 3, 2) if stress else None)


def bs_get_tridiagonal(cell: Cell, nmat: Optional[int] = None):
    """d, e (nmat, 2N) of the last bs_bands / bs_bands_batch call led by ``cell`` (nmat is taken from that call)."""
    known = getattr(cell, "last_nmat", None)
    if known is None:
        raise BsError(BS_ERR_STATE, "bs_get_tridiagonal: no bs_bands call led by this handle yet")
    if nmat is not None and nmat != known:
        raise BsError(BS_ERR_ARG, f"bs_get_tridiagonal: the last call had {known} matrices, not {nmat}")
    n = 2 * cell.N
    d = np.empty((known, n))
    e = np.empty((known, n))
    _check(lib.bs_get_tridiagonal(cell.handle, _ptr(d), _ptr(e)))
    return d, e


def bs_get_timings(cell: Cell) -> np.ndarray:
    ms = np.zeros(BS_T_COUNT)
    _check(lib.bs_get_timings(cell.handle, _ptr(ms)))
    return ms


KERNEL_CLASSES = ["table", "expand", "gemm_factor", "gemm_reduce", "gemm_tridiag", "hemv", "panel", "sturm", "pencil",
                  "combine", "potrf_diag", "other", "bulge", "gemm_hemm", "gemm_wy", "tridiag_small"]


def bs_get_kernel_timings(cell: Cell) -> dict:
    """{class: (ms, algorithmic work, launches)} of the last call led by ``cell`` under BS_OPT_TIMING = 2."""
    n = len(KERNEL_CLASSES)
    ms, work, cnt = np.zeros(n), np.zeros(n), np.zeros(n, dtype=np.int64)
    _check(lib.bs_get_kernel_timings(cell.handle, _ptr(ms), _ptr(work), cnt.ctypes.data_as(C.POINTER(C.c_int64))))
    return {k: (float(ms[i]), float(work[i]), int(cnt[i])) for i, k in enumerate(KERNEL_CLASSES)}


def bs_launch_count(cell: Cell) -> int:
    return int(lib.bs_launch_count(cell.handle))


def bs_fp64_peak(stream=None):
    """(DMMA TFLOP/s, DFMA TFLOP/s) of the current device, measured now."""
    a, b = C.c_double(0), C.c_double(0)
    _check(lib.bs_fp64_peak(C.byref(a), C.byref(b), _stream(stream)))
    return float(a.value), float(b.value)


# ---- diagnostics on torch CUDA tensors (complex128, column-major = the transpose of a contiguous torch tensor)
def bs_zgemm(opA, opB, M, N, K, alpha, A, lda, strideA, B, ldb, strideB, beta, Cm, ldc, strideC, batch=1, flags=0, stream=None):
    al = np.array([complex(alpha).real, complex(alpha).imag])
    be = np.array([complex(beta).real, complex(beta).imag])
    _check(lib.bs_zgemm(opA, opB, M, N, K, _ptr(al), C.c_void_p(A.data_ptr()), lda, strideA, C.c_void_p(B.data_ptr()), ldb,
                        strideB, _ptr(be), C.c_void_p(Cm.data_ptr()), ldc, strideC, batch, flags, _stream(stream)))


def bs_zpotrf_trtri(n, A, lda, strideA, X, tmp, dinv, info, batch=1, stream=None):
    _check(lib.bs_zpotrf_trtri(n, C.c_void_p(A.data_ptr()), lda, strideA, C.c_void_p(X.data_ptr()), C.c_void_p(tmp.data_ptr()),
                               C.c_void_p(dinv.data_ptr()), C.c_void_p(info.data_ptr()), batch, _stream(stream)))


def bs_zhetrd_scratch_elems(n: int, nb: int) -> int:
    return int(lib.bs_zhetrd_scratch_elems(n, nb))


def bs_zhetrd(n, A, lda, strideA, d, e, scratch, nb=32, algo=BS_TRIDIAG_TWO_STAGE, batch=1, stream=None):
    _check(lib.bs_zhetrd(n, C.c_void_p(A.data_ptr()), lda, strideA, C.c_void_p(d.data_ptr()), C.c_void_p(e.data_ptr()),
                         C.c_void_p(scratch.data_ptr()), nb, algo, batch, _stream(stream)))


BS_ZHETRD_STATIC_BYTES = 8 * 1024 * 1024


def bs_zhetrd_static_bytes(n: int, batch: int = 1) -> int:
    return int(lib.bs_zhetrd_static_bytes(n, batch))


def bs_zhetrd_static(n, A, lda, strideA, d, e, batch=1, stream=None):
    """bs_zhetrd with its scratch in the library's static device array: no allocation, no synchronisation (bs.h)."""
    _check(lib.bs_zhetrd_static(n, C.c_void_p(A.data_ptr()), lda, strideA, C.c_void_p(d.data_ptr()),
                                C.c_void_p(e.data_ptr()), batch, _stream(stream)))


def bs_sturm(n, d, e, nev, lam, batch=1, stream=None):
    _check(lib.bs_sturm(n, C.c_void_p(d.data_ptr()), C.c_void_p(e.data_ptr()), nev, C.c_void_p(lam.data_ptr()), batch,
                        _stream(stream)))
