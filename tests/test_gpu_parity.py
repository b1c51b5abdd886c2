"""GPU parity tests (-m gpu): the CUDA path through the C-ABI (ctypes binding) against the CPU oracle on the same
seeded inputs.  Tolerances: matrices <= 1e-12 norm-wise (R7 / SURVEY A14); eigenfrequencies
<= 1e-9 relative OR |dlambda| <= 64 eps lambda_max (R8 / SURVEY A15)."""
import os

import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu
EPS = 2.0 ** -53
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden(name, w):
    """Stored oracle result for EVERY k-point of config `name` (tests/golden/make_goldens.py, oracle only)."""
    g = np.load(os.path.join(GOLDEN, f"{name}_lambda.npz"))
    assert np.array_equal(g["kpts"], w.kpts), "golden file was written for a different k-path"
    return g


@pytest.fixture(scope="module")
def bs():
    import torch
    assert torch.cuda.is_available()
    import paper_1310_6380_b200 as bs
    return bs


def make_cell(bs, cell, Mt, nk, mode=None, panel=None, algo=None):
    comp = bs.bs_isotropic_plane_strain(cell.E, cell.nu)
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho)
    if mode is not None:
        bs.bs_set_option(h, bs.BS_OPT_PENCIL_MODE, mode)
    if panel is not None:
        bs.bs_set_option(h, bs.BS_OPT_PANEL, panel)
    if algo is not None:
        bs.bs_set_option(h, bs.BS_OPT_TRIDIAG, algo)
    bs.allocate_workspace(h, Mt, nk)
    return h


def check_bands(lam_gpu, lam_ref, lmax, tag=""):
    """R8: pass if |omega_gpu - omega_ref| <= 1e-9 omega_ref or |dlambda| <= 64 eps lambda_max.  Returns the number of
    (k, band) pairs that needed the second clause."""
    om_g, om_r = np.sqrt(np.maximum(lam_gpu, 0)), np.sqrt(np.maximum(lam_ref, 0))
    with np.errstate(divide="ignore", invalid="ignore"):
        rel_ok = np.abs(om_g - om_r) <= 1e-9 * om_r
    back_ok = np.abs(lam_gpu - lam_ref) <= 64 * EPS * lmax[:, None]
    bad = ~(rel_ok | back_ok)
    assert not bad.any(), (tag, np.argwhere(bad)[:5], lam_gpu[bad][:5], lam_ref[bad][:5])
    return int((~rel_ok).sum())


def oracle_inputs(cell):
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
    return cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho


def test_compliance_matches_oracle(bs):
    E, nu = np.array([1e9, 70e9, 3.5e9]), np.array([0.2, 0.33, 0.45])
    assert np.allclose(bs.bs_isotropic_plane_strain(E, nu), oracle.isotropic_plane_strain_compliance(E, nu), rtol=1e-15)


# (C2, 1) and (C3, 1): the separable-phase table does not fit the scratch of so small a truncation -> direct kernel;
# (C3, 10), (C5, 15): the full-size tables of the bench workloads
@pytest.mark.parametrize("name,Mt", [("C1", 3), ("C2", 3), ("C3", 4), ("C2", 1), ("C3", 1), ("C2", 7), ("C3", 10), ("C5", 15)])
def test_table_and_matrices_parity(bs, name, Mt):
    cell = wl.get(name).cells[0]
    h = make_cell(bs, cell, Mt, 1)
    bs.bs_assemble(h, Mt)
    Phi, Psi = bs.bs_get_matrices(h)
    Pr, Sr = oracle.assemble(*oracle_inputs(cell), Mt)
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
    assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    assert np.array_equal(Phi, Phi.conj().T) and np.array_equal(Psi, Psi.conj().T)   # exactly Hermitian by construction
    # the table, channel by channel (general-D channel order of include/bs.h)
    Dv = oracle.voigt_compliance(oracle_inputs(cell)[3])
    W = np.stack([Dv[:, 0, 0], Dv[:, 1, 1], Dv[:, 0, 1], Dv[:, 0, 2], Dv[:, 1, 2], Dv[:, 2, 2], cell.rho])
    tr = oracle.shape_integral_table(cell.lattice, cell.vert_offset, cell.verts, W, Mt)
    tg = bs.bs_get_table(h)
    for c in range(7):
        scale = np.max(np.abs(tr[c]))
        if scale == 0:
            assert np.max(np.abs(tg[c])) == 0
        else:
            assert np.max(np.abs(tg[c] - tr[c])) <= 1e-12 * scale
    bs.bs_destroy_cell(h)


def test_table_when_q_is_perpendicular_to_edges_up_to_rounding(bs):
    """S1 divides sin(q.e/2) by q.e/2.  Triangles on a 0.2 grid (not exact in binary) have edges (0.2, 0), (0, 0.2) and
    (0.2, 0.2): for D1 = -D2 the exact q.e vanishes but its floating-point value is a rounding residue of ~1e-17, and for
    other index differences it is an integer multiple of 0.2 pi; the kernel's product form of sin(pi u) (absolute error
    ~2e-16) must not be divided by such a residue."""
    rng = np.random.default_rng(99)
    polys = []
    for i in range(5):
        for j in range(5):
            x0, y0, x1, y1 = 0.2 * i, 0.2 * j, 0.2 * (i + 1), 0.2 * (j + 1)
            polys.append(np.array([[x0, y0], [x1, y0], [x1, y1]]))
            polys.append(np.array([[x0, y0], [x1, y1], [x0, y1]]))
    P = len(polys)
    cell = wl.Cell(lattice=np.eye(2), vert_offset=np.arange(0, 3 * P + 1, 3, dtype=np.int32), verts=np.concatenate(polys),
                   E=rng.uniform(1e9, 2e11, P), nu=rng.uniform(0.2, 0.4, P), rho=rng.uniform(1e3, 8e3, P))
    Mt = 4
    h = make_cell(bs, cell, Mt, 1)
    bs.bs_assemble(h, Mt)
    Phi, Psi = bs.bs_get_matrices(h)
    Pr, Sr = oracle.assemble(*oracle_inputs(cell), Mt)
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
    assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    bs.bs_destroy_cell(h)


def test_anisotropic_matrices_parity(bs):
    cell = wl.random_small_cell(21, 3, np.array([[1.0, 0.0], [0.3, 0.8]]))
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu).copy()
    comp[:, 3] = 0.01 * comp[:, 0]
    comp[:, 4] = -0.02 * comp[:, 0]
    comp[:, 1] *= 1.1
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho)
    bs.allocate_workspace(h, 2, 4)
    bs.bs_assemble(h, 2)
    Phi, Psi = bs.bs_get_matrices(h)
    Pr, Sr = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, 2)
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
    assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    kp = np.array([[0.1, 0.2], [0.5, 0.0], [0.0, 0.0], [0.33, 0.44]])
    lam = bs.bs_bands(h, kp, 10)
    for i, kr in enumerate(kp):
        lr, lmax = oracle.bands_at_k(Pr, Sr, cell.lattice, 2, kr, 10)
        check_bands(lam[i:i + 1], lr[None, :], np.array([lmax]))
    bs.bs_destroy_cell(h)


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("phi_general", [0, 1])
def test_pencil_parity(bs, mode, phi_general):
    # phi_general = 0: isotropic shortcut (two N x N inverses); 1: full 3N x 3N Cholesky inverse
    cell = wl.get("C1").cells[0]
    h = make_cell(bs, cell, 3, 1, mode=mode)
    bs.bs_set_option(h, bs.BS_OPT_PHI_INVERSE, phi_general)
    bs.bs_assemble(h, 3)
    Pr, _ = oracle.assemble(*oracle_inputs(cell), 3)
    for kr in [(0.31, 0.12), (0.5, 0.5), (0.0, 0.0)]:
        K = bs.bs_get_pencil(h, kr)
        Kr = oracle.pencil_K(Pr, cell.lattice, 3, kr)
        assert np.max(np.abs(K - Kr)) <= 1e-11 * np.max(np.abs(Kr))   # cond(Phi) ~ 1e2 amplifies the 1e-12 of Phi
    bs.bs_destroy_cell(h)


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("panel", [8, 16, 32])
@pytest.mark.parametrize("algo", [0, 1])
def test_config1_bands_parity(bs, mode, panel, algo):
    w = wl.get("C1")
    cell = w.cells[0]
    h = make_cell(bs, cell, w.Mt, w.nk, mode=mode, panel=panel, algo=algo)
    bs.bs_assemble(h, w.Mt)
    lam = bs.bs_bands(h, w.kpts, w.nbands)
    lr, lmax = oracle.band_structure(*oracle_inputs(cell), w.Mt, w.kpts, w.nbands)
    n2 = check_bands(lam, lr, lmax, "C1")
    assert n2 <= 8   # the two zero modes at each Gamma end (+ nearest neighbours)
    bs.bs_destroy_cell(h)


def test_homogeneous_dispersion_on_gpu(bs):
    # physics pin applied directly to the CUDA path: omega = c |k+G|
    E, nu, rho = 20e9, 0.28, 2500.0
    cell = wl.homogeneous_cell(wl.HEXAGONAL, E, nu, rho, n=2)
    Mt = 3
    h = make_cell(bs, cell, Mt, 3)
    bs.bs_assemble(h, Mt)
    kp = np.array([(0.31, 0.12), (0.5, 0.0), (0.05, 0.45)])
    nb = 2 * (2 * Mt + 1) ** 2
    lam = bs.bs_bands(h, kp, nb)
    lam_, mu_ = E * nu / ((1 + nu) * (1 - 2 * nu)), E / (2 * (1 + nu))
    cL, cT = np.sqrt((lam_ + 2 * mu_) / rho), np.sqrt(mu_ / rho)
    _, Q, _ = oracle.reciprocal_basis(cell.lattice)
    for i, kr in enumerate(kp):
        kap = np.linalg.norm((oracle.plane_wave_indices(Mt) + np.array(kr)) @ Q, axis=1)
        ref = np.sort(np.concatenate([cL * kap, cT * kap]))
        assert np.max(np.abs(np.sqrt(np.maximum(lam[i], 0)) - ref) / ref) < 1e-10
    bs.bs_destroy_cell(h)


def test_homogeneous_anisotropic_dispersion_on_gpu(bs):
    # PAPER.md:167-171 (eq. 20): the CUDA path's reading of the factors 2 / 4 on the shear-coupling compliances, pinned
    # directly to the Christoffel closed form of tests/closed_forms.py (independent of the oracle), general 3N x 3N path
    from closed_forms import ANISO_FIELDS, christoffel_frequencies
    rho, Mt = 3100.0, 2
    cell = wl.homogeneous_cell(wl.HEXAGONAL, 1.0, 0.3, rho, n=2)
    comp = np.tile(ANISO_FIELDS, (cell.nphase, 1))
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho)
    bs.allocate_workspace(h, Mt, 3)
    bs.bs_assemble(h, Mt)
    kp = np.array([(0.31, 0.12), (0.5, 0.0), (-0.2, 0.45)])
    nb = 2 * (2 * Mt + 1) ** 2
    lam = bs.bs_bands(h, kp, nb)
    _, Q, _ = oracle.reciprocal_basis(cell.lattice)
    for i, kr in enumerate(kp):
        kap = (oracle.plane_wave_indices(Mt) + np.array(kr)) @ Q
        ref = np.sort(christoffel_frequencies(ANISO_FIELDS, rho, kap).ravel())
        assert np.max(np.abs(np.sqrt(np.maximum(lam[i], 0)) - ref) / ref) < 1e-10
    bs.bs_destroy_cell(h)


def test_config2_bands_parity_every_kpoint(bs):
    w = wl.get("C2")
    cell = w.cells[0]
    h = make_cell(bs, cell, w.Mt, w.nk)
    bs.bs_assemble(h, w.Mt)
    lam = bs.bs_bands(h, w.kpts, w.nbands)
    Pr, Sr = oracle.assemble(*oracle_inputs(cell), w.Mt)
    Phi, Psi = bs.bs_get_matrices(h)
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
    assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    g = golden("C2", w)
    n2 = check_bands(lam, g["lam"], g["lam_max"], "C2")      # all 60 k-points x 10 bands
    assert n2 <= 6, n2    # the two zero modes at each Gamma end (+ the acoustic pair next to one of them)
    bs.bs_destroy_cell(h)


@pytest.mark.parametrize("algo,panel", [(0, 32), (0, 16), (1, 32)])
def test_config3_bands_parity_every_kpoint(bs, algo, panel):
    w = wl.get("C3")
    cell = w.cells[0]
    h = make_cell(bs, cell, w.Mt, w.nk, algo=algo, panel=panel)
    bs.bs_assemble(h, w.Mt)
    lam = bs.bs_bands(h, w.kpts, w.nbands)
    g = golden("C3", w)
    n2 = check_bands(lam, g["lam"], g["lam_max"], "C3")      # all 90 k-points x 18 bands
    assert n2 <= 8, n2
    bs.bs_destroy_cell(h)


def test_config4_batch_parity_sampled(bs):
    w = wl.get("C4", ncells=8)
    cells = [make_cell(bs, c, w.Mt, w.nk) for c in w.cells]
    bs.bs_assemble_batch(cells, w.Mt)
    lam = bs.bs_bands_batch(cells, w.kpts, w.nbands)
    assert lam.shape == (8, w.nk, w.nbands)
    for ci in [0, 5, 7]:
        Pr, Sr = oracle.assemble(*oracle_inputs(w.cells[ci]), w.Mt)
        Phi, Psi = bs.bs_get_matrices(cells[ci])
        assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
        for i in [0, 3, 21, 39]:
            lr, lmax = oracle.bands_at_k(Pr, Sr, w.cells[ci].lattice, w.Mt, w.kpts[i], w.nbands)
            check_bands(lam[ci, i:i + 1], lr[None, :], np.array([lmax]), f"C4 cell{ci} k{i}")
    for c in cells:
        bs.bs_destroy_cell(c)


def test_config5_bands_parity_every_kpoint(bs):
    # full size of config 5 (n = 1922, 120 k-points in one call, as bench.py launches it) against the stored oracle
    # result at EVERY k-point (tests/golden/C5_lambda.npz)
    w = wl.get("C5")
    cell = w.cells[0]
    h = make_cell(bs, cell, w.Mt, w.nk)
    bs.bs_assemble(h, w.Mt)
    lam = bs.bs_bands(h, w.kpts, w.nbands)
    assert lam.shape == (w.nk, w.nbands)
    Pr, Sr = oracle.assemble(*oracle_inputs(cell), w.Mt)
    Phi, Psi = bs.bs_get_matrices(h)
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
    assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    g = golden("C5", w)
    n2 = check_bands(lam, g["lam"], g["lam_max"], "C5")      # all 120 k-points x 18 bands
    assert n2 <= 10, n2     # the two zero modes at each Gamma end and the acoustic pairs at the 1-2 nearest points (R8)
    bs.bs_destroy_cell(h)


def test_config4_full_batch(bs):
    # the whole optimisation-loop batch (256 cells x 40 k-points = 10240 eigenproblems in one call)
    w = wl.get("C4")
    cells = [make_cell(bs, c, w.Mt, w.nk) for c in w.cells]
    bs.bs_assemble_batch(cells, w.Mt)
    lam = bs.bs_bands_batch(cells, w.kpts, w.nbands)
    assert lam.shape == (256, w.nk, w.nbands)
    g = golden("C4", w)
    n2 = 0
    for j, ci in enumerate(g["cells"]):          # 16 cells spread over the batch, all 40 k-points of each
        n2 += check_bands(lam[ci], g["lam"][j], g["lam_max"][j], f"C4 cell{ci}")
    assert n2 <= 6 * len(g["cells"]), n2
    # every other cell: same geometry, materials permuted -> its spectrum obeys the same bounds (physics, any size):
    # two zero modes at the Gamma ends, ascending, and lambda <= the largest lambda_max of the batch's golden cells
    assert np.all(np.diff(lam, axis=2) >= 0)
    assert np.all(np.abs(lam[:, [0, -1], :2]) <= 64 * EPS * 4 * g["lam_max"].max())
    assert np.all(lam[:, 1:-1, 2:] > 0) and np.all(lam <= g["lam_max"].max())
    Pr, Sr = oracle.assemble(*oracle_inputs(w.cells[255]), w.Mt)
    # a batch call equals the single-cell calls bit for bit (same kernels, same order of operations)
    one = bs.bs_bands(cells[131], w.kpts, w.nbands)
    assert np.array_equal(one, lam[131])
    # stage 2 streamed through the three-sweep ring (three CTAs per SM here) instead of the resident band: reproducible
    # bit for bit, and the same eigenvalues to the backward error of the reduction (64 eps lambda_max, reading R8)
    for c in cells:
        bs.bs_set_option(c, bs.BS_OPT_TRIDIAG, bs.BS_TRIDIAG_TWO_STAGE_STREAMED)
    ls = bs.bs_bands_batch(cells, w.kpts, w.nbands)
    assert np.array_equal(bs.bs_bands_batch(cells, w.kpts, w.nbands), ls)
    _, lmax = oracle.bands_at_k(Pr, Sr, w.cells[255].lattice, w.Mt, w.kpts[39], w.nbands)
    assert np.max(np.abs(ls - lam)) <= 64 * EPS * 4 * lmax  # lambda_max varies by less than 4x over the batch
    for c in cells:
        bs.bs_destroy_cell(c)


def test_centroid_rule_assembly_parity(bs):
    # BS_OPT_ASSEMBLY = centroid (eq. 12): matrices and bands against the oracle's centroid-rule assembly
    w = wl.get("C3")
    cell = w.cells[0]
    Mt = 4
    h = make_cell(bs, cell, Mt, 3)
    bs.bs_set_option(h, bs.BS_OPT_ASSEMBLY, bs.BS_ASSEMBLY_CENTROID)
    bs.bs_assemble(h, Mt)
    Phi, Psi = bs.bs_get_matrices(h)
    Pr, Sr = oracle.assemble(*oracle_inputs(cell), Mt, quadrature="centroid")
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
    assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    Pe, _ = oracle.assemble(*oracle_inputs(cell), Mt)
    assert 1e-6 < np.max(np.abs(Pr - Pe)) / np.max(np.abs(Pe)) < 0.2     # a different (coarser) quadrature, same limit
    kp = np.array([[0.2, 0.1], [0.5, 0.0], [0.0, 0.0]])
    lam = bs.bs_bands(h, kp, 12)
    for i, kr in enumerate(kp):
        lr, lmax = oracle.bands_at_k(Pr, Sr, cell.lattice, Mt, kr, 12)
        check_bands(lam[i:i + 1], lr[None, :], np.array([lmax]), f"centroid k{i}")
    bs.bs_destroy_cell(h)


def test_phi_inverse_paths_agree_on_bands(bs):
    w = wl.get("C2")
    cell = w.cells[0]
    out = []
    for general in (0, 1):
        h = make_cell(bs, cell, w.Mt, 6)
        bs.bs_set_option(h, bs.BS_OPT_PHI_INVERSE, general)
        bs.bs_assemble(h, w.Mt)
        out.append(bs.bs_bands(h, w.kpts[[0, 1, 9, 20, 40, 59]], w.nbands))
        bs.bs_destroy_cell(h)
    om0, om1 = np.sqrt(np.maximum(out[0], 0)), np.sqrt(np.maximum(out[1], 0))
    nz = om1 > 1e-3 * om1.max()
    assert np.max(np.abs(om0[nz] - om1[nz]) / om1[nz]) < 1e-9


def test_edge_cases_small_truncations_full_spectrum_single_k(bs):
    # Mt = 0 (one plane wave: K is 2 x 2), Mt = 1, nbands = 2N (the whole spectrum), nk = 1
    cell = wl.random_small_cell(31, 3, wl.HEXAGONAL)
    for Mt in (0, 1, 2):
        n2 = 2 * (2 * Mt + 1) ** 2
        h = make_cell(bs, cell, Mt, 1)
        bs.bs_assemble(h, Mt)
        Pr, Sr = oracle.assemble(*oracle_inputs(cell), Mt)
        kr = np.array([[0.37, 0.21]])
        lam = bs.bs_bands(h, kr, n2)
        lr, lmax = oracle.bands_at_k(Pr, Sr, cell.lattice, Mt, kr[0])
        check_bands(lam, lr[None, :], np.array([lmax]), f"Mt{Mt}")
        bs.bs_destroy_cell(h)


def test_truncation_limit_is_reported(bs):
    cell = wl.random_small_cell(1, 2)
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, bs.bs_isotropic_plane_strain(cell.E, cell.nu), cell.rho)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_workspace_bytes(h, 16, 1)          # 2N = 2178 > 2048
    assert ei.value.status == bs.BS_ERR_ARG
    assert bs.bs_workspace_bytes(h, 15, 1) > 0   # the maximum, config 5's truncation
    bs.bs_destroy_cell(h)


def test_nonconvex_and_translated_polygons(bs):
    # an L-shaped (non-convex) phase, and a phase given as a lattice-translated piece sticking out of the cell (R11)
    lattice = wl.SQUARE
    Lshape = np.array([[0, 0], [1, 0], [1, 0.4], [0.4, 0.4], [0.4, 1], [0, 1.0]])
    square = np.array([[0.4, 0.4], [1, 0.4], [1, 1], [0.4, 1.0]])
    E, nu, rho = np.array([5e9, 60e9]), np.array([0.3, 0.25]), np.array([1200.0, 2600.0])
    comp = oracle.isotropic_plane_strain_compliance(E, nu)
    results = []
    for shift in (np.zeros(2), np.array([1.0, 0.0]), np.array([-1.0, 2.0])):
        off, verts = wl._csr([Lshape, square + shift])
        h = bs.bs_create_cell(lattice, off, verts, bs.bs_isotropic_plane_strain(E, nu), rho)
        bs.allocate_workspace(h, 2, 2)
        bs.bs_assemble(h, 2)
        Phi, Psi = bs.bs_get_matrices(h)
        Pr, Sr = oracle.assemble(lattice, off, verts, comp, rho, 2)
        assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
        assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
        results.append(bs.bs_bands(h, [[0.3, 0.1], [0.5, 0.5]], 8))
        bs.bs_destroy_cell(h)
    # translating a phase by a lattice vector changes nothing (I_p(G) is invariant)
    assert np.allclose(results[0], results[1], rtol=1e-10) and np.allclose(results[0], results[2], rtol=1e-10)


def test_many_kpoints_and_repeated_calls(bs):
    w = wl.get("C1")
    cell = w.cells[0]
    kp = wl.kpath(cell.lattice, wl.SQUARE_PATH, 517)
    h = make_cell(bs, cell, w.Mt, 517)
    bs.bs_assemble(h, w.Mt)
    lam_all = bs.bs_bands(h, kp, 4)
    lam_part = bs.bs_bands(h, kp[100:133], 4)           # fewer k-points than the workspace was sized for
    assert np.array_equal(lam_part, lam_all[100:133])   # deterministic, independent of the batch it ran in
    import torch
    out = torch.empty(517, 4, dtype=torch.float64, device="cuda")
    bs.bs_bands(h, kp, 4, out=out)                      # device output pointer
    assert np.array_equal(out.cpu().numpy(), lam_all)
    bs.bs_destroy_cell(h)


def test_poly_and_direct_modes_agree_outside_first_zone(bs):
    # the k-polynomial form of A(k) (six k-independent matrices) against the per-k scaling kernel, also for k far outside
    # the first Brillouin zone, and against the oracle
    w = wl.get("C1")
    cell = w.cells[0]
    rng = np.random.default_rng(77)
    kp = np.concatenate([rng.uniform(-2.5, 2.5, size=(9, 2)), [[0.0, 0.0], [1.0, 0.0], [0.5, 0.5]]])
    lams = []
    for mode in (0, 1):
        h = make_cell(bs, cell, w.Mt, len(kp), mode=mode)
        bs.bs_assemble(h, w.Mt)
        lams.append(bs.bs_bands(h, kp, 12))
        bs.bs_destroy_cell(h)
    Pr, Sr = oracle.assemble(*oracle_inputs(cell), w.Mt)
    for i, kr in enumerate(kp):
        lr, lmax = oracle.bands_at_k(Pr, Sr, cell.lattice, w.Mt, kr, 12)
        for lam in lams:
            check_bands(lam[i:i + 1], lr[None, :], np.array([lmax]), f"k{i}")


def test_high_contrast_many_bands(bs):
    # stiffness contrast 1e4 and density contrast 50 (cond(Phi) ~ 1e5), 150 of 338 eigenvalues (several Sturm passes)
    cell = wl.get("C3").cells[0]
    rng = np.random.default_rng(5)
    E = np.where(rng.uniform(size=cell.nphase) < 0.5, 2e7, 2e11)
    rho = np.where(rng.uniform(size=cell.nphase) < 0.5, 200.0, 10000.0)
    nu = np.full(cell.nphase, 0.3)
    Mt = 6
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, bs.bs_isotropic_plane_strain(E, nu), rho)
    bs.allocate_workspace(h, Mt, 3)
    bs.bs_assemble(h, Mt)
    comp = oracle.isotropic_plane_strain_compliance(E, nu)
    Pr, Sr = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, rho, Mt)
    Phi, Psi = bs.bs_get_matrices(h)
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
    assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    kp = np.array([[0.5, 0.0], [0.21, 0.13], [2.0 / 3.0, 1.0 / 3.0]])
    lam = bs.bs_bands(h, kp, 150)
    for i, kr in enumerate(kp):
        lr, lmax = oracle.bands_at_k(Pr, Sr, cell.lattice, Mt, kr, 150)
        # the explicit inverse of an ill-conditioned Phi costs cond(Phi) eps in K: allow 1e-7 relative on omega here
        om_g, om_r = np.sqrt(np.maximum(lam[i], 0)), np.sqrt(np.maximum(lr, 0))
        assert np.max(np.abs(om_g - om_r) / om_r) < 1e-7, np.max(np.abs(om_g - om_r) / om_r)
    bs.bs_destroy_cell(h)


@pytest.mark.parametrize("Mt", [4, 6, 7])
def test_band_width_choices_agree_with_the_oracle(bs, Mt):
    # K is 162 x 162, 338 x 338 (automatic band width 16: the band stays in shared memory in stage 2) and 450 x 450
    # (automatic 32): the automatic choice and every explicit width give the oracle's eigenfrequencies
    cell = wl.get("C2").cells[0]
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
    Pr, Sr = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, Mt)
    kp = np.array([[0.0, 0.0], [0.5, 0.0], [0.31, 0.17]])
    refs = [oracle.bands_at_k(Pr, Sr, cell.lattice, Mt, kr, 12) for kr in kp]
    for panel in (None, 8, 16, 32):
        h = make_cell(bs, cell, Mt, len(kp), panel=panel)
        bs.bs_assemble(h, Mt)
        lam = bs.bs_bands(h, kp, 12)
        for i, (lr, lmax) in enumerate(refs):
            check_bands(lam[i:i + 1], lr[None, :], np.array([lmax]), f"Mt={Mt} panel={panel} k={i}")
        bs.bs_destroy_cell(h)


def test_output_omega_instead_of_omega_squared(bs):
    # S8 (omega_N = sqrt(lambda_N)): BS_OPT_OUTPUT = BS_OUTPUT_OMEGA writes sqrt(max(lambda, 0))
    w = wl.get("C1")
    cell = w.cells[0]
    h = make_cell(bs, cell, w.Mt, w.nk)
    bs.bs_assemble(h, w.Mt)
    lam = bs.bs_bands(h, w.kpts, w.nbands)
    bs.bs_set_option(h, bs.BS_OPT_OUTPUT, bs.BS_OUTPUT_OMEGA)
    om = bs.bs_bands(h, w.kpts, w.nbands)
    assert np.array_equal(om, np.sqrt(np.maximum(lam, 0.0)))  # sqrt is correctly rounded on both sides
    Pr, Sr = oracle.assemble(*oracle_inputs(cell), w.Mt)
    for i in (0, 3, 17):
        lr, lmax = oracle.bands_at_k(Pr, Sr, cell.lattice, w.Mt, w.kpts[i], w.nbands)
        om_r = np.sqrt(np.maximum(lr, 0.0))
        ok = (np.abs(om[i] - om_r) <= 1e-9 * om_r) | (np.abs(om[i] ** 2 - lr) <= 64 * EPS * lmax)
        assert ok.all()
    with pytest.raises(bs.BsError):
        bs.bs_set_option(h, bs.BS_OPT_OUTPUT, 2)
    bs.bs_destroy_cell(h)


def test_create_destroy_loop_reuses_device_blocks(bs):
    # An optimisation driver creates and destroys handles in a loop (bench.py's end-to-end arm does): the handle-owned
    # device blocks come from the library's cache of freed blocks, results stay bitwise equal and device memory does not grow.
    import torch
    w = wl.get("C1")
    cell = w.cells[0]
    ref = None
    free0 = None
    for it in range(25):
        h = make_cell(bs, cell, w.Mt, w.nk)
        bs.bs_assemble(h, w.Mt)
        lam = bs.bs_bands(h, w.kpts, w.nbands)
        bs.bs_destroy_cell(h)
        if ref is None:
            ref = lam.copy()
        assert np.array_equal(lam, ref)
        torch.cuda.synchronize()
        if it == 4:
            free0 = torch.cuda.mem_get_info()[0]
    torch.cuda.empty_cache()
    assert torch.cuda.mem_get_info()[0] >= free0 - (8 << 20)


def test_shared_geometry_batch_parity_and_property_updates(bs):
    # cells that share one geometry; S1 = polygon integrals once + T = W I per cell.
    # Matrices and bands against the oracle (which assembles every cell from scratch), against the per-cell path, and
    # after new properties are set on existing handles (the optimisation-loop iteration).
    w = wl.get("C4", ncells=6)
    c0 = w.cells[0]
    assert all(np.array_equal(c.verts, c0.verts) for c in w.cells)
    comps = np.stack([bs.bs_isotropic_plane_strain(c.E, c.nu) for c in w.cells])
    rhos = np.stack([c.rho for c in w.cells])
    shared = bs.bs_create_cells_shared(c0.lattice, c0.vert_offset, c0.verts, comps, rhos)
    for h in shared:
        bs.allocate_workspace(h, w.Mt, w.nk)
    bs.bs_assemble_batch(shared, w.Mt)
    lam = bs.bs_bands_batch(shared, w.kpts, w.nbands)
    single = [make_cell(bs, c, w.Mt, w.nk) for c in w.cells]
    bs.bs_assemble_batch(single, w.Mt)
    lam1 = bs.bs_bands_batch(single, w.kpts, w.nbands)
    for ci in (0, 3, 5):
        Pr, Sr = oracle.assemble(*oracle_inputs(w.cells[ci]), w.Mt)
        Phi, Psi = bs.bs_get_matrices(shared[ci])
        assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr))
        assert np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
        assert np.array_equal(Phi, Phi.conj().T)
        lr, lmax = oracle.band_structure(*oracle_inputs(w.cells[ci]), w.Mt, w.kpts, w.nbands)
        check_bands(lam[ci], lr, lmax, f"shared cell{ci}")
        check_bands(lam1[ci], lr, lmax, f"single cell{ci}")
    # one cell of the shared set alone gives the same bits as inside the batch
    bs.bs_assemble(shared[3], w.Mt)
    assert np.array_equal(bs.bs_bands(shared[3], w.kpts, w.nbands), lam[3])
    # optimisation-loop iteration: new properties on the same handles (cell j takes the materials of cell 5 - j)
    for j, h in enumerate(shared):
        bs.bs_set_properties(h, comps[5 - j], rhos[5 - j])
    with pytest.raises(bs.BsError):
        bs.bs_bands(shared[0], w.kpts, w.nbands)        # properties changed: must be assembled again
    bs.bs_assemble_batch(shared, w.Mt)
    lam2 = bs.bs_bands_batch(shared, w.kpts, w.nbands)
    assert np.array_equal(lam2, lam[::-1])
    # the centroid-rule quadrature goes through the shared path too
    for h in shared:
        bs.bs_set_option(h, bs.BS_OPT_ASSEMBLY, bs.BS_ASSEMBLY_CENTROID)
    bs.bs_assemble_batch(shared, 1)      # (at Mt = 5 the one-point rule aliases on the 8 x 8 pixels: Phi is then singular)
    Phi, _ = bs.bs_get_matrices(shared[1])
    Pc, _ = oracle.assemble(*oracle_inputs(w.cells[4]), 1, quadrature="centroid")
    assert np.max(np.abs(Phi - Pc)) <= 1e-12 * np.max(np.abs(Pc))
    # anisotropic phases and a skew lattice through the shared path
    cell = wl.random_small_cell(21, 3, np.array([[1.0, 0.0], [0.3, 0.8]]))
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu).copy()
    comp[:, 3] = 0.01 * comp[:, 0]
    comp[:, 4] = -0.02 * comp[:, 0]
    comp[:, 1] *= 1.1
    hs = bs.bs_create_cells_shared(cell.lattice, cell.vert_offset, cell.verts, np.stack([comp, 2 * comp]), np.stack([cell.rho, cell.rho]))
    for h in hs:
        bs.allocate_workspace(h, 2, 2)
    bs.bs_assemble_batch(hs, 2)
    Phi, Psi = bs.bs_get_matrices(hs[1])
    Pr, Sr = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, 2 * comp, cell.rho, 2)
    assert np.max(np.abs(Phi - Pr)) <= 1e-12 * np.max(np.abs(Pr)) and np.max(np.abs(Psi - Sr)) <= 1e-12 * np.max(np.abs(Sr))
    for h in shared + single + hs:
        bs.bs_destroy_cell(h)
