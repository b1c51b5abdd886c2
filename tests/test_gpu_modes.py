"""Mode shapes on the GPU (bs_modes) against the CPU oracle (oracle.modes_at_k = zhegv
with vectors).  Eigenvectors are unique only up to a phase and, inside a degenerate eigenvalue, up to the basis: compared
are what is unique (the eigenvalues, the Psi-orthogonal projector onto every well-separated cluster of branches) and the
defining equations (K U = Psi U Lambda, U^H Psi U = I, Phi S = H U, H^H S = Psi U Lambda: eq. 10)."""
import numpy as np
import pytest

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu
EPS = 2.0 ** -53


@pytest.fixture(scope="module")
def bs():
    import torch
    assert torch.cuda.is_available()
    import paper_1310_6380_b200 as bs
    return bs


def clusters(lam, lmax, rel=1e-7):
    """Index ranges of branches whose neighbours are closer than rel * lambda_max (degenerate or nearly so)."""
    out, start = [], 0
    for j in range(1, len(lam) + 1):
        if j == len(lam) or lam[j] - lam[j - 1] > rel * lmax:
            out.append((start, j))
            start = j
    return out


def check_modes(bs, cell, comp, Mt, kpts, nb, panel=None):
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho)
    if panel:
        bs.bs_set_option(h, bs.BS_OPT_PANEL, panel)
    bs.bs_set_option(h, bs.BS_OPT_MODES, nb + 2)
    bs.allocate_workspace(h, Mt, len(kpts))
    bs.bs_assemble(h, Mt)
    lam, U, S = bs.bs_modes(h, kpts, nb)
    lam_b = bs.bs_bands(h, kpts, nb)
    bs.bs_destroy_cell(h)
    Phi, Psi = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, Mt)
    _, _, V = oracle.reciprocal_basis(cell.lattice)
    N = (2 * Mt + 1) ** 2
    assert U.shape == (len(kpts), 2 * N, nb) and S.shape == (len(kpts), 3 * N, nb)
    worst = 0.0
    for i, kr in enumerate(kpts):
        K = oracle.pencil_K(Phi, cell.lattice, Mt, kr)
        H = V * oracle.coupling_B(cell.lattice, Mt, kr)
        lr_all, Ur_all = __import__("scipy.linalg", fromlist=["eigh"]).eigh(K, Psi, driver="gv")
        lmax = lr_all[-1]
        # eigenvalues: the same tolerance as bs_bands (reading R8)
        om_g, om_r = np.sqrt(np.maximum(lam[i], 0)), np.sqrt(np.maximum(lr_all[:nb], 0))
        with np.errstate(divide="ignore", invalid="ignore"):
            ok = (np.abs(om_g - om_r) <= 1e-9 * om_r) | (np.abs(lam[i] - lr_all[:nb]) <= 64 * EPS * lmax)
        assert ok.all(), (i, lam[i], lr_all[:nb])
        assert np.max(np.abs(lam[i] - lam_b[i])) <= 64 * EPS * lmax
        Ui, Si = U[i], S[i]
        # K U = Psi U Lambda, norm-wise: the residual of a backward-stable eigensolver is ~ eps ||K|| ||U||
        Rk = K @ Ui - (Psi @ Ui) * lam[i][None, :]
        scale = np.max(np.abs(K)) * np.max(np.abs(Ui))
        assert np.max(np.abs(Rk)) <= 1e-9 * scale, (i, np.max(np.abs(Rk)) / scale)
        worst = max(worst, np.max(np.abs(Rk)) / scale)
        G = Ui.conj().T @ Psi @ Ui
        assert np.max(np.abs(G - np.eye(nb))) <= 1e-9, (i, np.max(np.abs(G - np.eye(nb))))
        # eq. 10: Phi S = H U and H^H S = Psi U Lambda
        HU = H @ Ui
        assert np.max(np.abs(Phi @ Si - HU)) <= 1e-9 * np.max(np.abs(Phi)) * np.max(np.abs(Si))
        assert np.max(np.abs(H.conj().T @ Si - (Psi @ Ui) * lam[i][None, :])) <= 1e-8 * scale
        # projector onto every cluster that lies completely inside the computed branches, against the oracle's
        cl = clusters(lr_all[:nb + 1], lmax)
        for a, b in cl:
            if b > nb:
                continue                                        # the cluster continues beyond the last computed branch
            Pg = Ui[:, a:b] @ Ui[:, a:b].conj().T @ Psi
            Pr = Ur_all[:, a:b] @ Ur_all[:, a:b].conj().T @ Psi
            gap = min(lr_all[a] - lr_all[a - 1] if a > 0 else np.inf, lr_all[b] - lr_all[b - 1] if b < len(lr_all) else np.inf)
            tol = max(1e-10, 2e3 * EPS * lmax / gap)           # perturbation bound eps ||K|| / gap, with room
            assert np.max(np.abs(Pg - Pr)) <= tol * max(1.0, np.max(np.abs(Pr))), (i, a, b, np.max(np.abs(Pg - Pr)), tol)
    return worst


def test_modes_config1_every_kpoint(bs):
    w = wl.get("C1")
    cell = w.cells[0]
    comp = bs.bs_isotropic_plane_strain(cell.E, cell.nu)
    # all 30 k-points of the path: Gamma (two zero modes), X, M (symmetry-degenerate branches) and generic points
    check_modes(bs, cell, comp, w.Mt, w.kpts, 10)


@pytest.mark.parametrize("panel", [8, 16, 32])
def test_modes_every_band_width(bs, panel):
    cell = wl.random_small_cell(31, 3, wl.HEXAGONAL)
    comp = bs.bs_isotropic_plane_strain(cell.E, cell.nu)
    kp = np.array([[0.0, 0.0], [0.5, 0.0], [2.0 / 3.0, 1.0 / 3.0], [0.37, 0.21]])
    check_modes(bs, cell, comp, 4, kp, 12, panel=panel)        # n = 162: several panels at every width


def test_modes_tiny_truncations_and_anisotropic_phases(bs):
    cell = wl.random_small_cell(21, 3, np.array([[1.0, 0.0], [0.3, 0.8]]))
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu).copy()
    comp[:, 3] = 0.01 * comp[:, 0]
    comp[:, 4] = -0.02 * comp[:, 0]
    comp[:, 1] *= 1.1
    for Mt, nb in ((0, 2), (1, 18), (2, 7)):                    # Mt = 0: K is 2 x 2; Mt = 1 with the whole spectrum
        check_modes(bs, cell, comp, Mt, np.array([[0.1, 0.2], [0.5, 0.5]]), nb)


def test_modes_config2_sampled_kpoints(bs):
    # K 450 x 450, stiff disc in a soft matrix: flat localised branches next to steep ones
    w = wl.get("C2")
    cell = w.cells[0]
    comp = bs.bs_isotropic_plane_strain(cell.E, cell.nu)
    check_modes(bs, cell, comp, w.Mt, w.kpts[[0, 1, 20, 40, 59]], w.nbands)


def test_modes_homogeneous_cell_polarisation_on_gpu(bs):
    # physics pin applied directly to the CUDA path: plane waves polarised along / across kappa, Hooke-law stress
    E, nu, rho = 20e9, 0.28, 2500.0
    cell = wl.homogeneous_cell(wl.HEXAGONAL, E, nu, rho, n=2)
    Mt, kred = 2, (0.31, 0.12)
    N = (2 * Mt + 1) ** 2
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, bs.bs_isotropic_plane_strain(cell.E, cell.nu), cell.rho)
    bs.bs_set_option(h, bs.BS_OPT_MODES, 2 * N)
    bs.allocate_workspace(h, Mt, 1)
    bs.bs_assemble(h, Mt)
    lam, U, S = bs.bs_modes(h, [kred], 2 * N)
    bs.bs_destroy_cell(h)
    lam_, mu_ = E * nu / ((1 + nu) * (1 - 2 * nu)), E / (2 * (1 + nu))
    Cst = np.array([[lam_ + 2 * mu_, lam_, 0], [lam_, lam_ + 2 * mu_, 0], [0, 0, mu_]])
    _, Q, _ = oracle.reciprocal_basis(cell.lattice)
    kap = (oracle.plane_wave_indices(Mt) + np.array(kred)) @ Q
    for j in range(2 * N):
        u1, u2 = U[0][:N, j], U[0][N:, j]
        pw = np.abs(u1) ** 2 + np.abs(u2) ** 2
        g = int(np.argmax(pw))
        assert np.delete(pw, g).sum() < 1e-12 * pw[g]
        p = np.array([u1[g], u2[g]])
        khat = kap[g] / np.linalg.norm(kap[g])
        along, across = abs(khat @ p), abs(khat[0] * p[1] - khat[1] * p[0])
        cph = np.sqrt(lam[0, j]) / np.linalg.norm(kap[g])
        if abs(cph - np.sqrt((lam_ + 2 * mu_) / rho)) < 1e-6 * cph:
            assert across < 1e-7 * along
        else:
            assert abs(cph - np.sqrt(mu_ / rho)) < 1e-6 * cph and along < 1e-7 * across
        Bt = np.array([[kap[g][0], 0.0], [0.0, kap[g][1]], [kap[g][1], kap[g][0]]])
        sig = 1j * Cst @ Bt @ p
        got = np.array([S[0][g, j], S[0][N + g, j], S[0][2 * N + g, j]])
        assert np.max(np.abs(got - sig)) < 1e-8 * np.max(np.abs(sig))


def test_refined_frequencies_next_to_gamma_have_singular_value_accuracy(bs):
    """NEXT-4 (R8): next to Gamma the acoustic omega^2 are ~1e-8 .. 1e-12 of lambda_max, so the
    eigenvalues of the assembled pencil lose them in the 9th .. 5th digit (the backward-error clause of R8 is what lets
    bs_bands pass there).  With BS_OPT_REFINE bs_modes returns the factored Rayleigh quotients, which must agree with the
    oracle's singular-value route (omega = sigma(L_Phi^-1 H L_Psi^-dagger)) to <= 1e-9 relative on EVERY branch."""
    cell = wl.get("C1").cells[0]
    Mt, nb = 3, 6
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
    kpts = np.array([[1e-2, 3e-3], [1e-3, 3e-4], [1e-4, 3e-5], [3e-5, -1e-5], [0.31, 0.17]])
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho)
    bs.bs_set_option(h, bs.BS_OPT_MODES, nb)
    bs.allocate_workspace(h, Mt, len(kpts))
    bs.bs_assemble(h, Mt)
    lam_plain = bs.bs_bands(h, kpts, nb)
    bs.bs_set_option(h, bs.BS_OPT_REFINE, 1)
    lam_ref, U, S = bs.bs_modes(h, kpts, nb)
    bs.bs_set_option(h, bs.BS_OPT_REFINE, 0)
    lam_off, _, _ = bs.bs_modes(h, kpts, nb)
    bs.bs_destroy_cell(h)
    # the option off: the eigenvalues of the assembled pencil as bs_bands returns them (bs_modes always takes the two-stage
    # reduction, bs_bands the shared-memory kernel at this size: equal to the backward error of either)
    Phi, Psi = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, Mt)
    worst_plain = 0.0
    for i, kr in enumerate(kpts):
        lmax = oracle.bands_at_k(Phi, Psi, cell.lattice, Mt, kr)[1]
        assert np.max(np.abs(lam_off[i] - lam_plain[i])) <= 64 * EPS * lmax
        om = oracle.omega_svd_route(Phi, Psi, cell.lattice, Mt, kr)[:nb]
        err = np.abs(np.sqrt(lam_ref[i]) - om) / om
        assert np.all(lam_ref[i] > 0) and err.max() <= 1e-9, (i, err)
        worst_plain = max(worst_plain, np.max(np.abs(np.sqrt(np.maximum(lam_plain[i], 0)) - om) / om))
    # the plain route really is not good enough here (otherwise this test shows nothing)
    assert worst_plain > 1e-8


def test_modes_batch_equals_single_handle_calls(bs):
    """bs_modes_batch over three cells with different geometries and lattices of equal area: every matrix is treated as in
    the single-handle call, so eigenvalues, U and S agree bit for bit; with BS_OPT_REFINE the refined frequencies too."""
    Mt, nb = 3, 5
    kpts = np.array([[0.11, 0.07], [0.5, 0.5], [1e-3, 2e-3], [0.3, -0.2]])
    cells = [wl.random_small_cell(31, 3), wl.random_small_cell(32, 4),
             wl.random_small_cell(33, 3, np.array([[1.25, 0.0], [0.3, 0.8]]))]
    def make(c):
        h = bs.bs_create_cell(c.lattice, c.vert_offset, c.verts, oracle.isotropic_plane_strain_compliance(c.E, c.nu), c.rho)
        bs.bs_set_option(h, bs.BS_OPT_MODES, nb)
        bs.bs_set_option(h, bs.BS_OPT_REFINE, 1)
        bs.allocate_workspace(h, Mt, len(kpts))
        return h
    hs = [make(c) for c in cells]
    bs.bs_assemble_batch(hs, Mt)
    lam_b, U_b, S_b = bs.bs_modes_batch(hs, kpts, nb)
    N = (2 * Mt + 1) ** 2
    assert lam_b.shape == (3, len(kpts), nb) and U_b.shape == (3, len(kpts), 2 * N, nb) and S_b.shape == (3, len(kpts), 3 * N, nb)
    for c, h in enumerate(hs):
        lam, U, S = bs.bs_modes(h, kpts, nb)
        assert np.array_equal(lam, lam_b[c]) and np.array_equal(U, U_b[c]) and np.array_equal(S, S_b[c])
        # and they are modes: Phi S = H U to rounding, refined frequencies against the oracle's singular-value route
        cell = cells[c]
        comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
        Phi, Psi = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, Mt)
        _, _, V = oracle.reciprocal_basis(cell.lattice)
        for i, kr in enumerate(kpts):
            H = V * oracle.coupling_B(cell.lattice, Mt, kr)
            assert np.max(np.abs(Phi @ S[i] - H @ U[i])) <= 1e-10 * np.max(np.abs(H @ U[i]))
            om = oracle.omega_svd_route(Phi, Psi, cell.lattice, Mt, kr)[:nb]
            assert np.max(np.abs(np.sqrt(lam[i]) - om) / om) <= 1e-9
    for h in hs:
        bs.bs_destroy_cell(h)


def test_modes_error_paths(bs):
    cell = wl.random_small_cell(1, 2)
    h = bs.bs_create_cell(cell.lattice, cell.vert_offset, cell.verts, bs.bs_isotropic_plane_strain(cell.E, cell.nu), cell.rho)
    bs.allocate_workspace(h, 1, 1)
    bs.bs_assemble(h, 1)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_modes(h, [[0.1, 0.2]], 2)                      # BS_OPT_MODES not set
    assert ei.value.status == bs.BS_ERR_STATE
    bs.bs_set_option(h, bs.BS_OPT_MODES, 4)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_bands(h, [[0.1, 0.2]], 2)                      # the option changes the workspace: assemble again
    assert ei.value.status == bs.BS_ERR_STATE
    bs.allocate_workspace(h, 1, 1)
    bs.bs_assemble(h, 1)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_modes(h, [[0.1, 0.2]], 5)
    assert ei.value.status == bs.BS_ERR_ARG
    lam, U, S = bs.bs_modes(h, [[0.1, 0.2]], 4, stress=False)
    assert S is None and U.shape == (1, 18, 4)
    bs.bs_destroy_cell(h)
