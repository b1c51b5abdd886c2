"""Pins of the CPU oracle against things other than itself (CPU only; `-m "not gpu"`).

Each test names the plausible mistake it would catch.
"""
import os

import numpy as np
import pytest

import oracle
import workloads as wl
from closed_forms import ANISO_FIELDS, christoffel_frequencies, compliance_tensor, voigt_from_tensor

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
HEX = wl.HEXAGONAL


# ----------------------------------------------------------------------------- shape integral
def _rect_closed_form(x0, y0, w, h, q):
    """Textbook: int over a rectangle of e^{iq.x} = w h e^{iq.c} sinc(qx w/2) sinc(qy h/2)."""
    c = np.array([x0 + w / 2, y0 + h / 2])
    return w * h * np.exp(1j * (q @ c)) * np.sinc(q[0] * w / 2 / np.pi) * np.sinc(q[1] * h / 2 / np.pi)


@pytest.mark.parametrize("q", [(3.1, -2.2), (0.0, 5.0), (7.0, 0.0), (1e-3, 2e-3), (40.0, 33.0)])
def test_shape_integral_rectangle_closed_form(q):
    # catches: wrong sign of i, dropped 1/|q|^2, wrong edge normal, j0 at 0 (q parallel to an edge)
    q = np.array(q)
    x0, y0, w, h = 0.2, -0.1, 0.7, 0.45
    rect = np.array([[x0, y0], [x0 + w, y0], [x0 + w, y0 + h], [x0, y0 + h]])
    ref = _rect_closed_form(x0, y0, w, h, q)
    got = oracle.shape_integral(rect, q)
    assert abs(got - ref) <= 1e-13 * max(abs(ref), w * h * 1e-3)


def test_shape_integral_square_equals_two_triangles():
    # north_star pin: a square phase split into two triangles gives the identical integral
    sq = np.array([[0.1, 0.2], [0.6, 0.2], [0.6, 0.7], [0.1, 0.7]])
    t1, t2 = sq[[0, 1, 2]], sq[[0, 2, 3]]
    for q in [(2.0, 3.0), (-12.5, 4.0), (0.0, 9.0), (25.1, -25.1)]:
        q = np.array(q)
        a = oracle.shape_integral(sq, q)
        b = oracle.shape_integral(t1, q) + oracle.shape_integral(t2, q)
        assert abs(a - b) < 1e-15


def _brute_quadrature(poly, q, n=1200):
    """Midpoint rule on an n x n grid over the bounding box with an even-odd inside test."""
    from matplotlib.path import Path  # pragma: no cover
    raise RuntimeError


def _inside(poly, X, Y):
    inside = np.zeros(X.shape, dtype=bool)
    m = len(poly)
    for i in range(m):
        x1, y1 = poly[i]
        x2, y2 = poly[(i + 1) % m]
        cond = (y1 > Y) != (y2 > Y)
        with np.errstate(divide="ignore", invalid="ignore"):
            xin = (x2 - x1) * (Y - y1) / (y2 - y1) + x1
        inside ^= cond & (X < xin)
    return inside


@pytest.mark.parametrize("poly", [
    np.array([[0.0, 0.0], [0.5, 0.05], [0.3, 0.45]]),                                   # triangle
    np.array([[0.0, 0.0], [0.6, 0.0], [0.6, 0.5], [0.3, 0.2], [0.0, 0.5]]),            # non-convex
])
def test_shape_integral_brute_force_quadrature(poly):
    # north_star pin: brute-force quadrature of I_p on tiny polygons (O(h^2) midpoint rule)
    n = 1500
    lo, hi = poly.min(0), poly.max(0)
    xs = lo[0] + (np.arange(n) + 0.5) * (hi[0] - lo[0]) / n
    ys = lo[1] + (np.arange(n) + 0.5) * (hi[1] - lo[1]) / n
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    mask = _inside(poly, X, Y)
    dA = (hi[0] - lo[0]) * (hi[1] - lo[1]) / n ** 2
    for q in [(4.0, -7.0), (15.0, 11.0), (0.0, 0.0)]:
        q = np.array(q)
        ref = np.sum(np.exp(1j * (q[0] * X + q[1] * Y))[mask]) * dA
        got = oracle.shape_integral(poly, q)
        assert abs(got - ref) < 2e-4 * oracle.polygon_area(poly) + 1e-6


def test_shape_integral_symmetries():
    rng = np.random.default_rng(1)
    poly = np.array([[0.0, 0.0], [1.0, 0.1], [1.2, 0.9], [0.4, 1.3], [-0.2, 0.6]])
    assert oracle.shape_integral(poly, np.zeros(2)) == pytest.approx(oracle.polygon_area(poly))
    for _ in range(5):
        q = rng.normal(size=2) * 10
        t = rng.normal(size=2)
        I = oracle.shape_integral(poly, q)
        assert abs(oracle.shape_integral(poly, -q) - np.conj(I)) < 1e-15        # I(-q) = conj I(q)
        It = oracle.shape_integral(poly + t, q)
        assert abs(It - np.exp(1j * (q @ t)) * I) < 1e-13                        # translation
    # small-q limit -> area (continuity: a wrong j0 Taylor or a 1/|q|^2 slip breaks it)
    I = oracle.shape_integral(poly, np.array([1e-5, -2e-5]))
    assert abs(I - oracle.polygon_area(poly)) < 1e-4


def test_tiling_identity_hex_mesh():
    # sum_p I_p(G) = V delta_{G,0} for every reciprocal-lattice vector when the polygons tile the cell
    cell = wl.get("C3").cells[0]
    _, Q, V = oracle.reciprocal_basis(cell.lattice)
    ones = np.ones((1, cell.nphase))
    tab = oracle.shape_integral_table(cell.lattice, cell.vert_offset, cell.verts, ones, 2)
    L = tab.shape[1]
    expect = np.zeros((L, L), dtype=complex)
    expect[L // 2, L // 2] = V
    assert np.max(np.abs(tab[0] - expect)) < 5e-15


def test_reciprocal_basis_definition():
    # q^i . h^j = 2 pi delta_ij; catches the T vs T^T slip of eq. 16 vs eq. 23
    for A in [wl.SQUARE, HEX, np.array([[1.3, 0.2], [-0.4, 0.9]])]:
        T, Q, V = oracle.reciprocal_basis(A)
        assert np.allclose(Q @ A.T, 2 * np.pi * np.eye(2), atol=1e-14)
        assert V == pytest.approx(abs(np.linalg.det(A)))


# ----------------------------------------------------------------------------- compliance
def test_compliance_is_inverse_of_plane_strain_stiffness():
    # textbook: Voigt plane-strain stiffness [[l+2m, l, 0],[l, l+2m, 0],[0,0,m]] (engineering shear)
    E, nu = 70e9, 0.33
    lam = E * nu / ((1 + nu) * (1 - 2 * nu))
    mu = E / (2 * (1 + nu))
    C = np.array([[lam + 2 * mu, lam, 0], [lam, lam + 2 * mu, 0], [0, 0, mu]])
    Dv = oracle.voigt_compliance(oracle.isotropic_plane_strain_compliance(E, nu))[0]
    assert np.allclose(Dv, np.linalg.inv(C), rtol=1e-13, atol=0)
    # closed forms of SURVEY 8c-3
    assert Dv[0, 0] == pytest.approx((1 - nu ** 2) / E, rel=1e-13)
    assert Dv[0, 1] == pytest.approx(-nu * (1 + nu) / E, rel=1e-13)
    assert Dv[2, 2] == pytest.approx(2 * (1 + nu) / E, rel=1e-13)


# ----------------------------------------------------------------------------- matrices
def _small_cell(seed=3, n=3, lattice=wl.SQUARE):
    c = wl.random_small_cell(seed, n, lattice)
    comp = oracle.isotropic_plane_strain_compliance(c.E, c.nu)
    return c, comp


def test_table_assembly_equals_direct_definition():
    # the index-difference table against the N^2 P definition, including a skew lattice
    for lattice in (wl.SQUARE, np.array([[1.0, 0.0], [0.3, 0.8]])):
        c, comp = _small_cell(lattice=lattice)
        comp = comp.copy()
        comp[:, 3] = 0.01 * comp[:, 0]        # make it anisotropic so every block is exercised
        comp[:, 4] = -0.02 * comp[:, 0]
        comp[:, 1] *= 1.1
        Pd, Sd = oracle.assemble_direct(c.lattice, c.vert_offset, c.verts, comp, c.rho, 1)
        Pt, St = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, 1)
        assert np.max(np.abs(Pd - Pt)) <= 1e-14 * np.max(np.abs(Pd))
        assert np.max(np.abs(Sd - St)) <= 1e-14 * np.max(np.abs(Sd))


def test_matrices_hermitian_positive_definite_and_block_structure():
    c, comp = _small_cell(seed=5, n=4)
    Mt = 2
    N = (2 * Mt + 1) ** 2
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    assert Phi.shape == (3 * N, 3 * N) and Psi.shape == (2 * N, 2 * N)
    assert np.max(np.abs(Phi - Phi.conj().T)) <= 1e-15 * np.max(np.abs(Phi))
    assert np.max(np.abs(Psi - Psi.conj().T)) <= 1e-15 * np.max(np.abs(Psi))
    np.linalg.cholesky(Phi)
    np.linalg.cholesky(Psi)
    b = lambda i, j: Phi[i * N:(i + 1) * N, j * N:(j + 1) * N]
    # isotropic plane strain: (1,3),(2,3) vanish, (1,1)=(2,2), (3,3)=2[(1,1)-(1,2)]
    assert np.max(np.abs(b(0, 2))) == 0 and np.max(np.abs(b(1, 2))) == 0
    assert np.array_equal(b(0, 0), b(1, 1))
    assert np.allclose(b(2, 2), 2 * (b(0, 0) - b(0, 1)), rtol=0, atol=1e-14 * np.max(np.abs(Phi)))
    # Omega has only the (1,1),(2,2) blocks, equal
    assert np.array_equal(Psi[:N, :N], Psi[N:, N:]) and np.max(np.abs(Psi[:N, N:])) == 0
    # Toeplitz in the index difference
    idx = oracle.plane_wave_indices(Mt)
    R = Psi[:N, :N]
    seen = {}
    for a in range(N):
        for bb in range(N):
            key = tuple(idx[bb] - idx[a])
            seen.setdefault(key, R[a, bb])
            assert R[a, bb] == seen[key]


def test_homogeneous_cell_gives_scaled_identity():
    E, nu, rho = 10e9, 0.3, 2000.0
    c = wl.homogeneous_cell(HEX, E, nu, rho, n=3)
    comp = oracle.isotropic_plane_strain_compliance(c.E, c.nu)
    Mt = 2
    N = (2 * Mt + 1) ** 2
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    V = abs(np.linalg.det(HEX))
    Dv = oracle.voigt_compliance(comp)[0]
    assert np.max(np.abs(Phi - V * np.kron(Dv, np.eye(N)))) < 1e-14 * np.max(np.abs(Phi))
    assert np.max(np.abs(Psi - rho * V * np.eye(2 * N))) < 1e-14 * rho * V


def test_refinement_invariance():
    # splitting every pixel into two triangles with the same properties leaves the matrices unchanged
    c, comp = _small_cell(seed=9, n=3)
    polys, E, nu, rho = [], [], [], []
    for p in range(c.nphase):
        sq = c.polygon(p)
        for tri in (sq[[0, 1, 2]], sq[[0, 2, 3]]):
            polys.append(tri)
            E.append(c.E[p]); nu.append(c.nu[p]); rho.append(c.rho[p])
    off, verts = wl._csr(polys)
    comp2 = oracle.isotropic_plane_strain_compliance(np.array(E), np.array(nu))
    P1, S1 = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, 2)
    P2, S2 = oracle.assemble(c.lattice, off, verts, comp2, np.array(rho), 2)
    assert np.max(np.abs(P1 - P2)) < 1e-14 * np.max(np.abs(P1))
    assert np.max(np.abs(S1 - S2)) < 1e-14 * np.max(np.abs(S1))


def test_coupling_structure():
    # [H]* = -[H]^T in the paper's convention <=> B is purely imaginary with the printed pattern
    Mt = 1
    N = 9
    B = oracle.coupling_B(HEX, Mt, (0.2, 0.1))
    assert B.shape == (3 * N, 2 * N)
    assert np.max(np.abs(B.real)) == 0
    assert np.array_equal(B[2 * N:, :N], B[N:2 * N, N:]) and np.array_equal(B[2 * N:, N:], B[:N, :N])
    assert np.count_nonzero(B) <= 4 * N
    _, Q, _ = oracle.reciprocal_basis(HEX)
    g = 5                                                # (a1,a2) = (0,1)
    kap = (np.array([0, 1]) + np.array([0.2, 0.1])) @ Q
    assert B[g, g] == pytest.approx(1j * kap[0]) and B[N + g, N + g] == pytest.approx(1j * kap[1])


# ----------------------------------------------------------------------------- pencil
@pytest.mark.parametrize("lattice", [wl.SQUARE, HEX])
def test_homogeneous_dispersion_is_analytic(lattice):
    # north_star pin: omega = c |k+G| for a homogeneous isotropic cell, c_L^2=(l+2m)/rho, c_T^2=m/rho
    E, nu, rho = 20e9, 0.28, 2500.0
    c = wl.homogeneous_cell(lattice, E, nu, rho, n=2)
    comp = oracle.isotropic_plane_strain_compliance(c.E, c.nu)
    Mt = 3
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    lam_, mu_ = E * nu / ((1 + nu) * (1 - 2 * nu)), E / (2 * (1 + nu))
    cL, cT = np.sqrt((lam_ + 2 * mu_) / rho), np.sqrt(mu_ / rho)
    _, Q, _ = oracle.reciprocal_basis(lattice)
    for kred in [(0.31, 0.12), (0.5, 0.0), (0.05, 0.45)]:
        lam, _ = oracle.bands_at_k(Phi, Psi, lattice, Mt, kred)
        kap = np.linalg.norm((oracle.plane_wave_indices(Mt) + np.array(kred)) @ Q, axis=1)
        ref = np.sort(np.concatenate([cL * kap, cT * kap]))
        assert np.max(np.abs(np.sqrt(np.maximum(lam, 0)) - ref) / ref) < 5e-12


def test_homogeneous_anisotropic_dispersion_pins_eq20_shear_coupling_factors():
    # PAPER.md:167-171 (eq. 20): the factors 2 on D1112, D2212 and 4 on D1212.  A homogeneous ANISOTROPIC cell (all six
    # compliance fields non-zero, D1112 != D2212) has omega^2 = eig(Bt(kappa)^T C Bt(kappa)) / rho with C the inverse of
    # the engineering-shear Voigt compliance, which tests/closed_forms.py derives from the 4-index tensor by applying
    # eps = D : sigma to unit stresses (no call into the oracle).  A factor 1 (or 4) on the 13/23 entries, a swapped
    # D1112 <-> D2212, or a 2 instead of 4 on D1212 fails this test.
    rho, Mt = 3100.0, 2
    c = wl.homogeneous_cell(HEX, 1.0, 0.3, rho, n=2)
    comp = np.tile(ANISO_FIELDS, (c.nphase, 1))
    S = voigt_from_tensor(compliance_tensor(ANISO_FIELDS))
    assert np.all(np.linalg.eigvalsh(S) > 0) and abs(S[0, 2]) > 0 and abs(S[0, 2]) != abs(S[1, 2])
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    _, Q, _ = oracle.reciprocal_basis(HEX)
    for kred in [(0.31, 0.12), (0.5, 0.0), (-0.2, 0.45)]:
        lam, _ = oracle.bands_at_k(Phi, Psi, HEX, Mt, kred)
        kap = (oracle.plane_wave_indices(Mt) + np.array(kred)) @ Q
        ref = np.sort(christoffel_frequencies(ANISO_FIELDS, rho, kap).ravel())
        assert np.max(np.abs(np.sqrt(np.maximum(lam, 0)) - ref) / ref) < 1e-11
    # the same closed form separates the readings: the spectrum with factor 1 on the shear-coupling entries is far away
    wrong = ANISO_FIELDS.copy()
    wrong[3:5] *= 0.5
    kap = (oracle.plane_wave_indices(Mt) + np.array((0.31, 0.12))) @ Q
    a = np.sort(christoffel_frequencies(ANISO_FIELDS, rho, kap).ravel())
    b = np.sort(christoffel_frequencies(wrong, rho, kap).ravel())
    assert np.max(np.abs(a - b) / a) > 1e-3


def test_j0_has_no_inaccurate_branch():
    # sin(t)/t is accurate for every t != 0 (one rounding each for sin, the division): compare with the alternating
    # series summed in extended precision at small arguments, where a wrong Taylor coefficient would show at 1e-9
    from fractions import Fraction
    for t in [3e-5, 9.9e-5, 1.0001e-4, 1e-3, 1e-8, 1e-160]:
        ft, term, s = Fraction(t), Fraction(1), Fraction(0)
        for k in range(12):
            s += term
            term = -term * ft * ft / ((2 * k + 2) * (2 * k + 3))
        assert abs(float(oracle.bandstructure._j0(t)) - float(s)) <= 2.3e-16
    assert float(oracle.bandstructure._j0(0.0)) == 1.0


def test_two_zero_modes_at_gamma_and_translation_invariance():
    c, comp = _small_cell(seed=11, n=3, lattice=HEX)
    Mt = 2
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    lam, lmax = oracle.bands_at_k(Phi, Psi, c.lattice, Mt, (0.0, 0.0))
    assert np.all(np.abs(lam[:2]) < 64 * 2.0 ** -53 * lmax) and lam[2] > 1e-6 * lmax
    # shifting every polygon by t leaves omega unchanged
    t = np.array([0.137, -0.29])
    Phi2, Psi2 = oracle.assemble(c.lattice, c.vert_offset, c.verts + t, comp, c.rho, Mt)
    for kred in [(0.3, 0.1), (0.5, 0.5)]:
        l1, _ = oracle.bands_at_k(Phi, Psi, c.lattice, Mt, kred, 8)
        l2, _ = oracle.bands_at_k(Phi2, Psi2, c.lattice, Mt, kred, 8)
        assert np.max(np.abs(l1 - l2) / l1) < 1e-10


def test_svd_route_agrees_with_zhegv():
    c, comp = _small_cell(seed=13, n=4)
    Mt = 2
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    kred = (0.23, 0.4)
    lam, _ = oracle.bands_at_k(Phi, Psi, c.lattice, Mt, kred)
    om = oracle.omega_svd_route(Phi, Psi, c.lattice, Mt, kred)
    assert np.max(np.abs(np.sqrt(lam) - om) / om) < 1e-10


# ----------------------------------------------------------------------------- the paper's numbers
def _circle_overlay_cell(a, d, nseg):
    """Steel cylinder (regular nseg-gon of equal AREA to the disc) in epoxy, hexagonal lattice.
    The matrix phase is realised as the whole parallelogram with epoxy properties plus the
    polygon carrying the property CONTRAST (integrals are linear in the property fields)."""
    lattice = a * HEX
    centre = 0.5 * (lattice[0] + lattice[1])
    r = d / 2
    r_eq = r * np.sqrt(2 * np.pi / (nseg * np.sin(2 * np.pi / nseg)))
    th = 2 * np.pi * np.arange(nseg) / nseg
    circ = centre + r_eq * np.stack([np.cos(th), np.sin(th)], axis=1)
    par = np.array([[0, 0], lattice[0], lattice[0] + lattice[1], lattice[1]], dtype=float)
    return lattice, wl._csr([par, circ])


def test_paper_stopbands_steel_epoxy_hexagonal():
    # stop-bands 120-262 kHz and 427-473 kHz at M=5, first 12 branches.
    gold = np.loadtxt(os.path.join(GOLDEN, "paper_stopbands.txt"))
    a, d = 6.023e-3, 4e-3
    lattice, (off, verts) = _circle_overlay_cell(a, d, 512)
    lam_s, mu_s = oracle.lame_from_C11_C44(264e9, 81e9)
    lam_e, mu_e = oracle.lame_from_C11_C44(7.54e9, 1.48e9)
    from oracle.bandstructure import _compliance_from_lame
    Ds = _compliance_from_lame(np.array([lam_s]), np.array([mu_s]))[0]
    De = _compliance_from_lame(np.array([lam_e]), np.array([mu_e]))[0]
    comp = np.stack([De, Ds - De])
    rho = np.array([1142.0, 7780.0 - 1142.0])
    kp = wl.kpath(lattice, wl.HEX_PATH, 31)
    lam, _ = oracle.band_structure(lattice, off, verts, comp, rho, 5, kp, 12)
    f = np.sqrt(np.maximum(lam, 0)) / (2 * np.pi) / 1e3            # kHz
    gaps = []
    for b in range(11):
        lo, hi = f[:, b].max(), f[:, b + 1].min()
        if hi - lo > 5.0:
            gaps.append((lo, hi))
    assert len(gaps) == 2, gaps
    for (lo, hi), (glo, ghi) in zip(gaps, gold):
        assert abs(lo - glo) < 0.02 * glo and abs(hi - ghi) < 0.02 * ghi, (gaps, gold)


# ----------------------------------------------------------------------------- centroid rule (eq. 12)
def test_centroid_rule_is_the_leading_term_and_converges():
    # textbook centroids; I(0) = area; |I_exact - A e^{iq.c}| = O(|q|^2 h^2) A: refining a pixel grid by 2 cuts the
    # error of the assembled table by ~4 (second order), and it tends to the exact table
    assert np.allclose(oracle.polygon_centroid(np.array([[0, 0], [3, 0], [0, 3.0]])), [1, 1])
    assert np.allclose(oracle.polygon_centroid(np.array([[1, 1], [3, 1], [3, 2], [1, 2.0]])), [2, 1.5])
    poly = np.array([[0.1, 0.2], [0.5, 0.25], [0.3, 0.6]])
    assert oracle.shape_integral_centroid(poly, np.zeros(2)) == pytest.approx(oracle.polygon_area(poly))
    for scale in (1.0, 0.5):
        q = np.array([3.0, -2.0])
        small = poly * scale
        err = abs(oracle.shape_integral(small, q) - oracle.shape_integral_centroid(small, q)) / oracle.polygon_area(small)
        assert err < 0.2 * (np.linalg.norm(q) * scale * 0.5) ** 2
    errs = []
    for n in (8, 16, 32):
        rho = np.array([1000.0 + 500.0 * ((i * 7 + j * 3) % 5) for i in range(4) for j in range(4)])
        # the same 4x4 property field carried by n x n pixels
        polys = wl.pixel_polygons(n)
        w = np.array([[rho[(i * 4 // n) * 4 + (j * 4 // n)] for i in range(n) for j in range(n)]])
        off, verts = wl._csr(polys)
        ex = oracle.shape_integral_table(wl.SQUARE, off, verts, w, 1)
        ce = oracle.shape_integral_table(wl.SQUARE, off, verts, w, 1, quadrature="centroid")
        errs.append(np.max(np.abs(ex - ce)) / np.max(np.abs(ex)))
    assert errs[0] > errs[1] > errs[2] and errs[2] < 2e-2
    assert 3.5 < errs[0] / errs[1] < 4.6 and 3.8 < errs[1] / errs[2] < 4.2


# ----------------------------------------------------------------------------- mode shapes (NEXT-1)
def test_modes_homogeneous_cell_are_polarised_plane_waves_with_hooke_stress():
    # PAPER.md:104.  Homogeneous isotropic cell: every eigenvector is one plane wave exp(i kappa.x) polarised along kappa
    # (longitudinal, omega = c_L |kappa|) or across it (transverse, c_T |kappa|); its stress coefficients obey Hooke's law
    # sigma = C eps with eps = i Bt(kappa) p (textbook), i.e. S = i C Bt p on that plane wave.  Catches: a transposed or
    # conjugated U, the sign of S (the paper's H* is minus this H), a missing factor V, a stress ordering mistake.
    E, nu, rho = 20e9, 0.28, 2500.0
    c = wl.homogeneous_cell(HEX, E, nu, rho, n=2)
    comp = oracle.isotropic_plane_strain_compliance(c.E, c.nu)
    Mt = 2
    N = (2 * Mt + 1) ** 2
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    lam_, mu_ = E * nu / ((1 + nu) * (1 - 2 * nu)), E / (2 * (1 + nu))
    Cst = np.array([[lam_ + 2 * mu_, lam_, 0], [lam_, lam_ + 2 * mu_, 0], [0, 0, mu_]])   # textbook plane-strain stiffness
    _, Q, V = oracle.reciprocal_basis(HEX)
    kred = (0.31, 0.12)                                  # generic point: all 2N eigenvalues distinct
    kap = (oracle.plane_wave_indices(Mt) + np.array(kred)) @ Q
    lam, U, S = oracle.modes_at_k(Phi, Psi, HEX, Mt, kred, 2 * N)
    assert np.allclose(U.conj().T @ Psi @ U, np.eye(2 * N), atol=1e-10)
    seen = set()
    for j in range(2 * N):
        u1, u2 = U[:N, j], U[N:, j]
        g = int(np.argmax(np.abs(u1) ** 2 + np.abs(u2) ** 2))
        rest = np.delete(np.abs(u1) ** 2 + np.abs(u2) ** 2, g).sum()
        assert rest < 1e-16 * (abs(u1[g]) ** 2 + abs(u2[g]) ** 2)            # a single plane wave
        p = np.array([u1[g], u2[g]])
        khat = kap[g] / np.linalg.norm(kap[g])
        along, across = abs(khat @ p), abs(khat[0] * p[1] - khat[1] * p[0])
        cph = np.sqrt(lam[j]) / np.linalg.norm(kap[g])
        if abs(cph - np.sqrt((lam_ + 2 * mu_) / rho)) < 1e-6 * cph:
            assert across < 1e-9 * along                                       # longitudinal: polarised along kappa
            seen.add((g, "L"))
        else:
            assert abs(cph - np.sqrt(mu_ / rho)) < 1e-6 * cph and along < 1e-9 * across
            seen.add((g, "T"))
        Bt = np.array([[kap[g][0], 0.0], [0.0, kap[g][1]], [kap[g][1], kap[g][0]]])
        sig = 1j * Cst @ Bt @ p                                                # Hooke: sigma = C (i Bt p)
        got = np.array([S[g, j], S[N + g, j], S[2 * N + g, j]])
        assert np.max(np.abs(got - sig)) < 1e-9 * np.max(np.abs(sig))
        others = np.delete(np.abs(S[:, j]), [g, N + g, 2 * N + g])
        assert others.max() < 1e-9 * np.max(np.abs(sig))
    assert len(seen) == 2 * N                                                  # every plane wave once per polarisation


def test_modes_satisfy_the_mixed_system_of_eq10():
    # PAPER.md:94-97 (eq. 10) on a heterogeneous skew cell:  Phi S = H U  and  H^dagger S = lambda Psi U
    c, comp = _small_cell(seed=17, n=3, lattice=np.array([[1.0, 0.0], [0.3, 0.8]]))
    Mt = 2
    Phi, Psi = oracle.assemble(c.lattice, c.vert_offset, c.verts, comp, c.rho, Mt)
    _, _, V = oracle.reciprocal_basis(c.lattice)
    kred = (0.2, -0.35)
    lam, U, S = oracle.modes_at_k(Phi, Psi, c.lattice, Mt, kred, 9)
    H = V * oracle.coupling_B(c.lattice, Mt, kred)
    assert np.max(np.abs(Phi @ S - H @ U)) < 1e-10 * np.max(np.abs(H @ U))
    assert np.max(np.abs(H.conj().T @ S - (Psi @ U) * lam[None, :])) < 1e-9 * np.max(np.abs(H.conj().T @ S))
    lam2, _ = oracle.bands_at_k(Phi, Psi, c.lattice, Mt, kred, 9)
    assert np.allclose(lam, lam2, rtol=1e-12)
