"""Plain, slow, float64/complex128 NumPy + LAPACK oracle of the hot path.

TEST INFRASTRUCTURE (see ``oracle/__init__.py``).  Every function cites the passage of
``PAPER.md`` (arXiv:1310.6380) or the reading in ``DESIGN.md`` (section "Readings") it follows.
Parity status: every function here is pinned by ``tests/test_oracle_pins.py`` against
something other than itself (closed forms, brute-force quadrature, analytic dispersion,
the paper's printed stop-bands); nothing is "parity unpinned".

Conventions (DESIGN.md "Readings" R1-R9):
  * lattice rows are h^1, h^2 ([A]_{jk} = h^j . e^k); T = A^{-1};
    q^j = 2 pi * (column j of T) so that q^i . h^j = 2 pi delta_ij.
  * plane wave g <-> (a1, a2), a1 slow: g = (a1+Mt)(2Mt+1) + (a2+Mt)  (PAPER.md:150, 0-based).
  * matrix entry (row alpha = test function, column beta = trial function) uses
    q = G_beta - G_alpha  (north_star; the paper's eq. 19/20 index the transpose).
  * compliance per phase: [D1111, D2222, D1122, D1112, D2212, D1212].
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla


# --------------------------------------------------------------------------- bases
def reciprocal_basis(lattice):
    """PAPER.md:23-26 (eq. 1) and :138.  Returns (T, Q, V): T = A^{-1}, rows of Q are q^1, q^2
    (q^i . h^j = 2 pi delta_ij), V = |det A| the cell area."""
    A = np.asarray(lattice, dtype=np.float64).reshape(2, 2)
    T = np.linalg.inv(A)
    Q = 2.0 * np.pi * T.T            # row i = q^i = 2 pi * column i of T
    V = abs(float(np.linalg.det(A)))
    return T, Q, V


def plane_wave_indices(Mt):
    """PAPER.md:127 (eq. 15), :150.  (N,2) integer array of (a1, a2), a1 slow, N=(2Mt+1)^2."""
    r = np.arange(-Mt, Mt + 1)
    a1, a2 = np.meshgrid(r, r, indexing="ij")
    return np.stack([a1.ravel(), a2.ravel()], axis=1)


# --------------------------------------------------------------------------- shape integral
def polygon_area(poly):
    """Shoelace area of a simple polygon (positive when counter-clockwise)."""
    p = np.asarray(poly, dtype=np.float64)
    x, y = p[:, 0], p[:, 1]
    return 0.5 * float(np.sum(x * np.roll(y, -1) - np.roll(x, -1) * y))


def _j0(t):
    """sin(t)/t with j0(0)=1.  (sin(t)/t is accurate to two roundings for every t != 0; no series branch.)"""
    t = np.asarray(t, dtype=np.float64)
    zero = t == 0.0
    safe = np.where(zero, 1.0, t)
    return np.where(zero, 1.0, np.sin(safe) / safe)


def shape_integral(poly, q):
    """I_p(q) = int_{Omega_p} exp(i q.x) dx for a simple CCW polygon (north_star; replaces the
    centroid rule of PAPER.md:106 eq. 12 / :213 eq. 22).  Divergence theorem on
    div(q e^{iq.x}) = i|q|^2 e^{iq.x}; each edge integral is |e| e^{iq.m} j0(q.e/2):

        I_p(q) = (-i/|q|^2) sum_j (q_x e_{j,y} - q_y e_{j,x}) e^{i q.m_j} j0(q.e_j/2),   I_p(0)=area.
    """
    p = np.asarray(poly, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    q2 = float(q @ q)
    if q2 == 0.0:
        return complex(polygon_area(p))
    nxt = np.roll(p, -1, axis=0)
    e = nxt - p
    m = 0.5 * (nxt + p)
    cross = q[0] * e[:, 1] - q[1] * e[:, 0]
    s = np.sum(cross * np.exp(1j * (m @ q)) * _j0(0.5 * (e @ q)))
    return complex(-1j * s / q2)


def polygon_centroid(poly):
    """Area centroid of a simple polygon (textbook shoelace form)."""
    p = np.asarray(poly, dtype=np.float64)
    x, y = p[:, 0], p[:, 1]
    xn, yn = np.roll(x, -1), np.roll(y, -1)
    cr = x * yn - xn * y
    A = 0.5 * np.sum(cr)
    return np.array([np.sum((x + xn) * cr), np.sum((y + yn) * cr)]) / (6.0 * A)


def shape_integral_centroid(poly, q):
    """PAPER.md:106 (eq. 12) / :213 (eq. 22): the paper's one-point rule int_{Omega_p} F ~ F(c_p) V_p with
    F = exp(i q.x): I_p(q) ~ A_p exp(i q.c_p).  (The leading term of ``shape_integral``; reading R6.)"""
    q = np.asarray(q, dtype=np.float64)
    return complex(polygon_area(poly) * np.exp(1j * (polygon_centroid(poly) @ q)))


# --------------------------------------------------------------------------- property fields
def isotropic_plane_strain_compliance(E, nu):
    """PAPER.md:121 (eq. 14): D_jkmn = (1/2mu)[ (d_jm d_kn + d_jn d_km)/2 - lam/(2(mu+lam)) d_jk d_mn ].
    Returns (P,6): D1111 D2222 D1122 D1112 D2212 D1212."""
    E = np.atleast_1d(np.asarray(E, dtype=np.float64))
    nu = np.atleast_1d(np.asarray(nu, dtype=np.float64))
    lam = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu))
    mu = E / (2.0 * (1.0 + nu))
    return _compliance_from_lame(lam, mu)


def _compliance_from_lame(lam, mu):
    c = lam / (2.0 * (mu + lam))
    D1111 = (1.0 - c) / (2.0 * mu)
    D1122 = -c / (2.0 * mu)
    D1212 = 0.5 / (2.0 * mu)
    z = np.zeros_like(mu)
    return np.stack([D1111, D1111.copy(), D1122, z, z.copy(), D1212], axis=1)


def lame_from_C11_C44(C11, C44):
    """lambda + 2 mu = C11, mu = C44."""
    return C11 - 2.0 * C44, C44


def voigt_compliance(compliance):
    """PAPER.md:167-171 (eq. 20): 3x3 block weights with the printed factors 1/2/4.
    Returns (P,3,3): [[D1111, D1122, 2 D1112],[D1122, D2222, 2 D2212],[2 D1112, 2 D2212, 4 D1212]]."""
    c = np.asarray(compliance, dtype=np.float64).reshape(-1, 6)
    D = np.empty((c.shape[0], 3, 3))
    D[:, 0, 0] = c[:, 0]
    D[:, 1, 1] = c[:, 1]
    D[:, 0, 1] = D[:, 1, 0] = c[:, 2]
    D[:, 0, 2] = D[:, 2, 0] = 2.0 * c[:, 3]
    D[:, 1, 2] = D[:, 2, 1] = 2.0 * c[:, 4]
    D[:, 2, 2] = 4.0 * c[:, 5]
    return D


# --------------------------------------------------------------------------- matrices
def assemble_direct(lattice, vert_offset, verts, compliance, density, Mt):
    """THE DEFINITION (eq. 19-20 with the exact integral, reading R4):
    for every pair (alpha, beta):  Phi[(a,alpha),(b,beta)] = sum_p Dv[p,a,b] I_p(G_beta - G_alpha),
    R[alpha,beta] = sum_p rho_p I_p(G_beta - G_alpha), Psi = diag(R, R).  O(N^2 P): small cases only."""
    _, Q, _ = reciprocal_basis(lattice)
    idx = plane_wave_indices(Mt)
    N = idx.shape[0]
    G = idx @ Q
    Dv = voigt_compliance(compliance)
    rho = np.asarray(density, dtype=np.float64)
    P = rho.shape[0]
    verts = np.asarray(verts, dtype=np.float64).reshape(-1, 2)
    polys = [verts[vert_offset[p]:vert_offset[p + 1]] for p in range(P)]
    Phi = np.zeros((3 * N, 3 * N), dtype=np.complex128)
    R = np.zeros((N, N), dtype=np.complex128)
    for al in range(N):
        for be in range(N):
            q = G[be] - G[al]
            I = np.array([shape_integral(polys[p], q) for p in range(P)])
            R[al, be] = np.sum(rho * I)
            for a in range(3):
                for b in range(3):
                    Phi[a * N + al, b * N + be] = np.sum(Dv[:, a, b] * I)
    Psi = np.zeros((2 * N, 2 * N), dtype=np.complex128)
    Psi[:N, :N] = R
    Psi[N:, N:] = R
    return Phi, Psi


def shape_integral_table(lattice, vert_offset, verts, weights, Mt, quadrature="exact"):
    """T_c(D) = sum_p weights[c,p] I_p(D1 q^1 + D2 q^2) for every index difference
    D in [-2Mt,2Mt]^2 (reading R1: G_beta - G_alpha depends only on beta - alpha, so the
    N^2 entries of a block take (4Mt+1)^2 distinct values).  Vectorised over edges; the
    formula is ``shape_integral``'s, pinned to it and to ``assemble_direct`` in the tests.
    ``quadrature="centroid"`` uses the paper's one-point rule per polygon (``shape_integral_centroid``) instead.
    Returns complex (C, 4Mt+1, 4Mt+1), index [c, D1+2Mt, D2+2Mt]."""
    _, Q, _ = reciprocal_basis(lattice)
    verts = np.asarray(verts, dtype=np.float64).reshape(-1, 2)
    off = np.asarray(vert_offset)
    P = off.shape[0] - 1
    w = np.asarray(weights, dtype=np.float64).reshape(-1, P)
    # per-edge arrays
    start = verts
    nxt = np.empty_like(verts)
    phase_of_edge = np.empty(verts.shape[0], dtype=np.int64)
    area = np.empty(P)
    for p in range(P):
        s, t = off[p], off[p + 1]
        nxt[s:t] = np.roll(verts[s:t], -1, axis=0)
        phase_of_edge[s:t] = p
        area[p] = polygon_area(verts[s:t])
    if quadrature == "centroid":
        cent = np.array([polygon_centroid(verts[off[p]:off[p + 1]]) for p in range(P)])
    elif quadrature != "exact":
        raise ValueError(quadrature)
    e = nxt - start
    m = 0.5 * (nxt + start)
    we = w[:, phase_of_edge]                       # (C, nedge)
    L = 4 * Mt + 1
    out = np.zeros((w.shape[0], L, L), dtype=np.complex128)
    for i1, D1 in enumerate(range(-2 * Mt, 2 * Mt + 1)):
        for i2, D2 in enumerate(range(-2 * Mt, 2 * Mt + 1)):
            if D1 == 0 and D2 == 0:
                out[:, i1, i2] = w @ area
                continue
            q = D1 * Q[0] + D2 * Q[1]
            if quadrature == "centroid":
                out[:, i1, i2] = w @ (area * np.exp(1j * (cent @ q)))
                continue
            q2 = float(q @ q)
            cross = q[0] * e[:, 1] - q[1] * e[:, 0]
            term = cross * np.exp(1j * (m @ q)) * _j0(0.5 * (e @ q))
            out[:, i1, i2] = (-1j / q2) * (we @ term)
    return out


def assemble(lattice, vert_offset, verts, compliance, density, Mt, quadrature="exact"):
    """Phi (3N x 3N) and Psi (2N x 2N) through the index-difference table (same numbers as
    ``assemble_direct`` up to rounding; that equality is a test).  PAPER.md:150-171."""
    Dv = voigt_compliance(compliance)
    rho = np.asarray(density, dtype=np.float64)
    # channels: 6 distinct entries of the symmetric 3x3 weight block, then rho
    pairs = [(0, 0), (1, 1), (0, 1), (0, 2), (1, 2), (2, 2)]
    W = np.stack([Dv[:, a, b] for a, b in pairs] + [rho], axis=0)
    tab = shape_integral_table(lattice, vert_offset, verts, W, Mt, quadrature)
    idx = plane_wave_indices(Mt)
    N = idx.shape[0]
    d1 = idx[None, :, 0] - idx[:, None, 0] + 2 * Mt       # [alpha, beta] -> beta - alpha
    d2 = idx[None, :, 1] - idx[:, None, 1] + 2 * Mt
    blk = {pr: tab[c][d1, d2] for c, pr in enumerate(pairs)}
    Phi = np.zeros((3 * N, 3 * N), dtype=np.complex128)
    for a in range(3):
        for b in range(3):
            Phi[a * N:(a + 1) * N, b * N:(b + 1) * N] = blk[(min(a, b), max(a, b))]
    R = tab[6][d1, d2]
    Psi = np.zeros((2 * N, 2 * N), dtype=np.complex128)
    Psi[:N, :N] = R
    Psi[N:, N:] = R
    return Phi, Psi


def coupling_B(lattice, Mt, kred):
    """PAPER.md:157-160 (eq. 18) with int_Omega f = V delta (reading R3): B(k), 3N x 2N, N x N
    diagonal blocks  B[(1,g),(1,g)] = i kx_g, B[(2,g),(2,g)] = i ky_g, B[(3,g),(1,g)] = i ky_g,
    B[(3,g),(2,g)] = i kx_g  with kappa_g = k + G_g, k = Q1 q^1 + Q2 q^2.
    H(k) = V * B(k)."""
    _, Q, _ = reciprocal_basis(lattice)
    idx = plane_wave_indices(Mt)
    N = idx.shape[0]
    kap = (idx + np.asarray(kred, dtype=np.float64)[None, :]) @ Q     # (N,2) Cartesian k + G
    B = np.zeros((3 * N, 2 * N), dtype=np.complex128)
    g = np.arange(N)
    B[g, g] = 1j * kap[:, 0]
    B[N + g, N + g] = 1j * kap[:, 1]
    B[2 * N + g, g] = 1j * kap[:, 1]
    B[2 * N + g, N + g] = 1j * kap[:, 0]
    return B


def pencil_K(Phi, lattice, Mt, kred):
    """K(k) = H^dagger Phi^{-1} H (eq. 10-11; reading R5), by a solve, symmetrised."""
    _, _, V = reciprocal_basis(lattice)
    H = V * coupling_B(lattice, Mt, kred)
    K = H.conj().T @ np.linalg.solve(Phi, H)
    return 0.5 * (K + K.conj().T)


def bands_at_k(Phi, Psi, lattice, Mt, kred, nbands=None):
    """All (or the lowest nbands) eigenvalues lambda = omega^2 of K U = lambda Psi U, ascending
    (LAPACK zhegv).  Also returns lambda_max (needed by the backward-error clause, reading R8)."""
    K = pencil_K(Phi, lattice, Mt, kred)
    lam = sla.eigh(K, Psi, eigvals_only=True, driver="gv")
    lam_max = float(lam[-1])
    return (lam if nbands is None else lam[:nbands]), lam_max


def modes_at_k(Phi, Psi, lattice, Mt, kred, nbands):
    """Mode shapes of the lowest nbands branches at one k-point ("the eigenvectors U give the displacement
    mode shapes and S = -Phi^-1 H* U the stress mode shapes").  In the notation used here the paper's
    H* is -H with H = V B(k) (reading R3), so  S = Phi^-1 H U  and eq. 10 reads  Phi S = H U,
    H^dagger S = lambda Psi U.  zhegv with vectors: the columns of U are Psi-orthonormal, U^dagger Psi U = I.
    Returns (lam (nbands,), U (2N, nbands), S (3N, nbands))."""
    _, _, V = reciprocal_basis(lattice)
    H = V * coupling_B(lattice, Mt, kred)
    K = pencil_K(Phi, lattice, Mt, kred)
    lam, U = sla.eigh(K, Psi, driver="gv")
    U = U[:, :nbands]
    S = np.linalg.solve(Phi, H @ U)
    return lam[:nbands], U, S


def band_structure(lattice, vert_offset, verts, compliance, density, Mt, kpts, nbands):
    """Whole path: assemble once, then lambda[k, band] for every reduced k-point.  Returns
    (lam (nk,nbands), lam_max (nk,))."""
    Phi, Psi = assemble(lattice, vert_offset, verts, compliance, density, Mt)
    kpts = np.asarray(kpts, dtype=np.float64).reshape(-1, 2)
    lam = np.zeros((kpts.shape[0], nbands))
    lmax = np.zeros(kpts.shape[0])
    for i, kr in enumerate(kpts):
        lam[i], lmax[i] = bands_at_k(Phi, Psi, lattice, Mt, kr, nbands)
    return lam, lmax


def omega_svd_route(Phi, Psi, lattice, Mt, kred):
    """Secondary, more accurate route for small omega (reading R8): W = L_Phi^{-1} H L_Psi^{-dagger};
    the singular values of W, ascending, are omega directly (A = W^dagger W)."""
    _, _, V = reciprocal_basis(lattice)
    H = V * coupling_B(lattice, Mt, kred)
    Lp = np.linalg.cholesky(Phi)
    Ls = np.linalg.cholesky(Psi)
    X = sla.solve_triangular(Lp, H, lower=True)
    W = sla.solve_triangular(Ls, X.conj().T, lower=True).conj().T
    s = np.linalg.svd(W, compute_uv=False)
    return np.sort(s)
