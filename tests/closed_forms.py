"""Closed forms from textbook elasticity used as pins by both the oracle tests and the GPU tests.

Nothing here calls ``oracle`` or the CUDA package: these are the independent right-hand sides.
"""
import numpy as np

# a fully populated, positive definite plane compliance tensor (1/Pa): D1111 D2222 D1122 D1112 D2212 D1212,
# D1112 != D2212 so that a swapped or mis-scaled shear-coupling entry changes the spectrum
ANISO_FIELDS = np.array([5.0e-11, 8.0e-11, -1.5e-11, 0.6e-11, -0.9e-11, 4.0e-11])


def compliance_tensor(fields):
    """The 2x2x2x2 tensor D_jkmn with minor (jk, mn) and major (jk <-> mn) symmetries from its 6 independent entries."""
    D1111, D2222, D1122, D1112, D2212, D1212 = fields
    D = np.zeros((2, 2, 2, 2))
    D[0, 0, 0, 0] = D1111
    D[1, 1, 1, 1] = D2222
    D[0, 0, 1, 1] = D[1, 1, 0, 0] = D1122
    for (j, k) in [(0, 1), (1, 0)]:
        D[0, 0, j, k] = D[j, k, 0, 0] = D1112
        D[1, 1, j, k] = D[j, k, 1, 1] = D2212
        for (m, n) in [(0, 1), (1, 0)]:
            D[j, k, m, n] = D1212
    return D


def voigt_from_tensor(D):
    """Engineering-strain Voigt matrix S with (e11, e22, gamma12 = 2 e12) = S (s11, s22, s12), obtained by applying
    eps_jk = D_jkmn sigma_mn to the three unit Voigt stresses (s12 = 1 means sigma_12 = sigma_21 = 1)."""
    S = np.zeros((3, 3))
    unit = [np.array([[1.0, 0], [0, 0]]), np.array([[0, 0], [0, 1.0]]), np.array([[0, 1.0], [1.0, 0]])]
    for J, sig in enumerate(unit):
        eps = np.einsum("jkmn,mn->jk", D, sig)
        S[:, J] = [eps[0, 0], eps[1, 1], 2.0 * eps[0, 1]]
    return S


def christoffel_frequencies(fields, rho, kappa):
    """omega of the two plane-wave modes of a homogeneous anisotropic medium at each wave vector kappa (n,2):
    rho omega^2 u = Gamma(kappa) u,  Gamma = Bt^T C Bt,  C = S^{-1},  Bt = [[kx,0],[0,ky],[ky,kx]] (strain = Bt u).
    Returns (n,2), each row ascending."""
    C = np.linalg.inv(voigt_from_tensor(compliance_tensor(fields)))
    out = np.zeros((len(kappa), 2))
    for i, (kx, ky) in enumerate(kappa):
        Bt = np.array([[kx, 0.0], [0.0, ky], [ky, kx]])
        out[i] = np.sqrt(np.linalg.eigvalsh(Bt.T @ C @ Bt) / rho)
    return out
