"""GPU tests (-m gpu) of the dense building blocks exposed by the C-ABI for diagnostics (bs_zgemm, bs_zpotrf_trtri,
bs_zhetrd, bs_sturm) against NumPy/LAPACK, plus the error paths of the boundary."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bs():
    import torch
    assert torch.cuda.is_available()
    import paper_1310_6380_b200 as bs
    return bs


def to_dev(a):
    """NumPy (rows, cols) complex -> torch CUDA tensor holding the column-major image (shape (cols, rows))."""
    import torch
    return torch.from_numpy(np.ascontiguousarray(a.T)).cuda()


def from_dev(t):
    return t.cpu().numpy().T


def rand_c(rng, m, n):
    return rng.normal(size=(m, n)) + 1j * rng.normal(size=(m, n))


@pytest.mark.parametrize("opA,opB", [(0, 0), (0, 1), (1, 0), (1, 1)])
@pytest.mark.parametrize("M,N,K", [(64, 64, 8), (130, 75, 37), (257, 199, 64), (5, 3, 1)])
def test_zgemm(bs, opA, opB, M, N, K):
    import torch
    rng = np.random.default_rng(M * 1000 + N + K + 7 * opA + 3 * opB)
    A = rand_c(rng, K, M) if opA else rand_c(rng, M, K)
    B = rand_c(rng, N, K) if opB else rand_c(rng, K, N)
    Cm = rand_c(rng, M, N)
    al, be = 0.7 - 0.2j, -0.3 + 1.1j
    ref = al * ((A.conj().T if opA else A) @ (B.conj().T if opB else B)) + be * Cm
    dA, dB, dC = to_dev(A), to_dev(B), to_dev(Cm)
    bs.bs_zgemm(opA, opB, M, N, K, al, dA, A.shape[0], 0, dB, B.shape[0], 0, be, dC, M, 0)
    torch.cuda.synchronize()
    got = from_dev(dC)
    assert np.max(np.abs(got - ref)) <= 1e-13 * K * np.max(np.abs(ref))


@pytest.mark.parametrize("M,N", [(64, 32), (200, 32), (333, 17), (130, 64), (226, 16), (97, 9)])
def test_zgemm_hermitian_lower(bs, M, N):
    # HEMM: only the lower triangle of A is read (the upper one holds garbage), diagonal imaginary parts are ignored
    import torch
    rng = np.random.default_rng(M + N)
    G = rand_c(rng, M, M)
    H = G + G.conj().T
    stored = np.tril(H) + np.triu(rand_c(rng, M, M), 1) + 1j * np.diag(rng.normal(size=M))
    Bm = rand_c(rng, M, N)
    dA, dB = to_dev(stored), to_dev(Bm)
    dC = torch.zeros(N, M, dtype=torch.complex128, device="cuda")
    bs.bs_zgemm(0, 0, M, N, M, 1.0, dA, M, 0, dB, M, 0, 0.0, dC, M, 0, 1, bs.BS_GEMM_A_HERM_LOWER)
    torch.cuda.synchronize()
    Hc = H - 1j * np.diag(np.diag(H).imag)
    ref = Hc @ Bm
    assert np.max(np.abs(from_dev(dC) - ref)) <= 1e-13 * M * np.max(np.abs(ref))


def test_zgemm_batched_lower_only(bs):
    import torch
    rng = np.random.default_rng(5)
    n, k, batch = 150, 40, 3
    A = [rand_c(rng, n, k) for _ in range(batch)]
    C0 = [rand_c(rng, n, n) for _ in range(batch)]
    dA = torch.stack([to_dev(a) for a in A])
    dC = torch.stack([to_dev(c) for c in C0])
    bs.bs_zgemm(0, 1, n, n, k, -1.0, dA, n, n * k, dA, n, n * k, 1.0, dC, n, n * n, batch, bs.BS_GEMM_LOWER_ONLY)
    torch.cuda.synchronize()
    for b in range(batch):
        got = dC[b].cpu().numpy().T
        ref = C0[b] - A[b] @ A[b].conj().T
        lo = np.tril_indices(n)
        up = np.triu_indices(n, 1)
        assert np.max(np.abs(got[lo] - ref[lo])) <= 1e-12 * np.max(np.abs(ref))
        assert np.array_equal(got[up], C0[b][up])      # the strict upper triangle is untouched


def test_zgemm_3m_normwise_bound(bs):
    # The kernel forms Im(ab) as (ar+ai)(br+bi) - ar br - ai bi (three multiplications, include/bs.h): the error of an
    # entry is bounded norm-wise, c u K max|A| max|B|, also where real and imaginary parts differ by many orders of
    # magnitude (there the small part is NOT accurate relative to itself: that is the documented trade).
    import torch
    rng = np.random.default_rng(2024)
    M, N, K = 96, 80, 200
    A = rng.normal(size=(M, K)) + 1e-9j * rng.normal(size=(M, K))     # nearly real
    B = 1e-9 * rng.normal(size=(K, N)) + 1j * rng.normal(size=(K, N))  # nearly imaginary
    ref = A @ B
    dA, dB = to_dev(A), to_dev(B)
    dC = torch.zeros(N, M, dtype=torch.complex128, device="cuda")
    bs.bs_zgemm(0, 0, M, N, K, 1.0, dA, M, 0, dB, K, 0, 0.0, dC, M, 0)
    torch.cuda.synchronize()
    err = np.abs(from_dev(dC) - ref)
    bound = 8 * np.finfo(float).eps * K * np.max(np.abs(A)) * np.max(np.abs(B))
    assert np.max(err) <= bound
    # exact cases: purely real times purely real has a zero imaginary part bit for bit (ai = bi = 0: T3 == T1)
    Ar, Br = rng.normal(size=(M, K)) + 0j, rng.normal(size=(K, N)) + 0j
    dC.zero_()
    bs.bs_zgemm(0, 0, M, N, K, 1.0, to_dev(Ar), M, 0, to_dev(Br), K, 0, 0.0, dC, M, 0)
    torch.cuda.synchronize()
    got = from_dev(dC)
    assert np.all(got.imag == 0.0)
    assert np.max(np.abs(got.real - (Ar.real @ Br.real))) <= 1e-13 * K


@pytest.mark.parametrize("batch", [1, 700])
def test_zgemm_in_place_right_multiply(bs, batch):
    # C == A (the panel solve A21 <- A21 inv(L11)^H of the Cholesky factorisation): a CTA must own complete rows of C.
    # With many matrices in flight a tile that still reads what another tile has overwritten shows up here.
    import torch
    rng = np.random.default_rng(batch)
    M, N = 161, 64
    A = [rand_c(rng, M, N) for _ in range(min(batch, 4))]
    Bm = rand_c(rng, N, N)
    dA = torch.stack([to_dev(A[b % len(A)]) for b in range(batch)])
    dB = to_dev(Bm)
    bs.bs_zgemm(0, 1, M, N, N, 1.0, dA, M, M * N, dB, N, 0, 0.0, dA, M, M * N, batch)
    torch.cuda.synchronize()
    for b in (0, batch // 2, batch - 1):
        ref = A[b % len(A)] @ Bm.conj().T
        got = dA[b].cpu().numpy().T
        assert np.max(np.abs(got - ref)) <= 1e-13 * N * np.max(np.abs(ref))


@pytest.mark.parametrize("n", [17, 64, 100, 363, 450])
def test_zpotrf_trtri(bs, n):
    import torch
    rng = np.random.default_rng(n)
    batch = 2
    mats = []
    for _ in range(batch):
        G = rand_c(rng, n, n)
        mats.append(G @ G.conj().T + n * np.eye(n))
    dA = torch.stack([to_dev(m) for m in mats])
    dX = torch.zeros_like(dA)
    tmp = torch.zeros_like(dA)
    dinv = torch.zeros(batch * ((n + 63) // 64) * 4096, dtype=torch.complex128, device="cuda")
    info = torch.zeros(batch, dtype=torch.int32, device="cuda")
    bs.bs_zpotrf_trtri(n, dA, n, n * n, dX, tmp, dinv, info, batch)
    torch.cuda.synchronize()
    assert info.cpu().numpy().tolist() == [0] * batch
    for b in range(batch):
        L = np.tril(dA[b].cpu().numpy().T)
        Lr = np.linalg.cholesky(mats[b])
        assert np.max(np.abs(L - Lr)) <= 1e-12 * np.max(np.abs(Lr))
        X = dX[b].cpu().numpy().T
        assert np.max(np.abs(np.triu(X, 1))) == 0
        assert np.max(np.abs(X @ Lr - np.eye(n))) <= 1e-11


def test_zpotrf_reports_not_pd(bs):
    import torch
    n = 70
    A = np.eye(n, dtype=complex)
    A[66, 66] = -1.0
    dA = to_dev(A)[None].contiguous()
    dX, tmp = torch.zeros_like(dA), torch.zeros_like(dA)
    dinv = torch.zeros(2 * 4096, dtype=torch.complex128, device="cuda")
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    bs.bs_zpotrf_trtri(n, dA, n, n * n, dX, tmp, dinv, info, 1)
    assert int(info.cpu()[0]) == 67


@pytest.mark.parametrize("algo", [0, 1])
@pytest.mark.parametrize("n,nb", [(1, 8), (2, 8), (5, 4), (9, 8), (64, 8), (98, 32), (242, 32), (242, 16), (450, 16), (130, 32),
                                  (333, 8), (700, 32), (1210, 16), (1217, 16), (1230, 8)])   # n >= 1200, b <= 16: panels in pairs
def test_zhetrd_eigenvalues(bs, n, nb, algo):
    import torch
    rng = np.random.default_rng(n + nb)
    batch = 3
    if algo == 1 and nb % 4:
        pytest.skip("one-stage panel must be a multiple of 4")
    mats = []
    for _ in range(batch):
        G = rand_c(rng, n, n)
        mats.append(G + G.conj().T)
    dA = torch.stack([to_dev(m) for m in mats])
    d = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
    e = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
    scratch = torch.zeros(batch * bs.bs_zhetrd_scratch_elems(n, nb), dtype=torch.complex128, device="cuda")
    bs.bs_zhetrd(n, dA, n, n * n, d, e, scratch, nb, algo, batch)
    torch.cuda.synchronize()
    for b in range(batch):
        dd, ee = d[b].cpu().numpy(), e[b].cpu().numpy()[:n - 1]
        T = np.diag(dd) + np.diag(ee, 1) + np.diag(ee, -1)
        lt = np.linalg.eigvalsh(T)
        la = np.linalg.eigvalsh(mats[b])
        assert np.max(np.abs(lt - la)) <= 1e-13 * n * np.max(np.abs(la))


@pytest.mark.parametrize("scale", [1e-100, 1e100])
@pytest.mark.parametrize("n,nb,algo", [(98, 16, 0), (300, 16, 0), (300, 16, 2), (300, 8, 0), (500, 16, 0)])
def test_zhetrd_scaled_matrices(bs, n, nb, algo, scale):
    """The reflectors of the chase and of the small-matrix kernel take their norm from rsqrt and their reciprocals from
    rcp.approx + Newton steps (chase item (7)): matrices at 1e-100 and 1e100 must give the scaled
    eigenvalues to the usual backward error (squares of the entries stay far inside the exponent range)."""
    import torch
    rng = np.random.default_rng(7 * n + nb)
    G = rand_c(rng, n, n)
    A = G + G.conj().T
    dA = to_dev(A * scale)[None].contiguous()
    d = torch.zeros(1, n, dtype=torch.float64, device="cuda")
    e = torch.zeros(1, n, dtype=torch.float64, device="cuda")
    scratch = torch.zeros(bs.bs_zhetrd_scratch_elems(n, nb), dtype=torch.complex128, device="cuda")
    bs.bs_zhetrd(n, dA, n, n * n, d, e, scratch, nb, algo, 1)
    torch.cuda.synchronize()
    dd, ee = d[0].cpu().numpy() / scale, e[0].cpu().numpy()[:n - 1] / scale
    T = np.diag(dd) + np.diag(ee, 1) + np.diag(ee, -1)
    la = np.linalg.eigvalsh(A)
    assert np.max(np.abs(np.linalg.eigvalsh(T) - la)) <= 1e-13 * n * np.max(np.abs(la))


@pytest.mark.parametrize("n,nb,batch", [(242, 16, 1500), (242, 8, 1500), (338, 16, 900), (242, 32, 600)])
def test_zhetrd_forced_streaming_large_batch(bs, n, nb, batch):
    """BS_TRIDIAG_TWO_STAGE_STREAMED runs stage 2 through the ring of three sweeps with several CTAs per SM (the I/O
    warps of different CTAs then drift against the compute warps: the setting in which the write-back / fetch race of
    the streamed kernel showed as run-to-run different results).  Must be reproducible bit for bit, give the same bits
    for equal matrices anywhere in the batch, agree with the resident-band kernel to rounding, and have the eigenvalues of
    the dense matrix."""
    import torch
    rng = np.random.default_rng(11 * n + nb)
    base = []
    for _ in range(4):
        G = rand_c(rng, n, n)
        base.append(to_dev(G + G.conj().T))
    A = torch.stack([base[i % 4] for i in range(batch)]).contiguous()
    res = {}
    for key, algo in [("resident", 0), ("streamed", 2), ("streamed again", 2)]:
        dA = A.clone()
        d = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
        e = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
        scratch = torch.zeros(batch * bs.bs_zhetrd_scratch_elems(n, nb), dtype=torch.complex128, device="cuda")
        bs.bs_zhetrd(n, dA, n, n * n, d, e, scratch, nb, algo, batch)
        torch.cuda.synchronize()
        res[key] = (d.cpu().numpy(), e.cpu().numpy())
    dd, ee = res["streamed"]
    assert np.array_equal(dd, res["streamed again"][0]) and np.array_equal(ee, res["streamed again"][1])
    for j in range(4):
        assert np.array_equal(dd[j::4], np.broadcast_to(dd[j], dd[j::4].shape))
        assert np.array_equal(ee[j::4], np.broadcast_to(ee[j], ee[j::4].shape))
    scale = np.max(np.abs(res["resident"][0]))
    assert np.max(np.abs(dd - res["resident"][0])) <= 1e-12 * scale
    assert np.max(np.abs(np.abs(ee) - np.abs(res["resident"][1]))) <= 1e-12 * scale
    T = np.diag(dd[5]) + np.diag(ee[5][:n - 1], 1) + np.diag(ee[5][:n - 1], -1)
    la = np.linalg.eigvalsh(from_dev(base[1]))
    assert np.max(np.abs(np.linalg.eigvalsh(T) - la)) <= 1e-13 * n * np.max(np.abs(la))


@pytest.mark.parametrize("n,nb,batch", [(450, 16, 320), (820, 8, 200), (400, 32, 320)])
def test_zhetrd_streamed_band_large_batch_is_reproducible(bs, n, nb, batch):
    """Band streamed through the shared-memory ring (n too large for a resident band of this width) with more matrices
    than SMs: the I/O warps of the chasing kernel write columns back and fetch new ones into the same ring slots, so a
    missing ordering shows as run-to-run differences.  Two runs must agree bitwise, every matrix of the batch (the same
    matrix repeated) must give the same d, e bitwise, and the eigenvalues must be those of the dense matrix."""
    import torch
    rng = np.random.default_rng(7 * n + nb)
    G = rand_c(rng, n, n)
    A = G + G.conj().T
    dA0 = to_dev(A)
    out = []
    for _ in range(2):
        dA = dA0.unsqueeze(0).repeat(batch, 1, 1).contiguous()
        d = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
        e = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
        scratch = torch.zeros(batch * bs.bs_zhetrd_scratch_elems(n, nb), dtype=torch.complex128, device="cuda")
        bs.bs_zhetrd(n, dA, n, n * n, d, e, scratch, nb, 0, batch)
        torch.cuda.synchronize()
        out.append((d.cpu().numpy(), e.cpu().numpy()))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    dd, ee = out[0]
    assert np.array_equal(dd, np.broadcast_to(dd[0], dd.shape)) and np.array_equal(ee, np.broadcast_to(ee[0], ee.shape))
    T = np.diag(dd[0]) + np.diag(ee[0][:n - 1], 1) + np.diag(ee[0][:n - 1], -1)
    la = np.linalg.eigvalsh(A)
    assert np.max(np.abs(np.linalg.eigvalsh(T) - la)) <= 1e-13 * n * np.max(np.abs(la))


def test_sturm_constant_tridiagonal_textbook(bs):
    # constant-coefficient tridiagonal: eigenvalues d + 2 e cos(j pi/(n+1)), j = 1..n
    import torch
    n, dd, ee = 333, 1.5, -0.75
    d = torch.full((1, n), dd, dtype=torch.float64, device="cuda")
    e = torch.full((1, n), ee, dtype=torch.float64, device="cuda")
    nev = 40
    lam = torch.zeros(1, nev, dtype=torch.float64, device="cuda")
    bs.bs_sturm(n, d, e, nev, lam, 1)
    ref = np.sort(dd + 2 * ee * np.cos(np.arange(1, n + 1) * np.pi / (n + 1)))[:nev]
    assert np.max(np.abs(lam.cpu().numpy()[0] - ref)) <= 1e-14 * 3.0


def test_sturm_random_and_degenerate(bs):
    import torch
    rng = np.random.default_rng(3)
    n, batch, nev = 257, 4, 257
    dn = rng.normal(size=(batch, n))
    en = rng.normal(size=(batch, n))
    en[1, 100] = 0.0              # a split matrix
    dn[2, :] = 2.0; en[2, :] = 0.0    # diagonal with a fully repeated eigenvalue
    d, e = torch.from_numpy(dn).cuda(), torch.from_numpy(en).cuda()
    lam = torch.zeros(batch, nev, dtype=torch.float64, device="cuda")
    bs.bs_sturm(n, d, e, nev, lam, batch)
    got = lam.cpu().numpy()
    for b in range(batch):
        T = np.diag(dn[b]) + np.diag(en[b, :n - 1], 1) + np.diag(en[b, :n - 1], -1)
        ref = np.linalg.eigvalsh(T)
        assert np.max(np.abs(got[b] - ref)) <= 1e-14 * n * max(1.0, np.max(np.abs(ref)))


@pytest.mark.parametrize("scale", [1e-60, 1.0, 1e12, 1e60])
@pytest.mark.parametrize("n", [5, 98, 1023, 1922])
def test_sturm_scaled_matrices(bs, n, scale):
    """The Sturm recurrence is renormalised by an exact power of two every fourth step (S7): matrices
    whose entries sit at 1e-60 .. 1e60 make the unscaled pair grow or shrink by hundreds of orders of magnitude over n steps
    (lengths with every remainder modulo four).  The eigenvalues must scale with the matrix, to rounding."""
    import torch
    rng = np.random.default_rng(n)
    dn = rng.normal(size=(2, n)) * scale
    en = rng.normal(size=(2, n)) * scale
    dn[1] = np.abs(dn[1]) + 3.0 * scale   # second matrix: diagonally dominant, positive definite
    nev = min(n, 18)
    d, e = torch.from_numpy(dn).cuda(), torch.from_numpy(en).cuda()
    lam = torch.zeros(2, nev, dtype=torch.float64, device="cuda")
    bs.bs_sturm(n, d, e, nev, lam, 2)
    got = lam.cpu().numpy()
    for b in range(2):
        T = np.diag(dn[b] / scale) + np.diag(en[b, :n - 1] / scale, 1) + np.diag(en[b, :n - 1] / scale, -1)
        ref = np.linalg.eigvalsh(T)
        assert np.max(np.abs(got[b] / scale - ref[:nev])) <= 1e-14 * n * max(1.0, np.max(np.abs(ref)))


def test_error_paths(bs):
    c = wl.random_small_cell(1, 2)
    comp = bs.bs_isotropic_plane_strain(c.E, c.nu)
    # clockwise polygon
    v = c.verts.copy()
    v[:4] = v[:4][::-1]
    with pytest.raises(bs.BsError) as ei:
        bs.bs_create_cell(c.lattice, c.vert_offset, v, comp, c.rho)
    assert ei.value.status == bs.BS_ERR_GEOMETRY
    # tiling does not cover the cell
    with pytest.raises(bs.BsError) as ei:
        bs.bs_create_cell(2.0 * c.lattice, c.vert_offset, c.verts, comp, c.rho)
    assert ei.value.status == bs.BS_ERR_GEOMETRY
    with pytest.raises(bs.BsError) as ei:
        bs.bs_isotropic_plane_strain([1.0], [0.5])
    assert ei.value.status == bs.BS_ERR_ARG
    h = bs.bs_create_cell(c.lattice, c.vert_offset, c.verts, comp, c.rho)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_assemble(h, 2)                      # no workspace
    assert ei.value.status == bs.BS_ERR_NOMEM
    bs.allocate_workspace(h, 2, 2)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_bands(h, [[0.1, 0.2]], 4)           # not assembled
    assert ei.value.status == bs.BS_ERR_STATE
    bs.bs_assemble(h, 2)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_bands(h, [[0.1, 0.2]], 51)          # nbands > 2N = 50
    assert ei.value.status == bs.BS_ERR_ARG
    with pytest.raises(bs.BsError) as ei:
        bs.bs_bands(h, np.zeros((3, 2)), 4)       # workspace sized for 2 k-points
    assert ei.value.status == bs.BS_ERR_NOMEM
    # negative density contrast making R indefinite -> NOT_PD is reported, not a crash
    rho = c.rho.copy()
    h2 = bs.bs_create_cell(c.lattice, c.vert_offset, c.verts, -comp, rho)
    bs.allocate_workspace(h2, 1, 1)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_assemble(h2, 1)
    assert ei.value.status == bs.BS_ERR_NOT_PD
    bs.bs_destroy_cell(h)
    bs.bs_destroy_cell(h2)


@pytest.mark.parametrize("mode", [0, 1])
def test_batch_rejects_unequal_cell_areas_and_bad_output_buffers(bs, mode):
    # one V^2 scales every K(k) of a launch: a batch of cells with different lattice areas must be refused BEFORE any
    # launch, in both pencil modes (it used to return eigenvalues off by (V_c / V_lead)^2 in DIRECT mode)
    import torch
    a = wl.random_small_cell(3, 2)
    b = wl.random_small_cell(4, 2, 1.5 * wl.SQUARE)
    hs = []
    for c in (a, b):
        h = bs.bs_create_cell(c.lattice, c.vert_offset, c.verts, bs.bs_isotropic_plane_strain(c.E, c.nu), c.rho)
        bs.bs_set_option(h, bs.BS_OPT_PENCIL_MODE, mode)
        bs.allocate_workspace(h, 2, 2)
        hs.append(h)
    with pytest.raises(bs.BsError) as ei:
        bs.bs_assemble_batch(hs, 2)
    assert ei.value.status == bs.BS_ERR_ARG and "area" in str(ei.value)
    for h in hs:
        bs.bs_assemble(h, 2)                       # each alone is fine
    with pytest.raises(bs.BsError) as ei:
        bs.bs_bands_batch(hs, [[0.1, 0.2]], 4)
    assert ei.value.status == bs.BS_ERR_ARG
    # mismatching options across a batch
    bs.bs_set_option(hs[1], bs.BS_OPT_OUTPUT, bs.BS_OUTPUT_OMEGA)
    with pytest.raises(bs.BsError):
        bs.bs_bands_batch([hs[0], hs[0]][:1] + [hs[1]], [[0.1, 0.2]], 4)
    # result buffers of the wrong dtype / size / layout never reach the library
    for bad in (np.empty((1, 4), dtype=np.float32), np.empty((1, 3)), np.empty((4, 2)).T[:1],
                torch.empty(1, 4, dtype=torch.float32, device="cuda"), torch.empty(1, 5, dtype=torch.float64, device="cuda")):
        with pytest.raises(bs.BsError) as ei:
            bs.bs_bands(hs[0], [[0.1, 0.2]], 4, out=bad)
        assert ei.value.status == bs.BS_ERR_ARG
    lam = bs.bs_bands(hs[0], [[0.1, 0.2]], 4)
    d, e = bs.bs_get_tridiagonal(hs[0])
    assert d.shape == (1, 2 * hs[0].N)
    with pytest.raises(bs.BsError):
        bs.bs_get_tridiagonal(hs[0], 7)
    for h in hs:
        bs.bs_destroy_cell(h)


@pytest.mark.parametrize("batch", [3, 1500])
@pytest.mark.parametrize("n,nb", [(200, 8), (242, 16), (338, 16), (300, 32), (450, 32)])
def test_chase_is_bitwise_independent_of_the_number_of_overlapped_sweeps(bs, n, nb, batch):
    """Stage 2 streamed with G = 1 (sweeps strictly one after the other: the algorithm as defined), 2, 3, 4, 5 sweeps per
    train (test knob in bits 8.. of `algo`), several CTAs per SM and several CTAs per matrix following one another through
    L2, and the resident-band pipeline: all must give the same d, e BIT FOR BIT, for every matrix of the batch."""
    import torch
    rng = np.random.default_rng(3 * n + nb)
    base = []
    for _ in range(3):
        G = rand_c(rng, n, n)
        base.append(to_dev(G + G.conj().T))
    A = torch.stack([base[i % 3] for i in range(batch)]).contiguous()
    ref = None
    for algo in [2 | (1 << 8), 2 | (2 << 8), 2 | (3 << 8), 2 | (4 << 8), 2 | (5 << 8), 2, 0]:
        dA = A.clone()
        d = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
        e = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
        scratch = torch.zeros(batch * bs.bs_zhetrd_scratch_elems(n, nb), dtype=torch.complex128, device="cuda")
        bs.bs_zhetrd(n, dA, n, n * n, d, e, scratch, nb, algo, batch)
        torch.cuda.synchronize()
        got = (d.cpu().numpy(), e.cpu().numpy())
        if ref is None:
            ref = got
            for j in range(3):
                assert np.array_equal(got[0][j::3], np.broadcast_to(got[0][j], got[0][j::3].shape))
            T = np.diag(got[0][1]) + np.diag(got[1][1][:n - 1], 1) + np.diag(got[1][1][:n - 1], -1)
            la = np.linalg.eigvalsh(from_dev(base[1]))
            assert np.max(np.abs(np.linalg.eigvalsh(T) - la)) <= 1e-13 * n * np.max(np.abs(la))
        else:
            assert np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1]), hex(algo)
