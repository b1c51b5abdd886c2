"""GPU test (-m gpu) of bs_zhetrd_static, the allocation-free variant of bs_zhetrd whose scratch lives in a static device
array of BS_ZHETRD_STATIC_BYTES inside the library (include/bs.h).  Collected last on purpose (file name): the suite
runs with pytest -x.  The expected values come from the existing path (bs_zhetrd with caller-provided scratch, band width
16) and from LAPACK on the dense matrix; consecutive calls of different shapes share the array and must not see each
other's leftovers."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bs():
    import torch
    assert torch.cuda.is_available()
    import paper_1310_6380_b200 as bs
    return bs


def hermitian_batch(seed, n, batch):
    """Seeded random Hermitian matrices; returns the NumPy matrices and the column-major CUDA image (batch, n, n)."""
    import torch
    rng = np.random.default_rng(seed)
    mats = []
    for _ in range(batch):
        G = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
        mats.append(G + G.conj().T)
    dev = torch.stack([torch.from_numpy(np.ascontiguousarray(m.T)).cuda() for m in mats]).contiguous()
    return mats, dev


def existing_path(bs, dA, n, batch):
    import torch
    d = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
    e = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
    scratch = torch.zeros(batch * bs.bs_zhetrd_scratch_elems(n, 16), dtype=torch.complex128, device="cuda")
    bs.bs_zhetrd(n, dA.clone(), n, n * n, d, e, scratch, 16, 0, batch)
    torch.cuda.synchronize()
    return d.cpu().numpy(), e.cpu().numpy()


def static_path(bs, dA, n, batch):
    import torch
    d = torch.full((batch, n), np.nan, dtype=torch.float64, device="cuda")
    e = torch.full((batch, n), np.nan, dtype=torch.float64, device="cuda")
    bs.bs_zhetrd_static(n, dA.clone(), n, n * n, d, e, batch)   # enqueues only: no allocation, no synchronisation
    torch.cuda.synchronize()
    return d.cpu().numpy(), e.cpu().numpy()


def check(mats, n, got, ref):
    dd, ee = got
    scale = np.max(np.abs(ref[0]))
    # same tolerance as tests/test_gpu_blocks.py uses between two routes to the same tridiagonal matrix
    assert np.max(np.abs(dd - ref[0])) <= 1e-12 * scale
    assert np.max(np.abs(np.abs(ee[:, :n - 1]) - np.abs(ref[1][:, :n - 1]))) <= 1e-12 * scale
    for b, A in enumerate(mats):
        T = np.diag(dd[b]) + np.diag(ee[b][:n - 1], 1) + np.diag(ee[b][:n - 1], -1)
        la = np.linalg.eigvalsh(A)
        assert np.max(np.abs(np.linalg.eigvalsh(T) - la)) <= 1e-13 * n * np.max(np.abs(la))


def test_static_scratch_matches_existing_path_on_calls_in_a_row(bs):
    # three calls in a row on the shared array: a streamed band (n = 450), a band resident in shared memory with more
    # matrices (n = 242: different layout of the array, the progress words land where reflectors were), and the first
    # shape again with new matrices
    calls = [(450, 3, 101), (242, 5, 202), (450, 3, 303)]
    prepared = []
    for n, batch, seed in calls:
        mats, dA = hermitian_batch(seed, n, batch)
        prepared.append((n, batch, mats, dA, existing_path(bs, dA, n, batch)))
    for n, batch, mats, dA, ref in prepared:
        assert bs.bs_zhetrd_static_bytes(n, batch) <= bs.binding.BS_ZHETRD_STATIC_BYTES
        check(mats, n, static_path(bs, dA, n, batch), ref)


def test_static_scratch_same_input_twice_gives_the_same_bits(bs):
    n, batch = 338, 4
    mats, dA = hermitian_batch(7, n, batch)
    first = static_path(bs, dA, n, batch)
    second = static_path(bs, dA, n, batch)
    assert np.array_equal(first[0], second[0]) and np.array_equal(first[1][:, :n - 1], second[1][:, :n - 1])
    check(mats, n, second, existing_path(bs, dA, n, batch))


def test_static_scratch_small_and_largest_single_matrix(bs):
    for n, seed in [(98, 5), (1217, 6)]:   # shared-memory kernel (no scratch); paired panels of stage 1
        mats, dA = hermitian_batch(seed, n, 1)
        check(mats, n, static_path(bs, dA, n, 1), existing_path(bs, dA, n, 1))
    assert bs.bs_zhetrd_static_bytes(2048, 1) <= bs.binding.BS_ZHETRD_STATIC_BYTES


def test_static_scratch_rejects_sizes_beyond_the_array(bs):
    import torch
    n, batch = 450, 7
    assert bs.bs_zhetrd_static_bytes(n, batch) > bs.binding.BS_ZHETRD_STATIC_BYTES
    dA = torch.zeros(batch, n, n, dtype=torch.complex128, device="cuda")
    d = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
    e = torch.zeros(batch, n, dtype=torch.float64, device="cuda")
    with pytest.raises(bs.binding.BsError, match="static array holds"):
        bs.bs_zhetrd_static(n, dA, n, n * n, d, e, batch)
    with pytest.raises(bs.binding.BsError):
        bs.bs_zhetrd_static(2049, dA, 2049, 0, d, e, 1)
