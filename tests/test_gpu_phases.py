"""Phase-level parity (-m gpu): every phase of the 2-stage solver has its own
invariant, checked through the C ABI against the CPU oracle / independent dense algebra."""
import numpy as np
import pytest
import torch

import oracle
from gpu_util import cm, lg, randc
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu
EPS = np.finfo(np.float64).eps


def herm(n, seed):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    return 0.5 * (A + A.conj().T)


def band_to_dense(band, N, b):
    """band: numpy (N, ldab) row-major view of the (ldab x N) column-major band storage."""
    B = np.zeros((N, N), dtype=np.complex128)
    for o in range(min(b, N - 1) + 1):
        idx = np.arange(N - o)
        B[idx + o, idx] = band[idx, o]
    B = B + np.tril(B, -1).conj().T
    return B


def run_reduce(N, A, b=64):
    from paper_2310_03341_b200 import binding
    eng = binding.Eigh(N, band_width=b)
    ldab = 2 * b + 2
    G = A.copy()
    G[np.triu_indices(N, 1)] = np.nan            # only the lower triangle may be read
    At = torch.from_numpy(np.ascontiguousarray(G.T)).cuda()
    band = torch.full((N, ldab), float("nan"), dtype=torch.complex128, device="cuda")
    eng.reduce_to_band(At, band)
    torch.cuda.synchronize()
    return eng, At, band


@pytest.mark.parametrize("N", [65, 130, 300, 517, 1024])
def test_reduce_to_band_preserves_spectrum(N):
    A = herm(N, N)
    eng, At, band = run_reduce(N, A)
    bd = band.cpu().numpy()
    assert np.isfinite(bd).all()
    assert np.abs(bd[:, 65:]).max() == 0.0        # fill-in rows zeroed
    B = band_to_dense(bd, N, 64)
    Wb = oracle.eigh(B, vectors=False)
    Wa = oracle.eigh(A, vectors=False)
    nrm = np.abs(Wa).max()
    assert np.abs(Wb - Wa).max() <= 1e-12 * nrm * max(1, N / 256)
    # trace and Frobenius norm preserved
    assert abs(np.trace(B).real - np.trace(A).real) <= 1e-11 * nrm
    assert abs(np.linalg.norm(B) - np.linalg.norm(A)) <= 1e-12 * np.linalg.norm(A)
    eng.close()


def random_band(N, b, seed):
    rng = np.random.default_rng(seed)
    B = np.zeros((N, N), dtype=np.complex128)
    for o in range(min(b, N - 1) + 1):
        n = N - o
        v = rng.standard_normal(n) + (0 if o == 0 else 1j) * rng.standard_normal(n)
        B[np.arange(n) + o, np.arange(n)] = v
    return B + np.tril(B, -1).conj().T


def dense_to_band(B, N, b, ldab):
    band = np.zeros((N, ldab), dtype=np.complex128)
    for o in range(min(b, N - 1) + 1):
        idx = np.arange(N - o)
        band[idx, o] = B[idx + o, idx]
    return band


@pytest.mark.parametrize("N", [2, 3, 64, 65, 66, 129, 200, 517, 1500])
def test_band_to_tridiag_preserves_spectrum(N):
    from paper_2310_03341_b200 import binding
    b = 64
    B = random_band(N, b, N)
    eng = binding.Eigh(N)
    band = torch.from_numpy(dense_to_band(B, N, b, 2 * b + 2)).cuda()
    d = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
    e = torch.full((max(N - 1, 1),), float("nan"), dtype=torch.float64, device="cuda")
    eng.band_to_tridiag(band, d, e)
    torch.cuda.synchronize()
    dn, en = d.cpu().numpy(), e.cpu().numpy()[: N - 1]
    assert np.isfinite(dn).all() and np.isfinite(en).all() and (en >= 0).all()
    Wt = oracle.tridiag_ql(dn, en, vectors=False)
    Wb = oracle.eigh(B, vectors=False)
    nrm = np.abs(Wb).max()
    assert np.abs(Wt - Wb).max() <= 1e-12 * nrm * max(1, N / 256)
    assert abs(dn.sum() - np.trace(B).real) <= 1e-11 * nrm
    assert abs(np.sum(dn ** 2) + 2 * np.sum(en ** 2) - np.linalg.norm(B) ** 2) <= 1e-11 * np.linalg.norm(B) ** 2
    eng.close()


def run_dc(d, e, nev=None):
    from paper_2310_03341_b200 import binding
    N = len(d)
    nev = N if nev is None else nev
    eng = binding.Eigh(N, nev)
    dd = torch.from_numpy(np.ascontiguousarray(d, dtype=np.float64)).cuda()
    ee = torch.from_numpy(np.ascontiguousarray(e if N > 1 else np.zeros(1), dtype=np.float64)).cuda()
    W = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
    ldq = N + 3
    Qt = torch.full((nev, ldq), float("nan"), dtype=torch.float64, device="cuda")
    nfail = eng.tridiag_dc(dd, ee, W, Qt)
    torch.cuda.synchronize()
    eng.close()
    assert nfail == 0
    return W.cpu().numpy(), Qt.cpu().numpy()[:, :N].T


def check_tridiag(d, e, W, Q, tol_scale=1.0):
    N = len(d)
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    nrm = max(np.abs(W).max(), 1e-300)
    assert np.isfinite(W).all() and np.isfinite(Q).all()
    assert np.all(np.diff(W) >= 0)
    res = np.linalg.norm(T @ Q - Q * W[None, :]) / (max(np.linalg.norm(T), 1e-300) * np.sqrt(N))
    orth = np.abs(Q.T @ Q - np.eye(Q.shape[1])).max()
    assert res <= 1e-14 * tol_scale, res
    assert orth <= 1e-13 * max(1, N / 100) * tol_scale, orth
    Wo = oracle.tridiag_ql(d, e, vectors=False)
    assert np.abs(W - Wo).max() <= 1e-13 * nrm * max(1, N / 100), np.abs(W - Wo).max()


@pytest.mark.parametrize("N", [1, 2, 3, 5, 30, 31, 33, 64, 100, 257, 500, 1000])
def test_dc_toeplitz_121(N):
    d, e = np.full(N, 2.0), np.full(N - 1, -1.0)
    e = np.abs(e)                      # the solver takes e >= 0; spectrum of the 1-2-1 matrix is sign-independent
    W, Q = run_dc(d, e)
    k = np.arange(1, N + 1)
    ref = 2 - 2 * np.cos(k * np.pi / (N + 1))
    assert np.abs(W - ref).max() <= 1e-14 * 4 * max(1, N / 50)
    check_tridiag(d, e, W, Q)


@pytest.mark.parametrize("N", [50, 200, 401])
def test_dc_clement_integer_spectrum(N):
    i = np.arange(1, N)
    d, e = np.zeros(N), np.sqrt(i * (N - i))
    W, Q = run_dc(d, e)
    ref = np.arange(-(N - 1), N, 2).astype(float)
    assert np.abs(W - ref).max() <= 1e-13 * N
    check_tridiag(d, e, W, Q)


def test_dc_wilkinson_and_glued_and_constant():
    m = 100
    d = np.abs(np.arange(-m, m + 1)).astype(float)
    e = np.ones(2 * m)
    W, Q = run_dc(d, e)
    check_tridiag(d, e, W, Q)
    # glued Wilkinson blocks with tiny couplings: clusters of nearly equal eigenvalues
    d = np.tile(np.abs(np.arange(-10, 11)).astype(float), 12)
    e = np.ones(len(d) - 1)
    for c, glue in enumerate([1e-8, 1e-10, 1e-12, 1e-14, 0.0, 1e-6, 1e-9, 1e-11, 1e-13, 1e-15, 1e-7]):
        e[21 * (c + 1) - 1] = glue
    W, Q = run_dc(d, e)
    check_tridiag(d, e, W, Q)
    # total deflation
    d, e = np.full(300, 2.5), np.zeros(299)
    W, Q = run_dc(d, e)
    assert np.array_equal(W, d)
    check_tridiag(d, e, W, Q)


@pytest.mark.parametrize("N,seed", [(777, 1), (2048, 2), (3001, 3)])
def test_dc_random_and_subset(N, seed):
    rng = np.random.default_rng(seed)
    d, e = rng.standard_normal(N), np.abs(rng.standard_normal(N - 1))
    W, Q = run_dc(d, e)
    check_tridiag(d, e, W, Q)
    nev = N // 3
    W2, Q2 = run_dc(d, e, nev=nev)
    assert np.array_equal(W2, W)
    assert Q2.shape == (N, nev)
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    assert np.linalg.norm(T @ Q2 - Q2 * W[None, :nev]) <= 1e-13 * np.linalg.norm(T)


@pytest.mark.parametrize("scale", [2.0 ** -400, 1e-200, 1e-100, 1e-5, 1e5, 1e100, 1e200])
def test_dc_scaled_tridiagonal(scale):
    """eigh_tridiag_dc on s T: eigenvalues s W, the same eigenvectors.  The deflation test of the merge step assumes a
    matrix of norm ~1 (tridiag_dc.cu scales by a power of two first, as xSTEDC does); without it a matrix of norm 1e-100
    deflated completely and came back as its own diagonal.  A power-of-two s must reproduce the unscaled run bit for bit."""
    rng = np.random.default_rng(11)
    N = 500
    d, e = rng.standard_normal(N), np.abs(rng.standard_normal(N - 1))
    W1, Q1 = run_dc(d, e)
    W, Q = run_dc(d * scale, e * scale)
    check_tridiag(d, e, W / scale, Q)
    assert np.abs(W / scale - W1).max() <= 1e-13 * np.abs(W1).max() * 5
    if scale == 2.0 ** -400:
        assert np.array_equal(W / scale, W1) and np.array_equal(Q, Q1)


@pytest.mark.parametrize("nev_of", [lambda N: 1, lambda N: 7, lambda N: N // 2, lambda N: N - 1])
def test_dc_subset_with_deflation_and_ties(nev_of):
    """nev < N shortens the last merge to the wanted secular roots: the subset must equal the leading columns of
    the full solve as a subspace, also when deflated values tie with or interleave the roots (Wilkinson pairs,
    glued blocks, integer Clement spectrum, total deflation)."""
    cases = []
    m = 60
    cases.append((np.abs(np.arange(-m, m + 1)).astype(float), np.ones(2 * m)))
    d = np.tile(np.abs(np.arange(-10, 11)).astype(float), 8)
    e = np.ones(len(d) - 1)
    for c, glue in enumerate([1e-8, 1e-12, 0.0, 1e-6, 1e-14, 1e-10, 1e-15]):
        e[21 * (c + 1) - 1] = glue
    cases.append((d, e))
    i = np.arange(1, 150)
    cases.append((np.zeros(150), np.sqrt(i * (150 - i))))
    cases.append((np.full(130, -1.5), np.zeros(129)))
    for d, e in cases:
        N = len(d)
        nev = max(1, nev_of(N))
        W, Q = run_dc(d, e)
        W2, Q2 = run_dc(d, e, nev=nev)
        assert np.array_equal(W2, W)
        assert Q2.shape == (N, nev) and np.isfinite(Q2).all()
        T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
        assert np.linalg.norm(T @ Q2 - Q2 * W[None, :nev]) <= 1e-13 * max(np.linalg.norm(T), 1.0) * np.sqrt(nev)
        assert np.abs(Q2.T @ Q2 - np.eye(nev)).max() <= 1e-13 * max(1, N / 100)
