"""End-to-end parity (-m gpu): eigh_solve through the C ABI vs the CPU oracle on the same seeded
inputs.  Tolerances are north_star's: |lambda - lambda_ref| <= 1e-11 ||H||_2;
||HZ - Z Lambda||_F / (||H||_F sqrt N) <= 1e-13;  ||Z^H Z - I||_max <= 1e-12 N.
Eigenvectors are never compared entrywise (phase / rotation freedom, SURVEY.md 8(c) reading 4)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def gpu_solve(H, nev=None, **opts):
    from paper_2310_03341_b200 import binding
    N = H.shape[0]
    solver = binding.Eigh(N, nev, **opts)
    G = np.array(H, dtype=np.complex128)
    G[np.triu_indices(N, 1)] = np.nan              # only the lower triangle may be read
    At = torch.from_numpy(np.ascontiguousarray(G.T)).cuda()
    W, Zt = solver.solve(At)
    torch.cuda.synchronize()
    info = {"phases_ms": solver.phase_times_ms(), "launches": solver.launch_count()}
    solver.close()
    return W.cpu().numpy(), Zt.cpu().numpy().T, info


def check(H, W, Z, Wref, nev=None):
    N = H.shape[0]
    nev = N if nev is None else nev
    nrm2 = np.abs(Wref).max() if N else 1.0
    assert np.isfinite(W).all() and np.isfinite(Z).all()
    assert np.all(np.diff(W) >= 0)
    assert np.abs(W - Wref).max() <= 1e-11 * max(nrm2, 1e-300)
    nf = max(np.linalg.norm(H), 1e-300)
    res = np.linalg.norm(H @ Z - Z * W[None, :nev]) / (nf * np.sqrt(N))
    orth = np.abs(Z.conj().T @ Z - np.eye(nev)).max()
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth
    return res, orth


def rand_herm(n, seed):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    return 0.5 * (A + A.conj().T)


@pytest.mark.parametrize("N", [1, 2, 3, 5, 31, 63, 64, 65, 66, 127, 128, 129, 130, 200, 333, 517])
def test_small_and_ragged_sizes(N):
    H = rand_herm(N, 1000 + N)
    W, Z, _ = gpu_solve(H)
    Wo = oracle.eigh(H, vectors=False)
    check(H, W, Z, Wo)


@pytest.mark.parametrize("method", [2, 1])
@pytest.mark.parametrize("scale", [2.0 ** -333, 1e-140, 1e-100, 1e-3, 1e100, 1e140])
def test_solve_of_a_scaled_matrix(method, scale):
    """eigh(s H) = s eigh(H), same eigenvectors, for matrix norms far from 1 (the squares of the entries must stay
    representable: include/eigh.h).  The merge step of the D&C deflates against 8 eps max(|d|_max, |z|_max) with a unit
    vector z -- a test that assumes a matrix of norm ~1; S3 scales the tridiagonal matrix by a power of two first (as
    LAPACK's xSTEDC does).  Without that a matrix of norm 1e-100 deflated everything: eigenvalue errors of 5 % of the
    norm at full orthogonality, no error code.  Expected values: the oracle on the UNSCALED matrix."""
    N = 200
    H = rand_herm(N, 77)
    Wo = oracle.eigh(H, vectors=False)
    W, Z, _ = gpu_solve(H * scale, method=method)
    check(H, W / scale, Z, Wo)
    if scale == 2.0 ** -333:                      # a power of two: the whole solve scales exactly
        W1, Z1, _ = gpu_solve(H, method=method)
        assert np.array_equal(W / scale, W1) and np.array_equal(Z, Z1)


def test_config0_closed_form_and_oracle():
    """Config 0: BdG uniform pairing 8x8x8 (N=1024), 64 distinct eigenvalues with multiplicity up to
    48: massive deflation.  Against the oracle and against the closed form."""
    w = wl.make_config(0)
    H = w.dense()
    W, Z, info = gpu_solve(H)
    Wo, Zo = oracle.eigh(H)
    check(H, W, Z, Wo)
    ks = [2 * np.pi * np.arange(-4, 4) / 8] * 3
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    eps_k = 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1)
    E = np.sqrt((eps_k - 0.5) ** 2 + 0.04)
    ref = np.sort(np.concatenate([-E, E]))
    assert np.abs(W - ref).max() <= 1e-11 * np.abs(ref).max()
    # particle-hole symmetry and projector agreement with the oracle on each degenerate shell
    assert np.abs(W + W[::-1]).max() <= 1e-11 * np.abs(ref).max()
    vals = np.unique(np.round(ref, 8))
    for v in vals[::7]:
        grp = np.abs(ref - v) < 1e-6
        P1 = Z[:, grp] @ Z[:, grp].conj().T
        P2 = Zo[:, grp] @ Zo[:, grp].conj().T
        assert np.linalg.norm(P1 - P2) <= 1e-9 * 14.4 / 0.045


def test_prescribed_spectrum_clusters():
    """Config-1 recipe at N=1500: clusters of width 1e-12 (deflation stress)."""
    A, lam = wl.random_hermitian_clustered(1500, wl.SEED_BASE + 1)
    W, Z, _ = gpu_solve(A)
    assert np.abs(W - lam).max() <= 1e-11
    Wo = oracle.eigh(A, vectors=False)
    check(A, W, Z, Wo)


def test_vortex_bdg_and_subset():
    """Config-2/3 recipe on a small lattice (N = 2*6*6*8 = 576): complex pairing field; nev = N/2
    (lowest half) and the positive branch through -H (SURVEY.md 8(c) reading 3)."""
    p = wl.bdg_vortex_tangle((6, 6, 8), 4, 1.0, wl.SEED_BASE + 3, 0.02)
    H = p.dense()
    N = H.shape[0]
    Wo = oracle.eigh(H, vectors=False)
    W, Z, _ = gpu_solve(H)
    check(H, W, Z, Wo)
    assert np.abs(W + W[::-1]).max() <= 1e-11 * np.abs(Wo).max()
    W2, Z2, _ = gpu_solve(H, nev=N // 2)
    assert Z2.shape == (N, N // 2)
    check(H, W2, Z2, Wo, nev=N // 2)
    W3, Z3, _ = gpu_solve(-H, nev=N // 2)
    check(-H, W3, Z3, -Wo[::-1], nev=N // 2)
    assert np.all(-W3[: N // 2][::-1] > 0)          # positive quasiparticle energies


def test_degenerate_inputs():
    """Diagonal, zero, identity-like and already-banded matrices."""
    N = 200
    D = np.diag(np.linspace(-3, 5, N)).astype(np.complex128)
    W, Z, _ = gpu_solve(D)
    check(D, W, Z, np.sort(np.diag(D).real))
    Zr = np.zeros((N, N), dtype=np.complex128)
    W, Z, _ = gpu_solve(Zr)
    assert np.abs(W).max() == 0.0
    assert np.abs(Z.conj().T @ Z - np.eye(N)).max() <= 1e-12 * N
    I = 2.5 * np.eye(N, dtype=np.complex128)
    W, Z, _ = gpu_solve(I)
    assert np.abs(W - 2.5).max() <= 1e-14
    assert np.abs(Z.conj().T @ Z - np.eye(N)).max() <= 1e-12 * N


@pytest.mark.parametrize("method", [2, 1])
@pytest.mark.parametrize("bad", [float("nan"), float("inf")])
def test_non_finite_input_fails_loudly_and_returns(method, bad):
    """A NaN or an infinity in the matrix: the call comes back (every iteration in the library is bounded) with a positive
    return code below EIGH_ERR_CUDA = 1000 -- the failure count is capped at 999 so that it cannot be read as a CUDA error --
    and a text that says what happened.  (Run under the suite's timeout: a hang here would be the bug.)"""
    import ctypes
    from paper_2310_03341_b200 import binding
    N = 300
    H = rand_herm(N, 99)
    H[200, 17] = H[17, 200] = bad
    eng = binding.Eigh(N, method=method)
    At = torch.from_numpy(np.ascontiguousarray(H.T)).cuda()
    W = torch.empty(N, dtype=torch.float64, device="cuda")
    Zt = torch.empty((N, N), dtype=torch.complex128, device="cuda")
    rc = eng.lib.eigh_solve(eng.h, ctypes.c_void_p(At.data_ptr()), N, ctypes.c_void_p(W.data_ptr()),
                            ctypes.c_void_p(Zt.data_ptr()), None)
    torch.cuda.synchronize()
    assert 0 < rc < 1000, rc
    assert "did not converge" in eng.last_error()
    with pytest.raises(binding.EighError):
        eng.solve(torch.from_numpy(np.ascontiguousarray(H.T)).cuda())
    eng.close()


@pytest.mark.parametrize("N", [130, 257, 389])
@pytest.mark.parametrize("nev_of", [lambda N: 1, lambda N: 7, lambda N: 63, lambda N: 65, lambda N: N - 1])
def test_ragged_subsets(N, nev_of):
    """Odd N with odd nev: ragged tiles in every GEMM of S3 / S4a / S4b (N-tails of 1, 7, 63, 65 columns), the column
    slabs of S4a with a partial last slab, and the nev-aware last merge of S3."""
    nev = nev_of(N)
    H = rand_herm(N, 5000 + N)
    W, Z, _ = gpu_solve(H, nev=nev)
    assert Z.shape == (N, nev)
    Wo = oracle.eigh(H, vectors=False)
    check(H, W, Z, Wo, nev=nev)
