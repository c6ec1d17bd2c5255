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
    for o in range(b + 1):
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
