"""The conventions include/eigh.h states for eigh_solve, checked through the C ABI on the GPU: only the lower triangle
is read, imaginary parts of the diagonal are ignored, lda > N is allowed, the result is deterministic, and
eigh_solve_host (host buffers, the e2e path bench.py times) gives the same answer."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _problem():
    p = wl.bdg_vortex_tangle((4, 6, 5), 3, 1.0, wl.SEED_BASE + 11, 0.02)      # N = 240: several panels, ragged
    return p.dense()


def _check(H, W, Z):
    N = H.shape[0]
    Wo = oracle.eigh(H, vectors=False)
    nrm = np.abs(Wo).max()
    assert np.abs(W - Wo).max() <= 1e-11 * nrm
    assert np.linalg.norm(H @ Z - Z * W[None, :]) / (np.linalg.norm(H) * np.sqrt(N)) <= 1e-13
    assert np.abs(Z.conj().T @ Z - np.eye(N)).max() <= 1e-12 * N


def test_lower_triangle_only_diag_imag_ignored_and_lda():
    from paper_2310_03341_b200 import binding
    H = _problem()
    N = H.shape[0]
    lda = N + 5
    A = np.full((lda, N), np.nan + 1j * np.nan, dtype=np.complex128, order="F")     # column-major, padding rows = NaN
    A[:N, :] = np.tril(H)
    iu = np.triu_indices(N, 1)
    A[:N, :][iu] = np.nan + 1j * np.nan                         # strict upper triangle must never be read
    A[np.arange(N), np.arange(N)] += 1j * np.linspace(-3, 3, N)  # imaginary diagonal must be ignored
    At = torch.from_numpy(np.ascontiguousarray(A.T)).cuda()      # (N, lda) row-major = A column-major with ld = lda
    eng = binding.Eigh(N)
    W = torch.empty(N, dtype=torch.float64, device="cuda")
    Zt = torch.empty((N, N), dtype=torch.complex128, device="cuda")
    rc = eng.lib.eigh_solve(eng.h, ctypes.c_void_p(At.data_ptr()), lda, ctypes.c_void_p(W.data_ptr()),
                            ctypes.c_void_p(Zt.data_ptr()), ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0, eng.last_error()
    torch.cuda.synchronize()
    eng.close()
    _check(H, W.cpu().numpy(), Zt.cpu().numpy().T)


def test_deterministic_and_input_overwritten():
    from paper_2310_03341_b200 import binding
    H = _problem()
    N = H.shape[0]
    eng = binding.Eigh(N)
    outs = []
    for _ in range(2):
        At = torch.from_numpy(np.ascontiguousarray(H.T)).cuda()
        W, Zt = eng.solve(At)
        torch.cuda.synchronize()
        outs.append((W.cpu().numpy().copy(), Zt.cpu().numpy().copy(), At.cpu().numpy()))
    eng.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert not np.array_equal(outs[0][2], H.T)                  # documented: A holds the stage-1 reflectors afterwards


@pytest.mark.parametrize("pinned", [True, False])
def test_solve_host_matches_device_solve(pinned):
    from paper_2310_03341_b200 import binding
    H = _problem()
    N = H.shape[0]
    eng = binding.Eigh(N)
    At = torch.from_numpy(np.ascontiguousarray(H.T)).cuda()
    W, Zt = eng.solve(At)
    torch.cuda.synchronize()
    Ah = torch.from_numpy(np.ascontiguousarray(H.T))
    Wh = torch.empty(N, dtype=torch.float64)
    Zh = torch.empty((N, N), dtype=torch.complex128)
    if pinned:
        Ah, Wh, Zh = Ah.pin_memory(), Wh.pin_memory(), Zh.pin_memory()
    Ad = torch.empty((N, N), dtype=torch.complex128, device="cuda")
    Wd = torch.empty(N, dtype=torch.float64, device="cuda")
    Zd = torch.empty((N, N), dtype=torch.complex128, device="cuda")
    eng.solve_host(Ah, Wh, Zh, Ad, Wd, Zd)
    eng.close()
    assert np.array_equal(Ah.numpy(), H.T)                      # A_host is not modified
    assert np.array_equal(Wh.numpy(), W.cpu().numpy()) and np.array_equal(Zh.numpy(), Zt.cpu().numpy())
    _check(H, Wh.numpy(), Zh.numpy().T)
