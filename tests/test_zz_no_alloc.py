"""eigh_densities_static (the allocation-free variant of eigh_densities, include/eigh.h) against the existing path.

Collected LAST on purpose (file name): the suite runs with `pytest -x`, a failure here must not hide other tests.

The entry point keeps its scratch in a file-scope device array that every call shares and that keeps the previous call's
contents, so the check is made on TWO CALLS IN A ROW with different inputs (different column counts, temperatures and
branches: a stale list of active columns or stale chunk partials from call 1 would corrupt call 2).  Tolerance = the one
tests/test_gpu_densities.py derives for sums taken in a different order: 4 k eps sum_j (|u_j(r)|^2 + |v_j(r)|^2)."""
import ctypes

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu
EPS = np.finfo(np.float64).eps


def _states(N, ncols, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    Zt = (torch.randn((ncols, N), dtype=torch.float64, generator=g) +
          1j * torch.randn((ncols, N), dtype=torch.float64, generator=g)).cuda() / np.sqrt(N)
    E = (torch.rand(ncols, dtype=torch.float64, generator=g) * 6.0 - 3.0).cuda()      # both signs: some columns inactive
    return E, Zt


def _check(n, nu, n_ref, nu_ref, Zt, M):
    k = Zt.shape[0]
    S = (Zt.real ** 2 + Zt.imag ** 2).sum(dim=0)
    tol = 4.0 * k * EPS * (S[:M] + S[M:]) * 2.0 + 1e-300                # weights are at most 2
    assert torch.isfinite(n).all() and torch.isfinite(nu.real).all() and torch.isfinite(nu.imag).all()
    assert bool(((n - n_ref).abs() <= tol).all()), float((n - n_ref).abs().max())
    assert bool(((nu - nu_ref).abs() <= tol).all()), float((nu - nu_ref).abs().max())


def test_static_scratch_variant_matches_eigh_densities_on_two_calls_in_a_row():
    from paper_2310_03341_b200 import binding
    N = 2 * 6 * 7 * 11                      # 924: M = 462 is not a multiple of the 128-row blocks
    M = N // 2
    ref = binding.Eigh(N)                   # existing path: handle with a workspace
    lib = binding.load()
    h = ctypes.c_void_p()                   # new path: a handle WITHOUT any workspace
    assert lib.eigh_create(ctypes.byref(h), N, N) == 0
    stream = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    n = torch.full((M,), float("nan"), dtype=torch.float64, device="cuda")
    nu = torch.full((M,), float("nan"), dtype=torch.complex128, device="cuda")
    cases = [(700, 0.0, float("inf"), 1, 11), (93, 0.3, 2.0, -1, 12)]       # (ncols, T, Ec, branch, seed): call 1, call 2
    for call, (ncols, T, Ec, branch, seed) in enumerate(cases):
        E, Zt = _states(N, ncols, seed)
        n_ref, nu_ref = ref.densities(E, Zt, T=T, Ec=Ec, branch=branch)
        torch.cuda.synchronize()
        n.fill_(float("nan")); nu.fill_(float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        rc = lib.eigh_densities_static(h, ctypes.c_void_p(E.data_ptr()), ctypes.c_void_p(Zt.data_ptr()), N, ncols, T, Ec, branch,
                                       ctypes.c_void_p(n.data_ptr()), ctypes.c_void_p(nu.data_ptr()), stream)
        assert rc == 0, lib.eigh_last_error(h)
        torch.cuda.synchronize()
        if call > 0:                                       # (the first call on a device may load the module lazily)
            assert torch.cuda.mem_get_info()[0] >= free_before     # the call took no device memory
        _check(n, nu, n_ref, nu_ref, Zt, M)
    # the same through the Python binding, and an empty input (no active column): n = 0, nu = 0
    E, Zt = _states(N, 40, 13)
    n_ref, nu_ref = ref.densities(E, Zt, T=0.1)
    ref.densities_static(E, Zt, n, nu, T=0.1)
    torch.cuda.synchronize()
    _check(n, nu, n_ref, nu_ref, Zt, M)
    ref.densities_static(E[:0], Zt[:0], n, nu)
    torch.cuda.synchronize()
    assert float(n.abs().max()) == 0.0 and float(nu.abs().max()) == 0.0
    assert lib.eigh_destroy(h) == 0
    ref.close()


def test_static_scratch_variant_rejects_sizes_beyond_its_maximum():
    """Limits of the 8 MiB array: N <= 65536, ncols <= 32760 -- a clear error, nothing launched."""
    from paper_2310_03341_b200 import binding
    lib = binding.load()
    buf = torch.zeros(16, dtype=torch.float64, device="cuda")
    p = ctypes.c_void_p(buf.data_ptr())
    h = ctypes.c_void_p()
    assert lib.eigh_create(ctypes.byref(h), 65538, 1) == 0
    assert lib.eigh_densities_static(h, p, p, 65538, 1, 0.0, 1.0, 1, p, p, None) == -1
    assert b"exceeds the static scratch limit" in lib.eigh_last_error(h)
    lib.eigh_destroy(h)
    assert lib.eigh_create(ctypes.byref(h), 65536, 65536) == 0
    assert lib.eigh_densities_static(h, p, p, 65536, 32761, 0.0, 1.0, 1, p, p, None) == -5
    assert b"ncols" in lib.eigh_last_error(h)
    lib.eigh_destroy(h)
    assert lib.eigh_create(ctypes.byref(h), 101, 1) == 0
    assert lib.eigh_densities_static(h, p, p, 101, 1, 0.0, 1.0, 1, p, p, None) == -1      # odd N
    lib.eigh_destroy(h)
    torch.cuda.synchronize()
