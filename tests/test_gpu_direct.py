"""The 1-stage and real-symmetric variants (PAPER.md:148 steps i-iii, the solver of the paper's Figs. 3-4;
PAPER.md:140, :158-160 real FP64) through the C ABI, against the CPU oracle:

  * `eigh_tridiagonalise_direct`: d and |e| element by element against `oracle.tridiagonalise` (the tridiagonal form is
    unique up to the phases of the off-diagonals -- pinned on the CPU in test_oracle_pins.py), spectrum of T against the
    spectrum of A, trace / Frobenius invariants, lower triangle only;
  * `eigh_solve` with method = 1 (complex) and with dtype = 1 (real symmetric): north_star's tolerances;
  * `eigh_backtransform_direct`: Q from the stored reflectors is unitary and Q^H A Q = T;
  * the real GEMM engine (`eigh_k_rgemm`) against torch.matmul (cuBLAS).
Eigenvectors are never compared entrywise (SURVEY.md 8(c) reading 4)."""
import numpy as np
import pytest
import torch

import oracle
from gpu_util import cm, lg, randr
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu
EPS = np.finfo(np.float64).eps


def rand_herm(n, seed, real=False):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((n, n))
    if not real:
        A = A + 1j * rng.standard_normal((n, n))
    return 0.5 * (A + A.conj().T)


def _engine(N, nev=None, real=False, **opts):
    from paper_2310_03341_b200 import binding
    o = {"method": 1}
    if real:
        o["dtype"] = 1
    o.update(opts)
    return binding.Eigh(N, nev, **o)


def _to_dev(H, real):
    G = np.array(H, dtype=np.float64 if real else np.complex128)
    N = G.shape[0]
    G[np.triu_indices(N, 1)] = np.nan                       # only the lower triangle may be read
    return torch.from_numpy(np.ascontiguousarray(G.T)).cuda()


def _check(H, W, Z, Wref, nev=None):
    N = H.shape[0]
    nev = N if nev is None else nev
    nrm2 = max(np.abs(Wref).max(), 1e-300)
    assert np.isfinite(W).all() and np.isfinite(Z).all()
    assert np.all(np.diff(W) >= 0)
    assert np.abs(W - Wref).max() <= 1e-11 * nrm2, np.abs(W - Wref).max()
    nf = max(np.linalg.norm(H), 1e-300)
    res = np.linalg.norm(H @ Z - Z * W[None, :nev]) / (nf * np.sqrt(N))
    orth = np.abs(Z.conj().T @ Z - np.eye(nev)).max()
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth


@pytest.mark.parametrize("real", [False, True])
@pytest.mark.parametrize("N", [2, 3, 5, 63, 64, 65, 66, 129, 200, 517, 1100])
def test_tridiagonalise_direct_against_the_oracle(N, real):
    H = rand_herm(N, 2000 + N, real)
    eng = _engine(N, real=real)
    At = _to_dev(H, real)
    d = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
    e = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
    eng.tridiagonalise_direct(At, d, e)
    torch.cuda.synchronize()
    eng.close()
    dn, en = d.cpu().numpy(), e.cpu().numpy()[: N - 1]
    assert np.isfinite(dn).all() and np.isfinite(en).all()
    do, eo, _ = oracle.tridiagonalise(H.astype(np.complex128))
    nrm = np.linalg.norm(H, 2)
    # unique tridiagonal form; the recursion loses accuracy slowly with N (not a backward-stable quantity): 1e-9 ||H||
    # at these sizes, and the backward-stable statements below at full accuracy
    assert np.abs(dn - do).max() <= 1e-9 * nrm, np.abs(dn - do).max()
    assert np.abs(np.abs(en) - eo).max() <= 1e-9 * nrm, np.abs(np.abs(en) - eo).max()
    Wt = oracle.tridiag_ql(dn, np.abs(en), vectors=False)
    Wa = oracle.eigh(H.astype(np.complex128), vectors=False)
    assert np.abs(Wt - Wa).max() <= 1e-12 * np.abs(Wa).max() * max(1, N / 256)
    assert abs(dn.sum() - np.trace(H).real) <= 1e-11 * np.abs(Wa).max() * max(1, N / 256)
    assert abs(np.sum(dn ** 2) + 2 * np.sum(en ** 2) - np.linalg.norm(H) ** 2) <= 1e-11 * np.linalg.norm(H) ** 2


@pytest.mark.parametrize("real", [False, True])
@pytest.mark.parametrize("grid", [1, 2, 7, 40])
def test_panel_kernel_grid_size_does_not_change_a_bit(grid, real):
    """Option `ht_grid` (thread blocks of the cooperative panel kernel).  The per-tile partial products are stored per tile
    and summed by the owner of a row block in a fixed order, so WHICH block computes a tile must not change any bit of d, e,
    tau or the stored reflectors.  A small grid also makes every block walk the tile ring many times per column (N = 453:
    36 tiles and up to 16 (V_I, W_I) jobs per column on 1-7 blocks): the loader warps' full / empty handshake wraps."""
    N = 453
    H = rand_herm(N, 2500, real)
    outs = []
    for g in (0, grid):                                      # 0 = the default (one block per SM, at most one per tile)
        eng = _engine(N, real=real, **({"ht_grid": g} if g else {}))
        At = _to_dev(H, real)
        d = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
        e = torch.full((N,), float("nan"), dtype=torch.float64, device="cuda")
        eng.tridiagonalise_direct(At, d, e)
        torch.cuda.synchronize()
        if g:
            assert eng.get_option("ht_grid") == g
        eng.close()
        outs.append((d.clone(), e.clone(), At.clone()))
    d0, e0, A0 = outs[0]
    d1, e1, A1 = outs[1]
    assert torch.equal(d0, d1) and torch.equal(e0[: N - 1], e1[: N - 1])
    # stored reflectors: the lower triangle of A (column-major = the upper triangle of At); the rest is NaN input
    iu = torch.triu_indices(N, N, device="cuda")
    a0, a1 = A0[iu[0], iu[1]], A1[iu[0], iu[1]]
    assert bool(torch.isfinite(torch.view_as_real(a0) if not real else a0).all())
    assert torch.equal(torch.view_as_real(a0) if not real else a0, torch.view_as_real(a1) if not real else a1)


@pytest.mark.parametrize("real", [False, True])
@pytest.mark.parametrize("N", [1, 2, 3, 5, 31, 64, 65, 127, 130, 200, 333, 517, 1300])
def test_one_stage_solve_small_and_ragged(N, real):
    H = rand_herm(N, 3000 + N, real)
    eng = _engine(N, real=real)
    W, Zt = eng.solve(_to_dev(H, real))
    torch.cuda.synchronize()
    assert Zt.dtype == (torch.float64 if real else torch.complex128)
    ph = eng.phase_times_ms()
    assert ph[1] == 0.0 and ph[3] == 0.0
    eng.close()
    _check(H.astype(np.complex128), W.cpu().numpy(), Zt.cpu().numpy().T.astype(np.complex128),
           oracle.eigh(H.astype(np.complex128), vectors=False))


@pytest.mark.parametrize("real", [False, True])
@pytest.mark.parametrize("N,nev", [(130, 1), (257, 7), (389, 65), (389, 388), (1024, 512)])
def test_one_stage_subsets(N, nev, real):
    H = rand_herm(N, 3500 + N, real)
    eng = _engine(N, nev, real=real)
    W, Zt = eng.solve(_to_dev(H, real))
    torch.cuda.synchronize()
    eng.close()
    assert Zt.shape == (nev, N)
    _check(H.astype(np.complex128), W.cpu().numpy(), Zt.cpu().numpy().T.astype(np.complex128),
           oracle.eigh(H.astype(np.complex128), vectors=False), nev=nev)


@pytest.mark.parametrize("real", [False, True])
def test_config0_on_the_one_stage_paths(real):
    """BASELINE.json config 0 is a REAL matrix with a closed-form spectrum (64 distinct values, multiplicities up to 48):
    the real-symmetric path and the complex 1-stage path against the closed form +-sqrt((eps_k - mu)^2 + Delta^2), the
    oracle, and the oracle's projectors on sampled shells."""
    w = wl.make_config(0)
    H = w.dense()
    N = H.shape[0]
    Hin = H.real.copy() if real else H
    eng = _engine(N, real=real)
    W, Zt = eng.solve(_to_dev(Hin, real))
    torch.cuda.synchronize()
    eng.close()
    Wn, Z = W.cpu().numpy(), Zt.cpu().numpy().T.astype(np.complex128)
    Wo, Zo = oracle.eigh(H)
    _check(H, Wn, Z, Wo)
    ks = [2 * np.pi * np.arange(-4, 4) / 8] * 3
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    eps_k = 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1)
    E = np.sqrt((eps_k - 0.5) ** 2 + 0.04)
    ref = np.sort(np.concatenate([-E, E]))
    assert np.abs(Wn - ref).max() <= 1e-11 * np.abs(ref).max()
    for v in np.unique(np.round(ref, 8))[::9]:
        grp = np.abs(ref - v) < 1e-6
        P1 = Z[:, grp] @ Z[:, grp].conj().T
        P2 = Zo[:, grp] @ Zo[:, grp].conj().T
        assert np.linalg.norm(P1 - P2) <= 1e-9 * 14.4 / 0.045


def test_one_stage_matches_two_stage_on_a_vortex_problem():
    """The same BdG vortex matrix through both methods: eigenvalues agree to 1e-11 ||H||_2, projectors of the separated
    low-energy group agree, and both meet the oracle."""
    from paper_2310_03341_b200 import binding
    p = wl.bdg_vortex_tangle((6, 8, 8), 4, 1.0, wl.SEED_BASE + 31, 0.02)
    H = p.dense()
    N = H.shape[0]
    Wo = oracle.eigh(H, vectors=False)
    e1 = _engine(N)
    W1, Z1 = e1.solve(_to_dev(H, False))
    e2 = binding.Eigh(N)
    W2, Z2 = e2.solve(_to_dev(H, False))
    torch.cuda.synchronize()
    e1.close(); e2.close()
    _check(H, W1.cpu().numpy(), Z1.cpu().numpy().T, Wo)
    assert np.abs(W1.cpu().numpy() - W2.cpu().numpy()).max() <= 1e-11 * np.abs(Wo).max()


@pytest.mark.parametrize("real", [False, True])
@pytest.mark.parametrize("N", [66, 300])
def test_backtransform_direct_reproduces_q(N, real):
    """Q (applied to the identity) is unitary and Q^H A Q equals tridiag(d, e)."""
    H = rand_herm(N, 4000 + N, real)
    eng = _engine(N, real=real)
    At = _to_dev(H, real)
    d = torch.empty(N, dtype=torch.float64, device="cuda")
    e = torch.empty(N, dtype=torch.float64, device="cuda")
    eng.tridiagonalise_direct(At, d, e)
    Zt = torch.eye(N, dtype=torch.float64 if real else torch.complex128, device="cuda")
    eng.backtransform_direct(At, Zt)
    torch.cuda.synchronize()
    eng.close()
    Q = Zt.cpu().numpy().T.astype(np.complex128)
    dn, en = d.cpu().numpy(), e.cpu().numpy()[: N - 1]
    T = np.diag(dn) + np.diag(en, 1) + np.diag(en, -1)
    assert np.abs(Q.conj().T @ Q - np.eye(N)).max() <= 1e-13 * N
    assert np.linalg.norm(Q.conj().T @ H @ Q - T) <= 1e-13 * N * np.linalg.norm(H)


def test_real_path_needs_method_one_and_phase_entries_check_the_method():
    from paper_2310_03341_b200 import binding
    with pytest.raises(binding.EighError):
        binding.Eigh(64, dtype=1)                          # real symmetric without method = 1
    eng = binding.Eigh(64)
    At = torch.zeros((64, 64), dtype=torch.complex128, device="cuda")
    d = torch.zeros(64, dtype=torch.float64, device="cuda")
    with pytest.raises(binding.EighError):
        eng.tridiagonalise_direct(At, d, d)                # two-stage handle
    eng.close()


@pytest.fixture(scope="module")
def geng():
    from paper_2310_03341_b200 import binding
    e = binding.Eigh(1024)
    yield e
    e.close()


def rel(a, b):
    return (a - b).abs().max().item() / max(b.abs().max().item(), 1e-300)


@pytest.mark.parametrize("opA,opB", [("N", "N"), ("N", "T"), ("T", "N"), ("T", "T")])
@pytest.mark.parametrize("M,N,K,sk", [(128, 64, 16, 1), (300, 200, 77, 1), (64, 64, 1000, 4), (257, 129, 64, 1), (1, 1, 1, 1),
                                      (515, 70, 131, 2), (5, 300, 9, 1)])
def test_rgemm_variants(geng, opA, opB, M, N, K, sk):
    A = randr(M, K, 1) if opA == "N" else randr(K, M, 1)
    B = randr(K, N, 2) if opB == "N" else randr(N, K, 2)
    C0 = randr(M, N, 3)
    As, Bs, Cs = cm(A), cm(B), cm(C0).clone()              # (cm() of a 1 x 1 tensor aliases its argument)
    geng.rgemm(opA, opB, M, N, K, 0.75, As, A.shape[0], Bs, B.shape[0], -0.5, Cs, M, splitk=sk)
    torch.cuda.synchronize()
    ref = 0.75 * (A if opA == "N" else A.t()) @ (B if opB == "N" else B.t()) - 0.5 * C0
    assert rel(lg(Cs), ref) < 1e-13
    Cn = torch.full((N, M), float("nan"), dtype=torch.float64, device="cuda")      # beta = 0 must not read C
    geng.rgemm(opA, opB, M, N, K, 1.0, As, A.shape[0], Bs, B.shape[0], 0.0, Cn, M, splitk=sk)
    torch.cuda.synchronize()
    assert rel(lg(Cn), (A if opA == "N" else A.t()) @ (B if opB == "N" else B.t())) < 1e-13


@pytest.mark.parametrize("m,k", [(128, 64), (517, 64), (700, 33)])
def test_rgemm_syr2k_lower(geng, m, k):
    """C <- C - V W^T - W V^T on the lower tiles only (the trailing update of the real 1-stage path): tiles strictly
    above the diagonal are NaN-poisoned and must stay untouched, the lower triangle must match."""
    V, Wm, C0 = randr(m, k, 5), randr(m, k, 6), randr(m, m, 7)
    C0 = 0.5 * (C0 + C0.t())
    Cp = C0.clone()
    for i0 in range(0, m, 128):
        for j0 in range(0, m, 64):
            if i0 + 127 < j0:
                Cp[i0:i0 + 128, j0:j0 + 64] = float("nan")
    Vs, Ws, Cs = cm(V), cm(Wm), cm(Cp)
    geng.rgemm("N", "T", m, m, k, -1.0, Vs, m, Ws, m, 1.0, Cs, m, K2=k, A2=Ws, lda2=m, B2=Vs, ldb2=m, lower_only=1)
    torch.cuda.synchronize()
    ref = C0 - V @ Wm.t() - Wm @ V.t()
    out = lg(Cs)
    low = torch.tril(torch.ones(m, m, dtype=torch.bool, device="cuda"))
    assert rel(out[low], ref[low]) < 1e-13
    skipped = torch.isnan(Cp)
    assert torch.isnan(out[skipped]).all()


@pytest.mark.parametrize("real", [False, True])
def test_one_stage_solve_host(real):
    """eigh_solve_host on the 1-stage path, both element types (8-byte elements on the real path: the host <-> device
    copies must use the working type's size): same answer as the device-resident solve, bit for bit."""
    N = 300
    H = rand_herm(N, 5100, real)
    eng = _engine(N, real=real)
    dt = torch.float64 if real else torch.complex128
    Ah = torch.from_numpy(np.ascontiguousarray((H.real if real else H).T)).to(dt)
    Wh = torch.empty(N, dtype=torch.float64)
    Zh = torch.empty((N, N), dtype=dt)
    At = torch.empty((N, N), dtype=dt, device="cuda")
    W = torch.empty(N, dtype=torch.float64, device="cuda")
    Zt = torch.empty((N, N), dtype=dt, device="cuda")
    eng.solve_host(Ah, Wh, Zh, At, W, Zt)
    W2, Zt2 = eng.solve(Ah.cuda())
    torch.cuda.synchronize()
    eng.close()
    assert torch.equal(Wh, W2.cpu()) and torch.equal(Zh, Zt2.cpu())
    _check(H.astype(np.complex128), Wh.numpy(), Zh.numpy().T.astype(np.complex128),
           oracle.eigh(H.astype(np.complex128), vectors=False))
