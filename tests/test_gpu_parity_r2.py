"""Parity cases added in round 2 (-m gpu), all through the C ABI against the CPU oracle at north_star's tolerances
(|lambda - lambda_ref| <= 1e-11 ||H||_2; ||HZ - Z Lambda||_F / (||H||_F sqrt N) <= 1e-13; ||Z^H Z - I||_max <= 1e-12 N):

  * BASELINE.json config 1 at its full size N = 4096 (409 values in 41 clusters of width 1e-12): prescribed spectrum
    and the oracle's eigenvalues;
  * config 2 at its full size N = 8192 (single vortex line): eigenvalues against `oracle.eigh(..., vectors=False)`,
    residual / orthogonality by an independent cuBLAS ZGEMM;
  * the extended-precision oracle (`oracle.eigh_ld`, SURVEY.md 8(c) "extended precision truth") at N <= 2048: the GPU
    result and the FP64 oracle both sit within c N eps ||H||_2 of it;
  * every `eigh_set_option` key that selects a different code path, at a size where that path is really exercised
    (`panel_smem = 0`: the L2-resident panel QR + Gram GEMM + T recurrence with panels thousands of rows tall -- the
    path the first 43 % of the panels take at N = 49152);
  * `eigh_tridiag_dc` with off-diagonals of either sign (eigenvector residual on the signed matrix);
  * `eigh_solve_host` with pageable and with pinned host buffers spanning several chunks of the staging ring.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu
EPS = np.finfo(np.float64).eps


def _solve_np(H, nev=None, **opts):
    from paper_2310_03341_b200 import binding
    N = H.shape[0]
    eng = binding.Eigh(N, nev, **opts)
    At = torch.from_numpy(np.ascontiguousarray(H.T)).cuda()
    W, Zt = eng.solve(At)
    torch.cuda.synchronize()
    eng.close()
    return W, Zt


def _residual_orth_dev(H, W, Zt, block=2048):
    """residual and orthogonality over all columns on the device (torch.matmul = cuBLAS, never the library's GEMM)."""
    Hd = torch.from_numpy(H).cuda()
    N, nev = H.shape[0], Zt.shape[0]
    W = W[:nev]
    r2, orth = 0.0, 0.0
    for s in range(0, nev, block):
        Zb = Zt[s:s + block].t()
        R = Hd @ Zb - Zb * W[s:s + block][None, :]
        r2 += float((R.real ** 2 + R.imag ** 2).sum().item())
        for s2 in range(0, nev, block):
            G = Zt[s:s + block].conj() @ Zt[s2:s2 + block].t()
            if s == s2:
                G = G - torch.eye(G.shape[0], device=G.device, dtype=G.dtype)
            orth = max(orth, float(G.abs().max().item()))
    hn = float(torch.linalg.norm(Hd).item())
    return (r2 ** 0.5) / (hn * (nev ** 0.5)), orth


def test_config1_full_size_clustered_spectrum():
    """BASELINE.json config 1: N = 4096, lambda uniform in [-1, 1] with 10 % of the values in clusters of width 1e-12
    (SURVEY.md 8(c) reading 12)."""
    w = wl.make_config(1)
    H = w.dense()
    N = H.shape[0]
    assert N == 4096
    lam = w.lam_exact
    W, Zt = _solve_np(H)
    Wn = W.cpu().numpy()
    assert np.all(np.diff(Wn) >= 0)
    # prescribed spectrum: within N eps ||A|| (+ the cluster width for members of a cluster)
    assert np.abs(Wn - np.sort(lam)).max() <= 1e-11, np.abs(Wn - np.sort(lam)).max()
    Wo = oracle.eigh(H, vectors=False)
    assert np.abs(Wn - Wo).max() <= 1e-11 * np.abs(Wo).max()
    res, orth = _residual_orth_dev(H, W, Zt)
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth
    # the 41 clusters: the computed members of each cluster stay within its width + N eps
    srt = np.sort(lam)
    gaps = np.diff(srt)
    in_cluster = np.zeros(N, dtype=bool)
    in_cluster[:-1] |= gaps < 2e-12
    in_cluster[1:] |= gaps < 2e-12
    assert 380 <= in_cluster.sum() <= 430
    assert np.abs(Wn[in_cluster] - srt[in_cluster]).max() <= 1e-12 + N * EPS


def test_config2_full_size_against_the_oracle():
    """BASELINE.json config 2: single vortex line on 16x16x16, N = 8192, all eigenpairs; eigenvalues against the oracle
    (values only: the O1 + O4 steps, minutes on the box's host cores)."""
    w = wl.make_config(2)
    H = w.dense()
    N = H.shape[0]
    assert N == 8192
    W, Zt = _solve_np(H)
    Wn = W.cpu().numpy()
    res, orth = _residual_orth_dev(H, W, Zt)
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth
    h2 = np.abs(Wn).max()
    assert np.abs(Wn + Wn[::-1]).max() <= 1e-11 * h2            # particle-hole symmetry (Eq. 7)
    assert abs(Wn.sum() - np.trace(H).real) <= 1e-11 * h2 * np.sqrt(N)
    del Zt
    Wo = oracle.eigh(H, vectors=False)
    assert np.abs(Wn - Wo).max() <= 1e-11 * np.abs(Wo).max(), np.abs(Wn - Wo).max()


@pytest.mark.parametrize("kind,N", [("herm", 700), ("bdg", 2 * 8 * 8 * 12), ("clustered", 2048)])
def test_against_the_long_double_oracle(kind, N):
    """the same oracle in x87 long double (eps = 1.1e-19) is the truth at N <= 2048; the GPU and the FP64
    oracle must both sit within c N eps_64 ||H||_2 of it (c = 4: two backward-stable methods)."""
    if kind == "herm":
        rng = np.random.default_rng(77)
        A = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        H = 0.5 * (A + A.conj().T)
    elif kind == "bdg":
        H = wl.bdg_vortex_tangle((8, 8, 12), 4, 1.0, wl.SEED_BASE + 21, 0.02).dense()
        assert H.shape[0] == N
    else:
        H, _ = wl.random_hermitian_clustered(N, wl.SEED_BASE + 22)
    Wld = oracle.eigh_ld(H, vectors=False)
    Wd = oracle.eigh(H, vectors=False)
    W, _ = _solve_np(H)
    Wn = W.cpu().numpy()
    h2 = np.abs(Wld).max()
    bound = 4.0 * N * EPS * h2
    assert np.abs(Wd - Wld).max() <= bound, (np.abs(Wd - Wld).max(), bound)
    assert np.abs(Wn - Wld).max() <= bound, (np.abs(Wn - Wld).max(), bound)
    assert bound <= 1e-11 * h2


_OPTION_CASES = [
    ({"panel_smem": 0}, 4000),           # L2 panel QR + Gram GEMM + tfactor with m up to 3936 rows
    ({"panel_smem": 0, "gemm_3m": 0}, 2100),
    ({"gemm_3m": 0}, 2100),
    ({"wy_group": 16}, 2100),
    ({"wy_group": 32}, 2100),
    ({"p4b_merge": 1}, 2100),
    ({"p4b_merge": 8}, 2100),
    ({"bt_chain": 4}, 2100),
    ({"dc_leaf": 8}, 2100),
    ({"dc_leaf": 17}, 2100),
    ({"panel_rows_min": 16}, 2100),
    ({"panel_rows_min": 192}, 2100),
    ({"hemm_waves": 1}, 2100),
    ({"hemm_waves": 40}, 2100),
    ({"bc_grid": 7}, 2100),
    ({"dgemm_mi": 4}, 2100),             # S3 merges with the 32 x 32 warp tiles (round-1 kernel shape)
    ({"dgemm_mi": 8}, 2100),             # ... and back to the default (the switch is process-wide)
    ({"bc_variant": 0}, 2100),           # S2: publisher warp, 168 registers (the round-1 kernel)
    ({"bc_variant": 2}, 2100),           # S2: no publisher warp, full register file
    ({"bc_variant": 3}, 2100),           # S2: publisher warp + setmaxnreg (compute warps 224 registers)
    ({"bc_dual_steps": 1}, 2100),        # every sweep on the two-blocks-per-SM kernel
    ({"bc_dual_steps": 20}, 2100),       # long sweeps on the dual kernel, the rest on the publisher kernel
]


@pytest.fixture(scope="module")
def option_problems():
    out = {}
    for N in sorted({n for _, n in _OPTION_CASES}):
        # BdG-like structure is not needed here: a seeded dense Hermitian matrix with a few exact degeneracies
        rng = np.random.default_rng(9000 + N)
        A = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
        Q, _ = np.linalg.qr(A)
        lam = rng.uniform(-2.0, 3.0, N)
        lam[: N // 8] = np.round(lam[: N // 8], 1)                  # multiplicities (deflation in every variant)
        H = (Q * lam[None, :]) @ Q.conj().T
        H = 0.5 * (H + H.conj().T)
        out[N] = (H, oracle.eigh(H, vectors=False))
    return out


@pytest.mark.parametrize("opts,N", _OPTION_CASES, ids=[",".join(f"{k}={v}" for k, v in o.items()) for o, _ in _OPTION_CASES])
def test_option_matrix(option_problems, opts, N):
    """Every documented eigh_set_option knob against the oracle (zero parity coverage before)."""
    H, Wo = option_problems[N]
    nev = N if "wy_group" not in opts else N - 37                  # a ragged last slab for the S4a variants
    W, Zt = _solve_np(H, nev=nev, **opts)
    Wn = W.cpu().numpy()
    assert np.isfinite(Wn).all()
    assert np.abs(Wn - Wo).max() <= 1e-11 * np.abs(Wo).max(), np.abs(Wn - Wo).max()
    res, orth = _residual_orth_dev(H, W, Zt)
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth


@pytest.mark.parametrize("N,seed", [(2, 1), (3, 2), (33, 3), (257, 4), (1500, 5)])
def test_tridiag_dc_signed_offdiagonal(N, seed):
    """include/eigh.h: e may have either sign.  Residual on the SIGNED matrix (the eigenvalues do not depend on the
    signs, the eigenvectors do)."""
    from paper_2310_03341_b200 import binding
    rng = np.random.default_rng(seed)
    d = rng.standard_normal(N)
    e = rng.standard_normal(N - 1)
    e[::7] = -np.abs(e[::7])
    if N > 40:
        e[20] = 0.0
        e[33] = -0.0
    eng = binding.Eigh(N)
    dd, ee = torch.from_numpy(d).cuda(), torch.from_numpy(np.concatenate([e, [0.0]])).cuda()
    W = torch.empty(N, dtype=torch.float64, device="cuda")
    Qt = torch.empty((N, N), dtype=torch.float64, device="cuda")
    assert eng.tridiag_dc(dd, ee, W, Qt) == 0
    torch.cuda.synchronize()
    fl, kf = eng.dc_stats()
    eng.close()
    Wn, Q = W.cpu().numpy(), Qt.cpu().numpy().T
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    assert np.linalg.norm(T @ Q - Q * Wn[None, :]) <= 1e-13 * max(np.linalg.norm(T), 1.0) * np.sqrt(N)
    assert np.abs(Q.T @ Q - np.eye(N)).max() <= 1e-13 * max(1, N / 100)
    Wo = oracle.tridiag_ql(d, e, vectors=False)
    assert np.abs(Wn - Wo).max() <= 1e-13 * max(np.abs(Wo).max(), 1.0) * max(1, N / 100)
    # statistics of the merge tree: one entry per level, fractions in [0, 1], flops bounded by the dense product
    assert all(0.0 <= k <= 1.0 for k in kf)
    assert sum(fl) <= 8.0 / 3.0 * N ** 3 + 64.0 * N * N


def test_dc_stats_total_deflation_and_none():
    """eigh_dc_stats: d = const, e = 0 deflates everything (kept fraction 0, no GEMM flops); a generic matrix keeps
    a sizeable part at the root."""
    from paper_2310_03341_b200 import binding
    N = 600
    for d, e, expect_zero in ((np.full(N, 2.5), np.zeros(N - 1), True),
                              (np.random.default_rng(3).standard_normal(N), np.ones(N - 1), False)):
        eng = binding.Eigh(N)
        W = torch.empty(N, dtype=torch.float64, device="cuda")
        Qt = torch.empty((N, N), dtype=torch.float64, device="cuda")
        assert eng.tridiag_dc(torch.from_numpy(d).cuda(), torch.from_numpy(np.concatenate([e, [0.0]])).cuda(), W, Qt) == 0
        fl, kf = eng.dc_stats()
        eng.close()
        assert len(fl) == len(kf) >= 4
        if expect_zero:
            assert sum(fl) == 0.0 and max(kf) == 0.0
        else:
            assert kf[-1] > 0.1 and fl[-1] > 0.0 and max(kf) <= 1.0


@pytest.mark.parametrize("pinned", [False, True])
def test_solve_host_streams_through_the_ring(pinned):
    """eigh_solve_host with host buffers larger than one 256 MiB chunk of the staging ring (N = 4200: A is 282 MB, so
    the H2D of A and the D2H of Z each take two chunks); pageable buffers go through the pinned ring, pinned ones are
    copied directly.  Same answer as eigh_solve, A_host untouched."""
    from paper_2310_03341_b200 import binding
    N = 4200
    rng = np.random.default_rng(4200)
    A = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    H = 0.5 * (A + A.conj().T)
    Ah = torch.from_numpy(np.ascontiguousarray(H.T))
    Wh = torch.empty(N, dtype=torch.float64)
    Zh = torch.empty((N, N), dtype=torch.complex128)
    if pinned:
        Ah, Wh, Zh = Ah.pin_memory(), Wh.pin_memory(), Zh.pin_memory()
    keep = Ah.clone()
    eng = binding.Eigh(N)
    At = torch.empty((N, N), dtype=torch.complex128, device="cuda")
    W = torch.empty(N, dtype=torch.float64, device="cuda")
    Zt = torch.empty((N, N), dtype=torch.complex128, device="cuda")
    eng.solve_host(Ah, Wh, Zh, At, W, Zt)
    assert torch.equal(Ah, keep)
    assert torch.equal(Wh, W.cpu()) and torch.equal(Zh, Zt.cpu())
    At.copy_(torch.from_numpy(np.ascontiguousarray(H.T)))
    W2, Zt2 = eng.solve(At)
    torch.cuda.synchronize()
    assert torch.equal(W2.cpu(), Wh)                     # deterministic: bit-identical to the device-resident solve
    assert torch.equal(Zt2.cpu(), Zh)
    eng.close()
    res, orth = _residual_orth_dev(H, W, Zt)
    assert res <= 1e-13 and orth <= 1e-12 * N


@pytest.mark.parametrize("method", [2, 1])
def test_column_shards_reproduce_the_unsharded_solve(method):
    """SURVEY.md 8(f)3, first slice: every "rank" solves with its own column shard (option col_begin,
    nev = shard width; S1-S3 replicated, back-transformations on the shard only).  Emulated on one GPU, one shard after
    the other: the gathered Z equals the unsharded Z column by column (up to the phase-free rounding of different GEMM
    splits), W is identical on every rank, and the gathered result meets the north_star tolerances."""
    from paper_2310_03341_b200 import binding, shard
    p = wl.bdg_vortex_tangle((6, 8, 8), 4, 1.0, wl.SEED_BASE + 71, 0.02)
    H = p.dense()
    N = H.shape[0]                              # 768
    nev = 500
    opts = {"method": 1} if method == 1 else {}
    ref = binding.Eigh(N, nev, **opts)
    W0, Z0 = ref.solve(torch.from_numpy(np.ascontiguousarray(H.T)).cuda())
    torch.cuda.synchronize()
    ref.close()
    parts = []
    for b, e in shard.column_shards(nev, 3):
        assert e > b
        eng = binding.Eigh(N, e - b, **dict(opts, col_begin=b))
        W, Zt = eng.solve(torch.from_numpy(np.ascontiguousarray(H.T)).cuda())
        torch.cuda.synchronize()
        eng.close()
        assert torch.equal(W, W0)                                   # replicated S1-S3: identical bits
        parts.append(Zt)
    Zg = torch.cat(parts, 0)
    assert Zg.shape == Z0.shape
    # same eigenvectors: |<z_sharded, z_ref>| = 1 column by column (non-degenerate spectrum), and the values agree closely
    ov = (Zg.conj() * Z0).sum(dim=1).abs()
    assert float((ov - 1.0).abs().max().item()) <= 1e-12
    assert float((Zg - Z0).abs().max().item()) <= 1e-12
    res, orth = _residual_orth_dev(H, W0, Zg)
    assert res <= 1e-13 and orth <= 1e-12 * N
    with pytest.raises(binding.EighError):
        binding.Eigh(N, 100, col_begin=N - 50)                      # shard beyond the spectrum
