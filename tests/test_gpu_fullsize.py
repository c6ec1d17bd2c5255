"""Full-size parity (-m gpu): the configuration bench.py times (config 3, N = 27648, all eigenpairs and the
nev = N/2 run on -H) checked by properties that hold at any size and certify the WHOLE result, plus
oracle spot checks on sampled outputs:

  * residual  ||H Z - Z Lambda||_F / (||H||_F sqrt N) <= 1e-13  and  ||Z^H Z - I||_max <= 1e-12 N  over ALL
    columns (an independent cuBLAS ZGEMM through torch.matmul, never the library's own GEMM): together
    they certify every eigenpair, hence the complete spectrum;
  * sum(lambda) = tr H, sum(lambda^2) = ||H||_F^2, W ascending, particle-hole symmetry
    lambda_i = -lambda_{N-1-i} (Eq. 7: the BdG matrix [[h, D], [D*, -h*]]);
  * oracle.sturm_count on the tridiagonal (d, e) that S1 + S2 produce: for sampled indices i the number of
    eigenvalues of T below W[i] -+ 1e-11 ||H||_2 brackets i (the oracle computes these one by one in O(N));
  * config 4 (N = 49152, the north_star target; needs ~150 GB and ~4 min): the same invariants, residual and
    orthogonality on 1536 sampled columns, and the lowest-N/2 run that bench.py times.

Tolerances are north_star's (SURVEY.md 8(c) reading 6)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _norms(Ht):
    """(||H||_F, tr H) of the device matrix."""
    return float(torch.linalg.norm(Ht).item()), float(torch.diagonal(Ht).real.sum().item())


def _residual_orth(Hl, Zt, W, cols=None, block=2048):
    """Hl: logical H (N x N); Zt: (nev, N) rows = eigenvectors.  Returns (residual, orth) over `cols`
    (all columns when None), computed block-wise with torch.matmul."""
    N = Hl.shape[0]
    nev = Zt.shape[0]
    idx = torch.arange(nev, device=Zt.device) if cols is None else cols
    r2 = 0.0
    orth = 0.0
    for s in range(0, idx.numel(), block):
        ii = idx[s:s + block]
        Zb = Zt[ii].t()                                  # N x nb
        R = Hl @ Zb - Zb * W[ii][None, :]
        r2 += float((R.real ** 2 + R.imag ** 2).sum().item())
        for s2 in range(0, idx.numel(), block):
            jj = idx[s2:s2 + block]
            G = Zt[ii].conj() @ Zt[jj].t()               # nb x nb2
            if s == s2:
                G = G - torch.eye(ii.numel(), device=G.device, dtype=G.dtype)
            orth = max(orth, float(G.abs().max().item()))
            del G
        del R, Zb
    hn = float(torch.linalg.norm(Hl).item())
    return (r2 ** 0.5) / (hn * (idx.numel() ** 0.5)), orth       # = north_star's ||R||_F / (||H||_F sqrt N) when all N columns are taken


def _solve_config(index, nev=None, sign=1.0):
    from paper_2310_03341_b200 import binding
    w = wl.make_config(index)
    N = w.N
    nev = N if nev is None else nev
    dev = torch.device("cuda")
    At = torch.empty((N, N), dtype=torch.complex128, device=dev)
    w.dense_torch(dev, out=At, sign=sign)
    hn, tr = _norms(At)
    solver = binding.Eigh(N, nev)
    W, Zt = solver.solve(At)
    torch.cuda.synchronize()
    phases = solver.phase_times_ms()
    solver.close()
    w.dense_torch(dev, out=At, sign=sign)               # A was overwritten: regenerate H for the checks
    return w, At.t(), W, Zt, hn, tr, phases


def _check_invariants(W, hn, tr, N, ph_symmetric=True):
    Wn = W.cpu().numpy()
    assert np.isfinite(Wn).all()
    assert np.all(np.diff(Wn) >= 0)
    h2 = np.abs(Wn).max()
    assert abs(Wn.sum() - tr) <= 1e-11 * h2 * np.sqrt(N)
    assert abs(np.sum(Wn ** 2) - hn ** 2) <= 1e-12 * hn ** 2
    if ph_symmetric:
        assert np.abs(Wn + Wn[::-1]).max() <= 1e-11 * h2
    return Wn, h2


def test_config3_full_spectrum_certified():
    w, Hl, W, Zt, hn, tr, _ = _solve_config(3)
    N = w.N
    Wn, h2 = _check_invariants(W, hn, tr, N)
    res, orth = _residual_orth(Hl, Zt, W)
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth


def test_config3_sturm_counts_of_the_gpu_tridiagonal():
    """S3 at full size against the oracle, independently of the eigenvectors: (d, e) from the library's own
    S1 + S2 phase entry points, eigenvalues from eigh_solve on the same matrix."""
    from paper_2310_03341_b200 import binding
    w = wl.make_config(3)
    N = w.N
    dev = torch.device("cuda")
    At = torch.empty((N, N), dtype=torch.complex128, device=dev)
    w.dense_torch(dev, out=At)
    eng = binding.Eigh(N)
    band = torch.zeros((N, eng.ldab), dtype=torch.complex128, device=dev)
    d = torch.empty(N, dtype=torch.float64, device=dev)
    e = torch.empty(N, dtype=torch.float64, device=dev)
    eng.reduce_to_band(At, band)
    eng.band_to_tridiag(band, d, e)
    w.dense_torch(dev, out=At)
    W, _ = eng.solve(At)
    torch.cuda.synchronize()
    eng.close()
    dn, en, Wn = d.cpu().numpy(), e.cpu().numpy()[: N - 1], W.cpu().numpy()
    h2 = np.abs(Wn).max()
    idx = np.unique(np.concatenate([np.linspace(0, N - 1, 96).astype(int), [0, 1, N // 2 - 1, N // 2, N - 2, N - 1]]))
    delta = 1e-11 * h2
    below = oracle.sturm_count(dn, en, Wn[idx] - delta)
    above = oracle.sturm_count(dn, en, Wn[idx] + delta)
    assert np.all(below <= idx), (below - idx).max()
    assert np.all(above >= idx + 1), (idx + 1 - above).max()


def test_config3_positive_branch_nev_half():
    """nev = N/2 "positive quasiparticle energies" (BASELINE.json config 3) = the lowest N/2 pairs of -H
    (reading 3).  Sampled residual / orthogonality plus the invariants on all N eigenvalues."""
    w = wl.make_config(3)
    N = w.N
    nev = N // 2
    w, Hl, W, Zt, hn, tr, _ = _solve_config(3, nev=nev, sign=-1.0)
    Wn, h2 = _check_invariants(W, hn, tr, N)
    assert Zt.shape == (nev, N)
    assert Wn[nev - 1] < 0.0 < Wn[nev]                   # the gap at zero separates the branches
    cols = torch.linspace(0, nev - 1, 1024, device=Zt.device).long().unique()
    res, orth = _residual_orth(Hl, Zt, W, cols=cols)
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth


def test_config3_densities_from_the_lowest_half():
    """SCF epilogue at the size bench.py times (Eq. 16a, 16d, 17): nev = N/2 LOWEST pairs of H
    (the negative branch) and eigh_densities with branch = -1.  The oracle recomputes n(r), nu(r) one point at a
    time on 48 sampled grid points from the mapped states [-conj(v), conj(u)]; properties that hold at any size
    cover every r: completeness n(r) -> 1, nu(r) -> 0 as T -> infinity, and the particle number."""
    from oracle import densities as od
    from paper_2310_03341_b200 import binding
    w = wl.make_config(3)
    N = w.N
    M, nev = N // 2, N // 2
    dev = torch.device("cuda")
    At = torch.empty((N, N), dtype=torch.complex128, device=dev)
    w.dense_torch(dev, out=At)
    eng = binding.Eigh(N, nev)
    W, Zt = eng.solve(At)
    del At
    assert float(W[nev - 1].item()) < 0.0 < float(W[nev].item())
    E = W[:nev].contiguous()
    pts = np.unique(np.linspace(0, M - 1, 48).astype(int))
    rows = torch.from_numpy(np.concatenate([pts, M + pts])).to(dev)
    Zs = Zt[:, rows].t().cpu().numpy()                   # (2 P) x nev: u rows then v rows of the sampled points
    En = E.cpu().numpy()
    for T, Ec in ((0.0, np.inf), (0.1, 8.0)):
        n, nu = eng.densities(E, Zt, T=T, Ec=Ec, branch=-1)
        torch.cuda.synchronize()
        n, nu = n.cpu().numpy(), nu.cpu().numpy()
        n_o, nu_o = od.densities(*od.particle_hole_map(En, Zs), T=T, Ec=Ec)
        S = (np.abs(Zs) ** 2).sum(axis=1)
        tol = 4.0 * nev * np.finfo(np.float64).eps * (S[:pts.size] + S[pts.size:])
        assert np.all(np.abs(n[pts] - n_o) <= tol), np.abs(n[pts] - n_o).max()
        assert np.all(np.abs(nu[pts] - nu_o) <= tol), np.abs(nu[pts] - nu_o).max()
        assert np.all(n >= 0.0) and np.all(n <= 2.0 + 1e-9)
        if T == 0.0:
            # N_particles = sum_r n(r) = 2 sum_n ||v_n||^2 of the positive states = 2 sum ||u'||^2 of the mapped ones
            unorm = float((Zt[:, :M].real ** 2 + Zt[:, :M].imag ** 2).sum().item())
            assert abs(n.sum() - 2.0 * unorm) <= 1e-9 * n.sum()
    n, nu = eng.densities(E, Zt, T=1e12, branch=-1)
    torch.cuda.synchronize()
    assert float((n - 1.0).abs().max().item()) <= 1e-9
    assert float(nu.abs().max().item()) <= 1e-9
    # Eq. 16b / 16c at the same size, EVERY grid point: the oracle needs whole states for the gradients, so the 2048
    # lowest-|E| states are taken (columns nev-2048 .. nev-1, contiguous rows of Zt) and mapped to the positive branch
    shape = w.problem.shape
    Ds = [wl.derivative_1d(L) for L in shape]
    Dd = [torch.from_numpy(np.ascontiguousarray(D.T)).to(dev) for D in Ds]
    k = 2048
    Zk = Zt[nev - k:]
    Ek = E[nev - k:].contiguous()
    tau, j = eng.gradient_densities(shape, Dd[0], Dd[1], Dd[2], Ek, Zk, T=0.05, branch=-1)
    torch.cuda.synchronize()
    Ep, Zp = od.particle_hole_map(Ek.cpu().numpy(), Zk.t().cpu().numpy())
    tau_o, j_o = od.gradient_densities(Ep, Zp, shape, *Ds, T=0.05)
    t_inf, _ = od.gradient_densities(np.ones(k), Zp, shape, *Ds, T=1e12)
    n_inf, _ = od.densities(np.ones(k), Zp, T=1e12)
    c = 8.0 * (k + 2 * max(shape)) * np.finfo(np.float64).eps
    assert np.abs(tau.cpu().numpy() - tau_o).max() <= c * 2.0 * t_inf.max()
    assert np.abs(j.cpu().numpy() - j_o).max() <= c * 2.0 * np.sqrt(t_inf.max() * n_inf.max())
    # completeness over all N/2 states at T -> infinity: tau(r) = sum_a (D_a D_a^T)[i_a, i_a] (constant), j(r) = 0
    tau, j = eng.gradient_densities(shape, Dd[0], Dd[1], Dd[2], E, Zt, T=1e12, branch=-1)
    torch.cuda.synchronize()
    ref = sum(float(np.sum(D * D, axis=1)[0]) for D in Ds)
    assert float((tau - ref).abs().max().item()) <= 1e-8 * ref
    assert float(j.abs().max().item()) <= 1e-8
    eng.close()


def test_config4_target_size_sampled():
    """The north_star target, BASELINE.json config 4 (N = 49152, all eigenpairs; ~150 GB of HBM, a few minutes): the
    invariants on all N eigenvalues and the residual / orthogonality of 1536 sampled columns against every other
    sampled column."""
    w, Hl, W, Zt, hn, tr, phases = _solve_config(4)
    N = w.N
    Wn, h2 = _check_invariants(W, hn, tr, N)
    cols = torch.linspace(0, N - 1, 1536, device=Zt.device).long().unique()
    res, orth = _residual_orth(Hl, Zt, W, cols=cols)
    print(f"config 4: phases_ms={phases} residual={res:.2e} orth={orth:.2e}")
    assert res <= 1e-13, res
    assert orth <= 1e-12 * N, orth
