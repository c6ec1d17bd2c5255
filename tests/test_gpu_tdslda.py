"""One TDSLDA step on the GPU (SURVEY.md 8(f)4; PAPER.md:91 Eq. 5, :113-115 Eq. 8, :134 ABM) against oracle/tdslda.py,
element by element, through the C ABI.

Tolerances (derived): the GPU applies the kinetic term as dense 1-D matrices (sums of L products per axis), the oracle
through FFTs: both are backward stable, |gpu - oracle| <= c (nx + ny + nz) eps max|H phi| with c = 8 for the right-hand
side; one ABM step adds dt times six such terms to the state."""
import numpy as np
import pytest
import torch

import oracle
from oracle import tdslda as td
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu
EPS = np.finfo(np.float64).eps


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _kin(shape):
    return [_dev(wl.kinetic_1d(L)) for L in shape]


@pytest.mark.parametrize("shape,ncols", [((4, 4, 6), 5), ((3, 5, 4), 1), ((8, 8, 8), 37), ((1, 9, 16), 4), ((10, 12, 33), 9),
                                         ((24, 3, 40), 6)])
def test_rhs_against_the_fft_oracle(shape, ncols):
    """-i H phi: dense-matrix kinetic term on the tensor cores vs Eq. 8 through numpy FFTs, ragged extents (L = 1..40:
    every MB instance, padded rows), ragged line tiles and column chunks, ld > N."""
    from paper_2310_03341_b200 import binding
    M = int(np.prod(shape))
    N = 2 * M
    rng = np.random.default_rng(100 + M)
    V = rng.uniform(-0.3, 0.3, M)
    Delta = 0.3 * np.exp(2j * np.pi * rng.uniform(size=M)) * rng.uniform(0.5, 1.0, M)
    mu = 0.8
    Phi = rng.standard_normal((N, ncols)) + 1j * rng.standard_normal((N, ncols))
    ref = td.rhs(Phi, shape, V, Delta, mu)
    eng = binding.Eigh(N)
    K = _kin(shape)
    ld = N + 3
    Pt = torch.full((ncols, ld), float("nan"), dtype=torch.complex128, device="cuda")
    Pt[:, :N] = _dev(Phi.T)
    Ft = torch.full((ncols, ld), float("nan"), dtype=torch.complex128, device="cuda")
    eng.tdslda_rhs(shape, K[0], K[1], K[2], _dev(V), _dev(Delta), mu, Pt, Ft)
    torch.cuda.synchronize()
    eng.close()
    out = Ft[:, :N].cpu().numpy().T
    assert np.isfinite(out).all()
    assert torch.isnan(Ft[:, N:].real).all()                       # padding untouched
    tol = 8.0 * sum(shape) * EPS * np.abs(ref).max()
    assert np.abs(out - ref).max() <= tol, (np.abs(out - ref).max(), tol)


def test_rhs_is_the_dense_hamiltonian_of_the_solver():
    """The same H the eigensolver diagonalises: for an eigenvector, -i H phi = -i E phi."""
    from paper_2310_03341_b200 import binding
    shape = (6, 6, 8)
    p = wl.bdg_vortex_tangle(shape, 3, 1.0, wl.SEED_BASE + 51, 0.02)
    N = p.N
    eng = binding.Eigh(N)
    At = _dev(p.dense().T)
    W, Zt = eng.solve(At)
    K = _kin(shape)
    Ft = eng.tdslda_rhs(shape, K[0], K[1], K[2], _dev(p.V), _dev(p.Delta), p.mu, Zt)
    torch.cuda.synchronize()
    eng.close()
    R = Ft + 1j * W[:, None] * Zt
    assert float(R.abs().max().item()) <= 1e-12 * float(W.abs().max().item())


@pytest.mark.parametrize("shape,branch", [((4, 4, 4), 1), ((4, 6, 5), -1)])
def test_abm_step_against_the_oracle(shape, branch):
    """eigh_tdslda_step vs oracle.tdslda.abm5_step on the same state, history, fields and dt: y_{n+1}, f_{n+1}, Delta and
    n element by element; the history buffers f_n .. f_{n-3} untouched; three consecutive steps with pointer rotation."""
    from oracle import densities as od
    from paper_2310_03341_b200 import binding
    p = wl.bdg_vortex_tangle(shape, 2, 1.0, wl.SEED_BASE + 61, 0.02)
    H = p.dense()
    N = H.shape[0]
    M = N // 2
    E, Z = oracle.eigh(H)
    sel = np.where(E > 0)[0] if branch == 1 else np.where(E < 0)[0]
    Y0, E0 = Z[:, sel], E[sel]
    ncols = Y0.shape[1]
    g, dt, T = -1.5, 0.004, 0.05
    # oracle side: branch = -1 means the states stand for their particle-hole partners in the densities
    def o_fields(Y):
        if branch == 1:
            return td.pairing_field(Y, E0, g, T)
        Ep, Yp = od.particle_hole_map(E0, Y)
        return td.pairing_field(Yp, Ep, g, T)
    def o_rhs(Y):
        return td.rhs(Y, shape, p.V, o_fields(Y), p.mu)
    def o_step(Y, F):
        Yp = Y + dt * sum(c * f for c, f in zip(td.AB5, F))
        fp = o_rhs(Yp)
        Yc = Y + dt * (td.AM4[0] * fp + sum(c * f for c, f in zip(td.AM4[1:], F[:4])))
        return Yc, [o_rhs(Yc)] + list(F[:4])
    # history: exact phases of the stationary start (any smooth history will do for a parity test)
    F = [(-1j * E0 * np.exp(-1j * E0 * (-k * dt)))[None, :] * Y0 for k in range(5)]
    eng = binding.Eigh(N)
    K = _kin(shape)
    Yt = _dev(Y0.T)
    Fl = [_dev(f.T) for f in F]
    keep = [f.clone() for f in Fl]
    Ypt = torch.empty_like(Yt)
    n_d = torch.empty(M, dtype=torch.float64, device="cuda")
    D_d = torch.empty(M, dtype=torch.complex128, device="cuda")
    Yo, Fo = Y0, F
    for step in range(3):
        Fl_new = eng.tdslda_step(shape, K[0], K[1], K[2], _dev(p.V), g, p.mu, _dev(E0), dt, Yt, Fl, Ypt, n_d, D_d, T=T,
                                 branch=branch)
        torch.cuda.synchronize()
        if step == 0:
            for k in range(4):
                assert torch.equal(Fl[k], keep[k])                 # f_n .. f_{n-3} are inputs only
        Fl = Fl_new
        Yo, Fo = o_step(Yo, Fo)
        scale = np.abs(Fo[0]).max()
        tol = 64.0 * sum(shape) * EPS * scale * (step + 1)
        assert np.abs(Yt.cpu().numpy().T - Yo).max() <= tol * dt * 8 + 16 * EPS
        assert np.abs(Fl[0].cpu().numpy().T - Fo[0]).max() <= tol
        assert np.abs(D_d.cpu().numpy() - o_fields(Yo)).max() <= 1e-12
    eng.close()
    # unitary evolution: the states are still orthonormal to the order of the method
    G = (Yt.conj() @ Yt.t()).cpu().numpy()
    assert np.abs(G - np.eye(ncols)).max() <= 1e-6


def test_argument_errors():
    from paper_2310_03341_b200 import binding
    eng = binding.Eigh(2 * 4 * 4 * 4)
    K = _kin((4, 4, 4))
    V = torch.zeros(64, dtype=torch.float64, device="cuda")
    D = torch.zeros(64, dtype=torch.complex128, device="cuda")
    P = torch.zeros((2, 128), dtype=torch.complex128, device="cuda")
    with pytest.raises(binding.EighError):
        eng.tdslda_rhs((4, 4, 5), K[0], K[1], K[2], V, D, 0.0, P)          # grid does not match N
    with pytest.raises(binding.EighError):
        eng.tdslda_rhs((4, 4, 4), K[0], K[1], K[2], V, D, 0.0, P, P)       # aliasing
    eng.close()
