"""GPU parity of eigh_densities (Eq. 16a, 16d, 17) against oracle/densities.py,
element by element on the same seeded inputs, through the C ABI.

Tolerance (derived from the arithmetic): both sides sum k = (active columns) products; any order of
summation differs from the exact sum by at most k eps sum_j |t_j(r)|, and |t_j| <= 2 (|u_j(r)|^2 + |v_j(r)|^2) for
the terms of n, <= (|u|^2 + |v|^2)/2 for those of nu.  Hence |gpu - oracle| <= 4 k eps S(r), S(r) = sum_j |u_j(r)|^2 +
|v_j(r)|^2, plus the rounding of the Fermi factors (a few eps, relative) which the same bound absorbs."""
import numpy as np
import pytest
import torch

import oracle
from oracle import densities as od
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu
EPS = np.finfo(np.float64).eps


def _random_states(M, ncols, seed):
    """Seeded stand-ins for quasiparticle states: unit columns, energies of both signs, one exactly zero."""
    rng = np.random.default_rng(seed)
    Z = rng.standard_normal((2 * M, ncols)) + 1j * rng.standard_normal((2 * M, ncols))
    Z /= np.maximum(np.linalg.norm(Z, axis=0), 1e-300)[None, :]
    E = rng.uniform(-2.0, 2.0, ncols)
    if ncols > 3:
        E[3] = 0.0
    return E, Z


def _gpu_densities(N, E, Z, ldz=None, **kw):
    from paper_2310_03341_b200 import binding
    ncols = Z.shape[1]
    ldz = N if ldz is None else ldz
    Zt = torch.zeros((max(ncols, 1), ldz), dtype=torch.complex128, device="cuda")
    if ncols:
        Zt[:ncols, :N] = torch.from_numpy(np.ascontiguousarray(Z.T)).cuda()
    Ed = torch.from_numpy(np.ascontiguousarray(E)).cuda() if ncols else torch.zeros(1, dtype=torch.float64, device="cuda")
    eng = binding.Eigh(N)
    n, nu = eng.densities(Ed, Zt[:ncols, :N] if ncols else Zt[:0, :N], **kw)
    torch.cuda.synchronize()
    eng.close()
    return n.cpu().numpy(), nu.cpu().numpy()


def _bound(Z, k):
    M = Z.shape[0] // 2
    S = (np.abs(Z[:M]) ** 2 + np.abs(Z[M:]) ** 2).sum(axis=1) if Z.shape[1] else np.zeros(M)
    return 4.0 * max(k, 1) * EPS * S + 1e-300


@pytest.mark.parametrize("M,ncols", [(1, 2), (5, 1), (77, 7), (128, 8), (129, 9), (300, 333), (1000, 2000), (1, 0), (77, 0)])
@pytest.mark.parametrize("T,Ec", [(0.0, np.inf), (0.3, np.inf), (0.25, 1.1)])
def test_same_states_elementwise(M, ncols, T, Ec):
    """Several row blocks (128 rows each) with a ragged tail, several column chunks with ragged ends, empty input."""
    E, Z = _random_states(M, ncols, 1000 * M + ncols)
    n, nu = _gpu_densities(2 * M, E, Z, T=T, Ec=Ec)
    n_o, nu_o = od.densities(E, Z, T=T, Ec=Ec)
    tol = _bound(Z, ncols)
    assert np.all(np.abs(n - n_o) <= tol), np.abs(n - n_o).max()
    assert np.all(np.abs(nu - nu_o) <= tol), np.abs(nu - nu_o).max()
    if ncols == 0:
        assert not n.any() and not nu.any()


@pytest.mark.parametrize("T", [0.0, 0.4])
def test_negative_branch_and_leading_dimension(T):
    """branch = -1 against the oracle applied to the explicitly mapped states [-conj(v), conj(u)]; ldz > N."""
    M, ncols = 211, 150
    E, Z = _random_states(M, ncols, 77)
    n, nu = _gpu_densities(2 * M, E, Z, ldz=2 * M + 6, T=T, Ec=1.5, branch=-1)
    n_o, nu_o = od.densities(*od.particle_hole_map(E, Z), T=T, Ec=1.5)
    tol = _bound(Z, ncols)
    assert np.all(np.abs(n - n_o) <= tol) and np.all(np.abs(nu - nu_o) <= tol)


def test_reproducible_bit_for_bit():
    E, Z = _random_states(700, 1200, 5)
    a = _gpu_densities(1400, E, Z, T=0.2)
    b = _gpu_densities(1400, E, Z, T=0.2)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_argument_errors():
    from paper_2310_03341_b200 import binding
    E = torch.zeros(4, dtype=torch.float64, device="cuda")
    Zt = torch.zeros((4, 6), dtype=torch.complex128, device="cuda")
    eng = binding.Eigh(6)
    for kw in ({"T": -1.0}, {"branch": 0}, {"Ec": float("nan")}):
        with pytest.raises(binding.EighError):
            eng.densities(E, Zt, **kw)
    eng.close()
    odd = binding.Eigh(7)
    with pytest.raises(binding.EighError):
        odd.densities(E, torch.zeros((4, 7), dtype=torch.complex128, device="cuda"))
    odd.close()


def _solve_gpu(H, nev=None):
    from paper_2310_03341_b200 import binding
    N = H.shape[0]
    At = torch.from_numpy(np.ascontiguousarray(H.T)).cuda()
    eng = binding.Eigh(N, nev)
    W, Zt = eng.solve(At)
    return eng, W, Zt


@pytest.mark.parametrize("T", [0.0, 0.2])
def test_pipeline_uniform_bcs_closed_form(T):
    """Config 0 (8x8x8, N = 1024) end to end on the GPU: eigh_solve then eigh_densities reproduce the BCS sums
    n = (1/M) sum_k [1 - xi_k/E_k tanh(E_k/2T)], nu = (1/M) sum_k Delta/(2 E_k) tanh(E_k/2T) (uniform in r).
    Degenerate shells: the densities are invariant under the rotation of the basis inside a shell."""
    shape, mu, delta = (8, 8, 8), 0.5, 0.2 * np.exp(0.4j)
    p = wl.bdg_uniform(shape, mu, delta)
    eng, W, Zt = _solve_gpu(p.dense())
    n, nu = eng.densities(W, Zt, T=T)
    torch.cuda.synchronize()
    eng.close()
    ks = [2 * np.pi * np.arange(-(L // 2), L - L // 2) / L for L in shape]
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    xi = 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1) - mu
    Ek = np.sqrt(xi ** 2 + abs(delta) ** 2)
    th = np.ones_like(Ek) if T == 0 else np.tanh(Ek / (2 * T))
    assert np.abs(n.cpu().numpy() - (1 - xi / Ek * th).mean()).max() <= 1e-11
    assert np.abs(nu.cpu().numpy() - (delta / (2 * Ek) * th).mean()).max() <= 1e-11


def test_pipeline_vortex_vs_oracle_and_branches():
    """Vortex-tangle BdG (6x6x8, N = 576): GPU solve + GPU densities against oracle solve + oracle densities (the
    eigenvectors differ by phases: the densities do not); the lowest N/2 pairs with branch = -1 give the same fields."""
    p = wl.bdg_vortex_tangle((6, 6, 8), 3, 1.0, wl.SEED_BASE + 3, 0.02)
    H = p.dense()
    N = H.shape[0]
    Wo, Zo = oracle.eigh(H)
    for T in (0.0, 0.15):
        n_o, nu_o = od.densities(Wo, Zo, T=T, Ec=6.0)
        eng, W, Zt = _solve_gpu(H)
        n, nu = eng.densities(W, Zt, T=T, Ec=6.0)
        torch.cuda.synchronize()
        eng.close()
        assert np.abs(n.cpu().numpy() - n_o).max() <= 1e-10
        assert np.abs(nu.cpu().numpy() - nu_o).max() <= 1e-10
        eng, W, Zt = _solve_gpu(H, nev=N // 2)
        n2, nu2 = eng.densities(W, Zt, T=T, Ec=6.0, branch=-1)
        torch.cuda.synchronize()
        eng.close()
        assert np.abs(n2.cpu().numpy() - n_o).max() <= 1e-10
        assert np.abs(nu2.cpu().numpy() - nu_o).max() <= 1e-10


# ----------------------------------------------------------------------------- Eq. 16b, 16c: tau(r), j(r)
def _gpu_gradient_densities(shape, Ds, E, Z, **kw):
    from paper_2310_03341_b200 import binding
    N = 2 * int(np.prod(shape))
    ncols = Z.shape[1]
    Zt = torch.from_numpy(np.ascontiguousarray(Z.T)).cuda() if ncols else torch.zeros((0, N), dtype=torch.complex128, device="cuda")
    Ed = torch.from_numpy(np.ascontiguousarray(E)).cuda() if ncols else torch.zeros(1, dtype=torch.float64, device="cuda")
    Dd = [torch.from_numpy(np.ascontiguousarray(D.T)).cuda() for D in Ds]      # column-major storage of D
    eng = binding.Eigh(N)
    tau, j = eng.gradient_densities(shape, Dd[0], Dd[1], Dd[2], Ed, Zt, **kw)
    torch.cuda.synchronize()
    eng.close()
    return tau.cpu().numpy(), j.cpu().numpy()


def _grad_tolerances(E, Z, shape, Ds, k):
    """Both sides sum k states of products whose factors are L-term sums: |gpu - oracle| <= 8 (k + 2 L) eps S with
    S >= sum_j |term_j|: for tau S = 2 max_r sum_j |grad u|^2 + |grad v|^2 (= 2 tau at f = 1/2, weights <= 2); for j the
    Cauchy-Schwarz bound 2 sqrt(max_r sum |w|^2 * max_r sum |grad w|^2)."""
    L = max(shape)
    if Z.shape[1] == 0:
        return 1e-300, 1e-300
    Eall = np.ones(Z.shape[1])
    t_inf, _ = od.gradient_densities(Eall, Z, shape, *Ds, T=1e12)      # = sum_j |grad u|^2 + |grad v|^2
    n_inf, _ = od.densities(Eall, Z, T=1e12)                           # = sum_j |u|^2 + |v|^2
    c = 8.0 * (k + 2 * L) * EPS
    return c * 2.0 * t_inf.max(), c * 2.0 * np.sqrt(t_inf.max() * n_inf.max())


@pytest.mark.parametrize("shape,ncols", [((1, 1, 2), 3), ((3, 5, 7), 40), ((8, 8, 8), 333), ((6, 10, 9), 1080), ((2, 33, 3), 17),
                                         ((4, 4, 6), 0), ((9, 1, 40), 100)])
@pytest.mark.parametrize("T,Ec", [(0.0, np.inf), (0.3, 1.1)])
def test_gradient_densities_elementwise(shape, ncols, T, Ec):
    """Distinct, non-antisymmetric random 1-D matrices (a transposed or swapped matrix shows); tiles with ragged ends
    along every axis (lines not a multiple of 32), L from 1 to 40, empty input."""
    M = int(np.prod(shape))
    rng = np.random.default_rng(M + ncols)
    Ds = [wl.derivative_1d(L) + 0.1 * rng.standard_normal((L, L)) for L in shape]
    E, Z = _random_states(M, ncols, 31 * M + ncols)
    tau, j = _gpu_gradient_densities(shape, Ds, E, Z, T=T, Ec=Ec)
    tau_o, j_o = od.gradient_densities(E, Z, shape, *Ds, T=T, Ec=Ec)
    tt, tj = _grad_tolerances(E, Z, shape, Ds, ncols)
    assert np.abs(tau - tau_o).max() <= tt, (np.abs(tau - tau_o).max(), tt)
    assert np.abs(j - j_o).max() <= tj, (np.abs(j - j_o).max(), tj)
    if ncols == 0:
        assert not tau.any() and not j.any()


def test_gradient_densities_negative_branch():
    shape, ncols = (5, 6, 7), 150
    M = int(np.prod(shape))
    Ds = [wl.derivative_1d(L) for L in shape]
    E, Z = _random_states(M, ncols, 99)
    tau, j = _gpu_gradient_densities(shape, Ds, E, Z, T=0.2, Ec=1.5, branch=-1)
    tau_o, j_o = od.gradient_densities(*od.particle_hole_map(E, Z), shape, *Ds, T=0.2, Ec=1.5)
    tt, tj = _grad_tolerances(E, Z, shape, Ds, ncols)
    assert np.abs(tau - tau_o).max() <= tt and np.abs(j - j_o).max() <= tj


def test_pipeline_moving_condensate_current():
    """Delta = D0 exp(2 i q r) on a 5x5x7 grid, end to end on the GPU (assemble -> solve -> gradient densities) against
    the oracle chain; the current is uniform, along q, and j_y = 0 (closed form pinned in test_oracle_densities.py)."""
    from paper_2310_03341_b200 import binding
    shape = (5, 5, 7)
    nx, ny, nz = shape
    M = nx * ny * nz
    X, Y, Zc = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    Delta = 0.3 * np.exp(2j * (2 * np.pi / nx * X + 2 * 2 * np.pi / nz * Zc)).reshape(-1)
    p = wl.BdGProblem("moving", shape, 0.9, np.zeros(M), Delta)
    Ds = [wl.derivative_1d(L) for L in shape]
    Wo, Zo = oracle.eigh(p.dense())
    tau_o, j_o = od.gradient_densities(Wo, Zo, shape, *Ds, T=0.0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()   # noqa: E731
    eng = binding.Eigh(2 * M)
    At = eng.assemble_bdg(shape, *[dev(wl.kinetic_1d(L)) for L in shape], dev(p.V), dev(p.Delta), p.mu)
    W, Zt = eng.solve(At)
    tau, j = eng.gradient_densities(shape, *[dev(D.T) for D in Ds], W, Zt, T=0.0)
    torch.cuda.synchronize()
    eng.close()
    assert np.abs(tau.cpu().numpy() - tau_o).max() <= 1e-10
    assert np.abs(j.cpu().numpy() - j_o).max() <= 1e-10
    jn = j.cpu().numpy()
    assert np.abs(jn[1]).max() <= 1e-10 and np.abs(jn[0]).min() > 1e-3 and np.abs(jn[0] - jn[0].mean()).max() <= 1e-10
