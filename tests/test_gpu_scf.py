"""GPU parity of eigh_assemble_bdg (SURVEY.md 8(f)1 prologue; Eq. 5/7/8) against oracle/assemble.py,
bit for bit, and one closed iteration of the paper's self-consistent loop (Eq. 18b) on the GPU:
fields -> H (eigh_assemble_bdg) -> eigenpairs (eigh_solve) -> densities (eigh_densities) -> fields."""
import numpy as np
import pytest
import torch

import oracle
from oracle import assemble as oa
from oracle import densities as od
from paper_2310_03341_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _assemble_gpu(shape, Ks, V, Delta, mu, sign=1.0, eng=None):
    from paper_2310_03341_b200 import binding
    N = 2 * int(np.prod(shape))
    own = eng is None
    eng = binding.Eigh(N) if own else eng
    At = eng.assemble_bdg(shape, _dev(Ks[0]), _dev(Ks[1]), _dev(Ks[2]), _dev(V), _dev(Delta), mu, sign=sign)
    torch.cuda.synchronize()
    if own:
        eng.close()
    return At


@pytest.mark.parametrize("shape", [(1, 1, 1), (2, 3, 4), (5, 3, 7), (8, 8, 8), (6, 10, 9)])
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_assemble_bit_exact(shape, sign):
    """Every element of H, both triangles; sizes with ragged row blocks (256) and column groups (16); non-circulant,
    distinct 1-D matrices so that a swapped axis or a transposed index shows."""
    rng = np.random.default_rng(sum(shape))
    M = int(np.prod(shape))
    V = rng.uniform(-0.3, 0.3, M)
    Delta = rng.standard_normal(M) + 1j * rng.standard_normal(M)
    Ks = []
    for L in shape:
        K = wl.kinetic_1d(L) + 0.01 * rng.standard_normal((L, L))
        Ks.append(0.5 * (K + K.T))
    H = _assemble_gpu(shape, Ks, V, Delta, 0.37, sign).cpu().numpy().T      # storage is column-major
    Ho = oa.assemble_bdg(*Ks, V, Delta, 0.37, sign)
    assert np.array_equal(H, Ho)


def test_assemble_matches_the_bench_generator_at_config2_size():
    """Config 2 (16^3, N = 8192): the kernel against workloads.dense_torch (the generator bench.py uses), on the device.
    Off-diagonal entries are single terms (exact); the diagonal sums four terms in a different order (<= 4 ulp)."""
    w = wl.make_config(2)
    p = w.problem
    Ks = [wl.kinetic_1d(L) for L in p.shape]
    At = _assemble_gpu(p.shape, Ks, p.V, p.Delta, p.mu)
    Ht = torch.empty_like(At)
    w.dense_torch("cuda", out=Ht)
    diff = (At - Ht).abs()
    dmax = float(torch.diagonal(diff).max().item())
    diff.fill_diagonal_(0.0)
    assert float(diff.max().item()) == 0.0
    assert dmax <= 4 * np.finfo(float).eps * float(torch.diagonal(Ht).abs().max().item())


def test_one_scf_iteration_against_the_oracle_chain():
    """fields -> H -> (E, phi) -> (n, nu) on the GPU against the same chain in the oracle (vortex fields, 4x4x6)."""
    p = wl.bdg_vortex_tangle((4, 4, 6), 3, 1.0, wl.SEED_BASE + 3, 0.02)
    Ks = [wl.kinetic_1d(L) for L in p.shape]
    from paper_2310_03341_b200 import binding
    eng = binding.Eigh(p.N)
    At = _assemble_gpu(p.shape, Ks, p.V, p.Delta, p.mu, eng=eng)
    W, Zt = eng.solve(At)
    n, nu = eng.densities(W, Zt, T=0.05)
    torch.cuda.synchronize()
    eng.close()
    Ho = oa.assemble_bdg(*Ks, p.V, p.Delta, p.mu)
    Wo, Zo = oracle.eigh(Ho)
    n_o, nu_o = od.densities(Wo, Zo, T=0.05)
    assert np.abs(W.cpu().numpy() - Wo).max() <= 1e-11 * np.abs(Wo).max()
    assert np.abs(n.cpu().numpy() - n_o).max() <= 1e-10
    assert np.abs(nu.cpu().numpy() - nu_o).max() <= 1e-10


def test_scf_loop_converges_to_the_bcs_gap():
    """Toy functional Delta = g nu (Eq. 18b with a constant coupling), uniform fields on the 8x8x8 lattice: the loop
    assemble -> solve -> densities -> Delta = g nu is the fixed-point iteration of the BCS gap equation
    1 = (g/M) sum_k 1 / (2 E_k).  With g chosen so that Delta* = 0.2 e^{0.3 i} solves it, the GPU loop started from
    0.35 e^{0.3 i} converges to Delta* linearly (the phase is preserved by the map, the modulus contracts)."""
    from paper_2310_03341_b200 import binding
    shape, mu = (8, 8, 8), 0.5
    M = int(np.prod(shape))
    target = 0.2 * np.exp(0.3j)
    ks = [2 * np.pi * np.arange(-(L // 2), L - L // 2) / L for L in shape]
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    xi = 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1) - mu
    g = 1.0 / (1.0 / (2.0 * np.sqrt(xi ** 2 + abs(target) ** 2))).mean()
    Ks = [_dev(wl.kinetic_1d(L)) for L in shape]
    V = torch.zeros(M, dtype=torch.float64, device="cuda")
    Delta = torch.full((M,), 0.35 * np.exp(0.3j), dtype=torch.complex128, device="cuda")
    eng = binding.Eigh(2 * M)
    At = None
    hist = []
    for it in range(60):
        At = eng.assemble_bdg(shape, Ks[0], Ks[1], Ks[2], V, Delta, mu, At=At)
        W, Zt = eng.solve(At)
        n, nu = eng.densities(W, Zt, T=0.0)
        Delta = (g * nu).contiguous()
        hist.append(abs(complex(Delta.mean().item()) - target))
        if hist[-1] < 1e-12:
            break
    torch.cuda.synchronize()
    eng.close()
    D = Delta.cpu().numpy()
    assert np.abs(D - D.mean()).max() <= 1e-12              # stays uniform
    assert hist[-1] <= 1e-7, hist[-5:]                      # linear convergence, rate ~0.77 per iteration
    assert all(b < a for a, b in zip(hist, hist[1:]))       # monotone: every iteration contracts
