"""Pins of oracle/assemble.py (SURVEY.md 8(f)1 prologue; Eq. 5/7/8): the Kronecker-product
definition against an independently written triplet assembly (the seeded input generator), against the closed-form
spectra the structure implies, and against the block symmetries of Eq. 7."""
import numpy as np

from oracle import assemble as oa
from paper_2310_03341_b200 import workloads as wl


def _fields(shape, seed):
    rng = np.random.default_rng(seed)
    M = int(np.prod(shape))
    V = rng.uniform(-0.3, 0.3, M)
    Delta = rng.standard_normal(M) + 1j * rng.standard_normal(M)
    return V, Delta


def test_matches_the_independent_triplet_assembly():
    """workloads.BdGProblem.dense() scatters COO triplets axis by axis; the oracle builds Kronecker products."""
    shape = (3, 4, 5)
    V, Delta = _fields(shape, 1)
    p = wl.BdGProblem("t", shape, 0.7, V, Delta)
    Ks = [wl.kinetic_1d(L) for L in shape]
    H = oa.assemble_bdg(*Ks, V, Delta, 0.7)
    Hw = p.dense()
    # off-diagonal entries are single terms (exact); the diagonal sums four terms in a different order
    off = ~np.eye(H.shape[0], dtype=bool)
    assert np.array_equal(H[off], Hw[off])
    assert np.abs(np.diag(H) - np.diag(Hw)).max() <= 4 * np.finfo(float).eps * np.abs(np.diag(Hw)).max()
    assert np.array_equal(oa.assemble_bdg(*Ks, V, Delta, 0.7, sign=-1.0), -H)


def test_kinetic_spectrum_is_the_sum_of_the_axis_spectra():
    """V = 0, Delta = 0, mu = 0: H = diag(T, -T) and T = sum of commuting 1-D operators, so its eigenvalues are all
    sums k_x^2/2 + k_y^2/2 + k_z^2/2 on the grid of PAPER.md:113 (closed form, evaluated by a library eigvalsh)."""
    shape = (4, 3, 6)
    Ks = [wl.kinetic_1d(L) for L in shape]
    M = int(np.prod(shape))
    H = oa.assemble_bdg(*Ks, np.zeros(M), np.zeros(M), 0.0)
    ks = [2 * np.pi * np.arange(-(L // 2), L - L // 2) / L for L in shape]
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    eps = 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1)
    ref = np.sort(np.concatenate([eps, -eps]))
    assert np.abs(np.linalg.eigvalsh(H) - ref).max() <= 1e-12


def test_block_structure_and_symmetries():
    """Eq. 7: Hermitian; lower-right block = -conj(upper-left); pairing blocks diagonal and mutually adjoint;
    particle-hole symmetry S conj(H) S^-1 = -H with S = [[0, -I], [I, 0]]; the index convention r = (ix Ny + iy) Nz + iz
    (a potential placed at one grid point lands on that diagonal entry; a z-neighbour couples through Kz only)."""
    shape = (2, 3, 4)
    M = int(np.prod(shape))
    V, Delta = _fields(shape, 2)
    Ks = [wl.kinetic_1d(L) + 0.01 * np.diag(np.arange(L)) for L in shape]      # distinct, non-circulant: no accidental symmetry
    H = oa.assemble_bdg(*Ks, V, Delta, 0.3)
    assert np.array_equal(H, H.conj().T)
    assert np.array_equal(H[M:, M:], -np.conj(H[:M, :M]))
    assert np.array_equal(H[:M, M:], np.diag(Delta)) and np.array_equal(H[M:, :M], np.diag(np.conj(Delta)))
    S = np.block([[np.zeros((M, M)), -np.eye(M)], [np.eye(M), np.zeros((M, M))]])
    assert np.abs(S @ np.conj(H) @ S.T + H).max() == 0.0
    ix, iy, iz = 1, 2, 1
    r = (ix * shape[1] + iy) * shape[2] + iz
    e = np.zeros(M); e[r] = 1.0
    dH = oa.assemble_bdg(*Ks, V + e, Delta, 0.3) - H
    assert dH[r, r] == 1.0 and dH[M + r, M + r] == -1.0 and np.count_nonzero(dH) == 2
    r2 = (ix * shape[1] + iy) * shape[2] + (iz + 2)
    assert H[r, r2] == Ks[2][iz, iz + 2]
    r3 = ((ix - 1) * shape[1] + iy) * shape[2] + iz
    assert H[r, r3] == Ks[0][ix, ix - 1]
    r4 = (ix * shape[1] + (iy - 2)) * shape[2] + iz
    assert H[r, r4] == Ks[1][iy, iy - 2]
    r5 = ((ix - 1) * shape[1] + iy) * shape[2] + (iz + 1)
    assert H[r, r5] == 0.0
