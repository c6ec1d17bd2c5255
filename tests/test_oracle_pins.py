"""Pins of the CPU oracle against what the paper and the mathematics fix
(SURVEY.md 8(c) "What pins each part").  None of these re-type the oracle's formulas:
they are closed forms, invariants, brute force on tiny inputs, or an independent library.
"""
import itertools

import numpy as np
import pytest

import oracle
from paper_2310_03341_b200 import workloads as wl

EPS = np.finfo(np.float64).eps


# ----------------------------------------------------------------------------- helpers
def bdg_uniform_closed_form(shape, mu, delta):
    """Eq. 7 with uniform Delta is block-diagonal 2x2 in the plane-wave basis:
    E = +/- sqrt((eps_k - mu)^2 + |Delta|^2), eps_k = |k|^2/2, k = 2 pi n/N, n in {-N/2..N/2-1}
    (PAPER.md:113)."""
    ks = []
    for L in shape:
        n = np.arange(-(L // 2), L - L // 2)
        ks.append(2 * np.pi * n / L)
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    eps_k = 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1)
    E = np.sqrt((eps_k - mu) ** 2 + abs(delta) ** 2)
    return np.sort(np.concatenate([-E, E]))


def residual(H, W, Z):
    n = H.shape[0]
    return np.linalg.norm(H @ Z - Z * W[None, :]) / (np.linalg.norm(H) * np.sqrt(n))


def orth(Z):
    return np.abs(Z.conj().T @ Z - np.eye(Z.shape[1])).max()


def rand_herm(n, seed):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    return 0.5 * (A + A.conj().T)


# ----------------------------------------------------------------------------- whole solve
def test_config0_closed_form_spectrum_small():
    """4x4x4 lattice (N=128): all eigenvalues equal the closed form; heavy degeneracy."""
    p = wl.bdg_uniform((4, 4, 4), 0.5, 0.2)
    H = p.dense()
    W, Z = oracle.eigh(H)
    ref = bdg_uniform_closed_form((4, 4, 4), 0.5, 0.2)
    nrm = np.abs(ref).max()
    assert np.abs(W - ref).max() <= 1e-12 * nrm
    assert residual(H, W, Z) <= 1e-14
    assert orth(Z) <= 1e-12


def test_config0_closed_form_spectrum_full():
    """Config 0 (8x8x8, N=1024): the pin of SURVEY.md 8(c): 1024 eigenvalues, 64 distinct."""
    w = wl.make_config(0)
    H = w.dense()
    assert np.abs(H - H.conj().T).max() == 0.0
    W, Z = oracle.eigh(H)
    ref = bdg_uniform_closed_form((8, 8, 8), 0.5, 0.2)
    nrm = np.abs(ref).max()
    assert abs(nrm - 14.306) < 1e-2          # ||H||_2 quoted in SURVEY.md 8(c)
    assert len(np.unique(np.round(ref, 9))) == 64
    assert np.abs(W - ref).max() <= 1e-11 * nrm
    assert residual(H, W, Z) <= 1e-13
    assert orth(Z) <= 1e-12 * 1024
    # each eigenvector lies in the span of the plane-wave 2-spinors of its energy shell:
    # project on the eigenspace of the closed-form shell built from plane waves.
    n = 512
    ks = [2 * np.pi * np.arange(-4, 4) / 8] * 3
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    eps_k = 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1)
    X, Y, Zc = wl.grid_coords((8, 8, 8))
    kv = np.stack([KX.reshape(-1), KY.reshape(-1), KZ.reshape(-1)], 1)
    pw = np.exp(1j * (np.outer(X, kv[:, 0]) + np.outer(Y, kv[:, 1]) + np.outer(Zc, kv[:, 2]))) / np.sqrt(n)
    Ek = np.sqrt((eps_k - 0.5) ** 2 + 0.04)
    for j in (0, 17, 300, 511, 512, 700, 1023):
        shell = np.abs(Ek - abs(W[j])) < 1e-8
        B = pw[:, shell]                                   # plane waves of this shell
        u, v = Z[:n, j], Z[n:, j]
        pu = B @ (B.conj().T @ u)
        pv = B @ (B.conj().T @ v)
        assert np.linalg.norm(pu) ** 2 + np.linalg.norm(pv) ** 2 >= 1 - 1e-10


def test_prescribed_spectrum_with_clusters():
    """Config-1 recipe at N=300: the computed spectrum equals the prescribed one."""
    A, lam = wl.random_hermitian_clustered(300, wl.SEED_BASE + 1)
    W, Z = oracle.eigh(A)
    assert np.abs(W - lam).max() <= 300 * EPS * 4
    assert residual(A, W, Z) <= 1e-14
    assert orth(Z) <= 1e-12


@pytest.mark.parametrize("n", [1, 2])
def test_tiny_closed_form(n):
    rng = np.random.default_rng(5 + n)
    if n == 1:
        H = np.array([[rng.standard_normal() + 0j]])
        W, Z = oracle.eigh(H)
        assert W[0] == H[0, 0].real and abs(abs(Z[0, 0]) - 1) < 1e-15
        return
    a, d = rng.standard_normal(2)
    b = rng.standard_normal() + 1j * rng.standard_normal()
    H = np.array([[a, np.conj(b)], [b, d]])
    W, Z = oracle.eigh(H)
    mid, rad = (a + d) / 2, np.sqrt(((a - d) / 2) ** 2 + abs(b) ** 2)
    assert np.allclose(W, [mid - rad, mid + rad], rtol=0, atol=4 * EPS * (abs(mid) + rad))
    assert residual(H, W, Z) <= 1e-15 and orth(Z) <= 1e-15


def faddeev_leverrier(H):
    """Coefficients c_k of det(x I - H) = x^n + c_1 x^(n-1) + ... + c_n."""
    n = H.shape[0]
    M = np.zeros_like(H)
    c = [1.0]
    for k in range(1, n + 1):
        M = H @ M + c[-1] * np.eye(n)
        c.append(-np.trace(H @ M).real / k)
    return np.array(c)


@pytest.mark.parametrize("n", [3, 4])
def test_tiny_characteristic_polynomial(n):
    """Brute force: elementary symmetric functions of the computed eigenvalues equal the
    characteristic-polynomial coefficients; det(H - lambda_i I) ~ 0."""
    for seed in range(4):
        H = rand_herm(n, 100 * n + seed)
        W = oracle.eigh(H, vectors=False)
        c = faddeev_leverrier(H)
        scale = np.abs(W).max()
        for k in range(1, n + 1):
            ek = sum(np.prod(cmb) for cmb in itertools.combinations(W, k))
            assert abs((-1) ** k * ek - c[k]) <= 50 * EPS * scale ** k * n
        for i in range(n):
            det = np.linalg.det(H - W[i] * np.eye(n))
            others = np.prod([abs(W[i] - W[j]) for j in range(n) if j != i])
            assert abs(det) <= 200 * EPS * scale * max(others, EPS) * n


# ----------------------------------------------------------------------------- O1..O3
@pytest.mark.parametrize("n", [2, 3, 7, 40, 129])
def test_tridiagonalisation_invariants(n):
    H = rand_herm(n, 7 * n)
    d, e, Q = oracle.tridiagonalise(H)
    T = np.diag(d) + np.diag(e, -1) + np.diag(e, 1)
    nH = np.linalg.norm(H)
    assert np.all(e >= 0)
    assert np.linalg.norm(Q.conj().T @ H @ Q - T) <= 20 * n * EPS * nH
    assert np.abs(Q.conj().T @ Q - np.eye(n)).max() <= 20 * n * EPS
    assert abs(d.sum() - np.trace(H).real) <= 20 * n * EPS * nH
    assert abs(np.sum(d ** 2) + 2 * np.sum(e ** 2) - nH ** 2) <= 40 * n * EPS * nH ** 2


def test_tridiagonalisation_reads_lower_triangle_only():
    H = rand_herm(12, 3)
    G = H.copy()
    G[np.triu_indices(12, 1)] = 99.0 + 5j          # garbage above the diagonal
    G[np.diag_indices(12)] += 3j                   # garbage imaginary diagonal
    W0 = oracle.eigh(H, vectors=False)
    W1 = oracle.eigh(G, vectors=False)
    assert np.array_equal(W0, W1)


def test_already_tridiagonal_and_diagonal_inputs():
    """nu = 0 branch of O1 (no reflector) and a zero subdiagonal."""
    D = np.diag([3.0, -1.0, 2.0, 2.0, 0.5]).astype(np.complex128)
    W, Z = oracle.eigh(D)
    assert np.array_equal(W, np.sort(np.diag(D).real))
    assert orth(Z) <= 1e-15
    T = np.diag([1.0, 2, 3, 4]) + np.diag([1j, 0, -2.0], -1)
    T = T + np.tril(T, -1).conj().T
    W, Z = oracle.eigh(T)
    assert residual(T, W, Z) <= 1e-15


# ----------------------------------------------------------------------------- O4 (QL)
@pytest.mark.parametrize("n", [1, 2, 5, 64, 257])
def test_ql_toeplitz_121(n):
    """d=2, e=-1: lambda_k = 2 - 2 cos(k pi/(n+1)); eigenvectors sqrt(2/(n+1)) sin(i k pi/(n+1))."""
    d = np.full(n, 2.0)
    e = np.full(n - 1, -1.0)
    W, Q = oracle.tridiag_ql(d, e)
    k = np.arange(1, n + 1)
    ref = 2 - 2 * np.cos(k * np.pi / (n + 1))
    assert np.abs(W - ref).max() <= 8 * n * EPS
    i = np.arange(1, n + 1)
    V = np.sqrt(2 / (n + 1)) * np.sin(np.outer(i, k) * np.pi / (n + 1))
    # eigenvalues are simple: compare up to sign
    dots = np.abs(np.sum(V * Q, axis=0))
    gap = np.min(np.diff(ref)) if n > 1 else 1.0
    assert np.abs(dots - 1).max() <= 100 * n * EPS / min(gap, 1.0)


@pytest.mark.parametrize("n", [2, 9, 50, 101])
def test_ql_clement_integer_spectrum(n):
    """Clement/Kac: d=0, e_i = sqrt(i (n-i)), i=1..n-1: lambda = -(n-1), -(n-3), ..., n-1."""
    i = np.arange(1, n)
    W, Q = oracle.tridiag_ql(np.zeros(n), np.sqrt(i * (n - i)))
    ref = np.arange(-(n - 1), n, 2).astype(float)
    assert np.abs(W - ref).max() <= 10 * n * EPS * n
    assert np.abs(Q.T @ Q - np.eye(n)).max() <= 50 * n * EPS


def test_ql_wilkinson_pairs():
    """Wilkinson W+_21: d = |i - 10|, e = 1. Largest eigenvalues come in pairs agreeing to
    ~1e-14 (textbook value 10.746194182903...)."""
    m = 10
    d = np.abs(np.arange(-m, m + 1)).astype(float)
    e = np.ones(2 * m)
    W, Q = oracle.tridiag_ql(d, e)
    Wl = oracle.tridiag_ql_ld(d, e, vectors=False)
    assert abs(W[-1] - 10.746194182903) < 2e-12
    assert 0 < W[-1] - W[-2] < 1e-12
    assert np.abs(W - Wl).max() <= 50 * EPS * 11
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    assert np.linalg.norm(T @ Q - Q * W[None, :]) <= 100 * EPS * 11 * np.sqrt(21)
    assert np.abs(Q.T @ Q - np.eye(21)).max() <= 200 * EPS


def test_ql_glued_and_constant():
    """Glued copies with tiny couplings (cluster stress) and d = const, e = 0 (nothing to do)."""
    base_d = np.array([1.0, 2.0, 3.0, 4.0, 5.0])
    base_e = np.array([0.5, 0.25, 0.5, 1.0])
    d = np.tile(base_d, 6)
    e = []
    for c, glue in enumerate([1e-8, 1e-10, 1e-12, 1e-14, 0.0]):
        e.extend(base_e); e.append(glue)
    e.extend(base_e)
    e = np.array(e)
    W, Q = oracle.tridiag_ql(d, e)
    T = np.diag(d) + np.diag(e, 1) + np.diag(e, -1)
    assert np.linalg.norm(T @ Q - Q * W[None, :]) <= 200 * EPS * 6 * np.sqrt(30)
    assert np.abs(Q.T @ Q - np.eye(30)).max() <= 200 * EPS
    Wb = oracle.tridiag_ql(base_d, base_e, vectors=False)
    assert np.abs(W.reshape(5, 6) - Wb[:, None]).max() <= 1e-7     # glue perturbs by <= 1e-8
    W, Q = oracle.tridiag_ql(np.full(9, 2.5), np.zeros(8))
    assert np.array_equal(W, np.full(9, 2.5)) and np.array_equal(Q, np.eye(9))


# ----------------------------------------------------------------------------- precision, symmetry
def test_long_double_agreement():
    n = 200
    H = rand_herm(n, 42)
    W = oracle.eigh(H, vectors=False)
    Wl, Zl = oracle.eigh_ld(H)
    nrm = np.abs(Wl).max()
    assert np.abs(W - Wl).max() <= 10 * n * EPS * nrm
    assert residual(H, Wl, Zl) <= 5 * EPS          # long-double result rounded to FP64


def test_particle_hole_symmetry_vortex():
    """BdG with a vortex tangle (small lattice): H Hermitian, lambda_i = -lambda_{N-1-i}
    (S H^* S^-1 = -H since Delta is diagonal), and (u,v) -> (-v^*, u^*) maps E to -E."""
    p = wl.bdg_vortex_tangle((4, 4, 6), 3, 1.0, wl.SEED_BASE + 3, 0.02)
    H = p.dense()
    assert np.abs(H - H.conj().T).max() == 0.0
    W, Z = oracle.eigh(H)
    nrm = np.abs(W).max()
    assert np.abs(W + W[::-1]).max() <= 1e-12 * nrm
    n = H.shape[0] // 2
    u, v = Z[:n, 5], Z[n:, 5]
    phi = np.concatenate([-v.conj(), u.conj()])
    assert np.linalg.norm(H @ phi + W[5] * phi) <= 1e-12 * nrm
    assert residual(H, W, Z) <= 1e-14 and orth(Z) <= 1e-12


def test_library_cross_check():
    """Sanity (not truth): LAPACK via numpy on the config-2 recipe at 6x6x4."""
    p = wl.bdg_single_vortex((6, 6, 4), 1.0, wl.SEED_BASE + 2)
    H = p.dense()
    W = oracle.eigh(H, vectors=False)
    Wn = np.linalg.eigvalsh(H)
    assert np.abs(W - Wn).max() <= 1e-12 * np.abs(Wn).max()
    assert abs(W.sum() - np.trace(H).real) <= 1e-11
    assert abs(np.sum(W ** 2) - np.linalg.norm(H) ** 2) <= 1e-10 * np.linalg.norm(H) ** 2


# ----------------------------------------------------------------------------- Sturm count (used by the full-size GPU tests)
def test_sturm_count_against_closed_forms():
    """oracle.sturm_count is pinned by spectra known in closed form: the 1-2-1 Toeplitz matrix
    (lambda_k = 2 - 2 cos(k pi/(n+1))) and the Clement/Kac matrix (integers -(n-1), -(n-3), ..., n-1)."""
    n = 200
    d = np.full(n, 2.0)
    e = np.full(n - 1, -1.0)
    lam = 2.0 - 2.0 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1))
    mids = 0.5 * (lam[:-1] + lam[1:])
    assert np.array_equal(oracle.sturm_count(d, e, mids), np.arange(1, n))
    assert oracle.sturm_count(d, e, -1.0) == 0 and oracle.sturm_count(d, e, 5.0) == n
    n = 51
    i = np.arange(1, n)
    ek = np.sqrt(i * (n - i))
    ints = np.arange(-(n - 1), n, 2).astype(float)
    assert np.array_equal(oracle.sturm_count(np.zeros(n), ek, ints + 0.5), np.arange(1, n + 1))
    assert np.array_equal(oracle.sturm_count(np.zeros(n), ek, ints - 0.5), np.arange(0, n))


def test_sturm_count_matches_oracle_ql_on_random_tridiagonal():
    rng = np.random.default_rng(7)
    n = 300
    d = rng.standard_normal(n)
    e = rng.standard_normal(n - 1)
    W = oracle.tridiag_ql(d, e, vectors=False)
    gaps = np.diff(W)
    ok = gaps > 1e-8
    mids = (0.5 * (W[:-1] + W[1:]))[ok]
    assert np.array_equal(oracle.sturm_count(d, e, mids), (np.arange(1, n))[ok])


# ---- pins for the rows widened in round 2 (the 1-stage and the real-symmetric variants).  The oracle for
# both is O1-O5 itself (PAPER.md:148 steps i-iii executed naively; the real case is the same oracle on a real matrix).
@pytest.mark.parametrize("n", [5, 40, 97])
def test_tridiagonal_form_is_unique_up_to_phases(n):
    """Implicit-Q theorem: with the first column of Q fixed to e_1, the Hermitian tridiagonal form of H has a unique
    diagonal and unique |off-diagonals|.  LAPACK's Hessenberg reduction (scipy, a different code with a different
    reflector convention) must therefore reproduce the oracle's d and e -- the element-wise reference the GPU's
    eigh_tridiagonalise_direct is compared with."""
    import scipy.linalg
    rng = np.random.default_rng(300 + n)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    H = 0.5 * (A + A.conj().T)
    d, e, Q = oracle.tridiagonalise(H)
    Hs = scipy.linalg.hessenberg(H)
    nrm = np.linalg.norm(H, 2)
    assert np.abs(np.diag(Hs).real - d).max() <= 1e-11 * nrm
    assert np.abs(np.abs(np.diag(Hs, -1)) - e).max() <= 1e-11 * nrm
    assert np.abs(np.triu(Hs, 2)).max() <= 1e-12 * nrm           # Hermitian input: the Hessenberg form is tridiagonal


def test_real_symmetric_input_gives_real_eigenvectors():
    """The real-symmetric case of PAPER.md:140 / :158-160 is the same oracle on a real matrix: every step stays in the
    reals (phi = +-1), so Z comes out exactly real and equals the textbook real decomposition; pinned on the closed form
    of the 1-2-1 Toeplitz matrix embedded as a dense matrix and on config 0 (a real BdG matrix)."""
    n = 64
    T = 2.0 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)
    rng = np.random.default_rng(5)
    Qr, _ = np.linalg.qr(rng.standard_normal((n, n)))
    H = Qr @ T @ Qr.T
    H = 0.5 * (H + H.T)
    W, Z = oracle.eigh(H.astype(np.complex128))
    assert np.abs(Z.imag).max() == 0.0
    k = np.arange(1, n + 1)
    assert np.abs(W - (2 - 2 * np.cos(k * np.pi / (n + 1)))).max() <= 1e-13
    Zr = Z.real
    assert np.abs(Zr.T @ Zr - np.eye(n)).max() <= 1e-13
    assert np.linalg.norm(H @ Zr - Zr * W[None, :]) <= 1e-13 * n
    H0 = wl.make_config(0).dense()
    assert np.abs(H0.imag).max() == 0.0                         # config 0 is real-valued
    p = wl.bdg_uniform((4, 4, 4), 0.5, 0.2)
    W4, Z4 = oracle.eigh(p.dense())
    assert np.abs(Z4.imag).max() == 0.0


def test_ql_survives_the_underflow_split():
    """The `r == 0` branch of the QL sweep (a rotation whose two components both underflow: split and restart) is only
    reachable with subnormal data.  These two inputs reach it (found with an instrumented copy of the oracle; integers
    times the smallest subnormal 5e-324, where every product rounds to an integer): no accuracy exists at that scale, so
    the pin is what still must hold -- the routine terminates without failure, returns finite ascending values, and the
    trace, which only involves exact additions there, is preserved.  A division by r = 0 would give NaN."""
    den = 5e-324
    for d, e in (([3, 0, -3, 2], [3, 3, 1]), ([0, -1, -1, -1, 0, 2], [3, 1, 3, 2, 2])):
        dd, ee = np.array(d, dtype=np.float64) * den, np.array(e, dtype=np.float64) * den
        W, Q = oracle.tridiag_ql(dd, ee)
        assert np.isfinite(W).all() and np.isfinite(Q).all()
        assert np.all(np.diff(W) >= 0)
        assert W.sum() == dd.sum()
        # the same matrix scaled into the normal range (exact scaling by 2^1000 / den) is solved to full accuracy
        s = 2.0 ** 1000
        Wn, Qn = oracle.tridiag_ql(np.array(d, dtype=np.float64) * s, np.array(e, dtype=np.float64) * s)
        T = np.diag(np.array(d, float)) + np.diag(np.array(e, float), 1) + np.diag(np.array(e, float), -1)
        assert np.abs(Wn / s - np.linalg.eigvalsh(T)).max() <= 1e-13 * np.abs(T).sum()
        assert np.abs(Qn.T @ Qn - np.eye(len(d))).max() <= 1e-14


@pytest.mark.parametrize("scale", [2.0 ** -333, 2.0 ** 333])
def test_oracle_is_equivariant_under_power_of_two_scaling(scale):
    """Every step of O1-O5 is homogeneous (reflectors, rotations, relative split tests): eigh(s H) = s eigh(H) BIT FOR BIT for a
    power of two s while the squares of the entries stay representable.  A pin for any absolute threshold that might creep
    in, and the expected values of the scaled-matrix GPU tests (tests/test_gpu_eigh.py::test_solve_of_a_scaled_matrix)."""
    rng = np.random.default_rng(4242)
    n = 60
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    H = 0.5 * (A + A.conj().T)
    W1, Z1 = oracle.eigh(H)
    W2, Z2 = oracle.eigh(H * scale)
    assert np.array_equal(W2 / scale, W1)
    assert np.array_equal(Z2, Z1)
