"""Pins of oracle/densities.py (Eq. 16a, 16d, 17) against what the
physics fixes: BCS closed forms for uniform pairing, completeness, particle number, the 2x2 problem.
None of them re-types the oracle's loop.
"""
import numpy as np
import pytest

import oracle
from oracle import densities as od
from paper_2310_03341_b200 import workloads as wl


def _k_shell_energies(shape, mu):
    """xi_k = |k|^2/2 - mu on the plane-wave grid of PAPER.md:113."""
    ks = []
    for L in shape:
        n = np.arange(-(L // 2), L - L // 2)
        ks.append(2 * np.pi * n / L)
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    return 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1) - mu


def _bcs_closed_form(shape, mu, delta, T):
    """Uniform pairing: Eq. 7 is 2x2 per k, [[xi, D], [D^*, -xi]].  Its E > 0 state has
    |u|^2 = (1 + xi/E)/2, |v|^2 = (1 - xi/E)/2, u v^* = D/(2E) (per plane wave, times 1/M on the lattice).
    With f(-E) - f(E) = tanh(E/2T) and f(-E) + f(E) = 1, Eq. 16a/16d give the textbook BCS sums
    n = (1/M) sum_k [1 - (xi/E) tanh(E/2T)],  nu = (1/M) sum_k D/(2E) tanh(E/2T)."""
    xi = _k_shell_energies(shape, mu)
    E = np.sqrt(xi ** 2 + abs(delta) ** 2)
    th = np.ones_like(E) if T == 0.0 else np.tanh(E / (2 * T))
    M = xi.size
    return (1.0 - xi / E * th).sum() / M, (delta / (2 * E) * th).sum() / M


@pytest.mark.parametrize("T", [0.0, 0.3])
@pytest.mark.parametrize("delta", [0.2, 0.25 * np.exp(0.7j)])
def test_uniform_bcs_closed_form(T, delta):
    """Catches swapped u/v, a dropped factor 2, a wrong conjugate or sign in nu, swapped Fermi factors."""
    shape = (4, 4, 6)
    p = wl.bdg_uniform(shape, 0.5, delta)
    H = p.dense()
    W, Z = oracle.eigh(H)
    n, nu = od.densities(W, Z, T=T)
    n_ref, nu_ref = _bcs_closed_form(shape, 0.5, delta, T)
    assert np.abs(n - n_ref).max() <= 1e-12
    assert np.abs(nu - nu_ref).max() <= 1e-12


def test_two_by_two():
    """M = 1: H = [[xi, D], [D^*, -xi]] by hand."""
    xi, D = 0.3, 0.4 * np.exp(-1.1j)
    E = np.hypot(xi, abs(D))
    H = np.array([[xi, D], [np.conj(D), -xi]])
    W, Z = oracle.eigh(H)
    n, nu = od.densities(W, Z, T=0.0)
    assert abs(n[0] - (1 - xi / E)) <= 1e-14
    assert abs(nu[0] - D / (2 * E)) <= 1e-14
    T = 0.2
    n, nu = od.densities(W, Z, T=T)
    th = np.tanh(E / (2 * T))
    assert abs(n[0] - (1 - xi / E * th)) <= 1e-14
    assert abs(nu[0] - D / (2 * E) * th) <= 1e-14


def test_fermi_function():
    """Eq. 17: f(E) + f(-E) = 1, f(0) = 1/2, large |E|/T limits, no overflow."""
    E = np.array([-800.0, -2.0, -1e-3, 0.0, 1e-3, 2.0, 800.0])
    f = od.fermi(E, 1.0)
    assert np.all(np.isfinite(f))
    assert np.abs(f + od.fermi(-E, 1.0) - 1.0).max() <= 2.3e-16
    assert f[3] == 0.5 and f[0] == 1.0 and f[-1] < 1e-300
    assert abs(f[5] - 1.0 / (1.0 + np.e ** 2)) <= 1e-16
    assert np.array_equal(od.fermi(E, 0.0), [1, 1, 1, 0.5, 0, 0, 0])


def _vortex_problem():
    p = wl.bdg_vortex_tangle((4, 4, 6), 3, 1.0, wl.SEED_BASE + 3, 0.02)
    H = p.dense()
    W, Z = oracle.eigh(H)
    return p, H, W, Z


def test_completeness_high_temperature():
    """f -> 1/2: the E > 0 states and their particle-hole partners are a complete basis, so
    sum_{E>0} |u_n(r)|^2 + |v_n(r)|^2 = 1 at every r: n(r) = 1 and nu(r) = 0 as T -> infinity."""
    _, _, W, Z = _vortex_problem()
    n, nu = od.densities(W, Z, T=1e12)
    assert np.abs(n - 1.0).max() <= 1e-10
    assert np.abs(nu).max() <= 1e-10


def test_particle_number_and_cutoff():
    """sum_r n(r) = 2 sum_n ||v_n||^2 at T = 0 (dx = 1); states outside 0 < E < Ec do not contribute."""
    _, _, W, Z = _vortex_problem()
    M = Z.shape[0] // 2
    n, nu = od.densities(W, Z, T=0.0)
    pos = W > 0
    assert abs(n.sum() - 2.0 * (np.abs(Z[M:, pos]) ** 2).sum()) <= 1e-11
    Ec = float(np.median(W[pos]))
    n_c, nu_c = od.densities(W, Z, T=0.0, Ec=Ec)
    keep = pos & (W < Ec)
    n_k, nu_k = od.densities(W[keep], Z[:, keep], T=0.0)
    assert np.array_equal(n_c, n_k) and np.array_equal(nu_c, nu_k)
    assert n_c.sum() < n.sum()


def test_points_subset_and_gap_equation_sign():
    """`points` evaluates the same sums on selected r; nu follows the phase of Delta where |Delta| is large
    (the gap equation Delta = -g nu of the functional has a real coupling): the winding of the
    vortices shows in arg nu."""
    p, _, W, Z = _vortex_problem()
    n, nu = od.densities(W, Z, T=0.0)
    pts = np.array([0, 5, 17, 95])
    n_s, nu_s = od.densities(W, Z, T=0.0, points=pts)
    assert np.array_equal(n_s, n[pts]) and np.array_equal(nu_s, nu[pts])
    big = np.abs(p.Delta) > 0.5 * np.abs(p.Delta).max()
    dphi = np.angle(nu[big] * np.conj(p.Delta[big]))
    assert np.abs(dphi).max() < np.pi / 2 and np.median(np.abs(dphi)) < 0.2   # tiny lattice: aligned, not equal


def test_particle_hole_map_gives_the_same_densities():
    """The negative branch mapped by [u, v] -> [-v^*, u^*] is an eigenbasis of the positive branch:
    residual of the mapped states, and equal densities from either branch."""
    _, H, W, Z = _vortex_problem()
    neg = W < 0
    Ep, Zp = od.particle_hole_map(W[neg], Z[:, neg])
    assert np.linalg.norm(H @ Zp - Zp * Ep[None, :]) <= 1e-12 * np.linalg.norm(H)
    for T in (0.0, 0.25):
        n1, nu1 = od.densities(W, Z, T=T)
        n2, nu2 = od.densities(Ep, Zp, T=T)
        assert np.abs(n1 - n2).max() <= 1e-11
        assert np.abs(nu1 - nu2).max() <= 1e-11


# ----------------------------------------------------------------------------- Eq. 16b, 16c
def _k_grid(shape, for_derivative):
    """Wave vectors of the plane waves exp(i k r) on the grid; for the first derivative the Nyquist
    component counts as 0 (workloads.derivative_1d)."""
    ks = []
    for L in shape:
        n = np.arange(-(L // 2), L - L // 2)
        k = 2 * np.pi * n / L
        if for_derivative and L % 2 == 0:
            k = np.where(n == -(L // 2), 0.0, k)
        ks.append(k)
    return [a.reshape(-1) for a in np.meshgrid(*ks, indexing="ij")]


def test_derivative_matrix_is_spectral():
    """D exp(i k x) = i k exp(i k x) on the grid; odd L: D D = -2 K (the kinetic matrix of Eq. 8)."""
    for L in (5, 8):
        D = wl.derivative_1d(L)
        assert np.abs(D + D.T).max() <= 1e-14
        x = np.arange(L)
        for n in range(-(L // 2), L - L // 2):
            k = 2 * np.pi * n / L
            w = np.exp(1j * k * x)
            keff = 0.0 if (L % 2 == 0 and n == -(L // 2)) else k
            assert np.abs(D @ w - 1j * keff * w).max() <= 1e-12
    assert np.abs(wl.derivative_1d(7) @ wl.derivative_1d(7) + 2 * wl.kinetic_1d(7)).max() <= 1e-12


@pytest.mark.parametrize("T", [0.0, 0.3])
def test_tau_uniform_bcs_closed_form(T):
    """Plane waves: |grad v_k|^2 = |k|^2 |v_k|^2, so tau = (1/M) sum_k |k|^2 [1 - xi/E tanh(E/2T)]; j = 0 (k <-> -k)."""
    shape = (4, 5, 6)
    delta = 0.25 * np.exp(0.7j)
    p = wl.bdg_uniform(shape, 0.5, delta)
    W, Z = oracle.eigh(p.dense())
    Ds = [wl.derivative_1d(L) for L in shape]
    tau, j = od.gradient_densities(W, Z, shape, *Ds, T=T)
    xi = _k_shell_energies(shape, 0.5)
    E = np.sqrt(xi ** 2 + abs(delta) ** 2)
    th = np.ones_like(E) if T == 0.0 else np.tanh(E / (2 * T))
    kx, ky, kz = _k_grid(shape, True)
    ref = ((kx ** 2 + ky ** 2 + kz ** 2) * (1.0 - xi / E * th)).mean()
    assert np.abs(tau - ref).max() <= 1e-11
    assert np.abs(j).max() <= 1e-11


def test_current_of_a_moving_condensate_closed_form():
    """Delta(r) = D0 exp(2 i q r): u ~ exp(i (k+q) r), v ~ exp(i (k-q) r), 2x2 blocks [[xi_{k+q}, D0], [D0, -xi_{k-q}]].
    At T = 0: n = (2/M) sum |v|^2, j = -(2/M) sum |v|^2 (k - q), tau = (2/M) sum |v|^2 |k - q|^2 over the E > 0 states
    (Im(v grad v^*) = -(k - q) |v|^2).  Odd grid (no Nyquist mode), q = one grid step along x and two along z.
    Catches a wrong sign, a conjugated gradient, a transposed derivative matrix and swapped axes (j_y = 0, j_x != j_z)."""
    shape = (5, 5, 7)
    nx, ny, nz = shape
    M = nx * ny * nz
    mu, D0 = 0.9, 0.3
    X, Y, Zc = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    q = np.array([2 * np.pi / nx, 0.0, 2 * 2 * np.pi / nz])
    Delta = D0 * np.exp(2j * (q[0] * X + q[1] * Y + q[2] * Zc)).reshape(-1)
    p = wl.BdGProblem("moving", shape, mu, np.zeros(M), Delta)
    W, Z = oracle.eigh(p.dense())
    Ds = [wl.derivative_1d(L) for L in shape]
    n, nu = od.densities(W, Z, T=0.0)
    tau, j = od.gradient_densities(W, Z, shape, *Ds, T=0.0)

    def wrap(k, L):                                   # wave number of exp(i k x) folded onto the grid values
        m = np.rint(k * L / (2 * np.pi)).astype(int)
        m = (m + L // 2) % L - L // 2
        return 2 * np.pi * m / L
    n_ref, tau_ref, j_ref = 0.0, 0.0, np.zeros(3)
    kx, ky, kz = _k_grid(shape, False)
    for k in zip(kx, ky, kz):
        kp = np.array([wrap(k[a] + q[a], shape[a]) for a in range(3)])
        km = np.array([wrap(k[a] - q[a], shape[a]) for a in range(3)])
        B = np.array([[0.5 * kp @ kp - mu, D0], [D0, -(0.5 * km @ km - mu)]])
        w, V2 = np.linalg.eigh(B)
        for e, vec in zip(w, V2.T):
            if e > 0:
                n_ref += 2 * vec[1] ** 2 / M
                tau_ref += 2 * vec[1] ** 2 * (km @ km) / M
                j_ref -= 2 * vec[1] ** 2 * km / M
    assert np.abs(n - n_ref).max() <= 1e-11
    assert np.abs(tau - tau_ref).max() <= 1e-11
    for a in range(3):
        assert np.abs(j[a] - j_ref[a]).max() <= 1e-11
    assert abs(j_ref[0]) > 1e-3 and abs(j_ref[2]) > 1e-3 and abs(j_ref[0] - j_ref[2]) > 1e-3 and abs(j_ref[1]) <= 1e-15


def test_gradient_densities_invariants_on_vortex_fields():
    """Any fields: (i) T -> infinity: completeness gives tau(r) = sum_a (D_a D_a^T)[i_a, i_a] and j(r) = 0;
    (ii) odd grid, T = 0: sum_r tau(r) = 4 sum_n <v_n| K |v_n> with the kinetic operator of Eq. 8 (D^T D = 2 K);
    (iii) states outside the cutoff do not contribute."""
    shape = (3, 5, 5)
    p = wl.bdg_vortex_tangle(shape, 2, 1.0, wl.SEED_BASE + 7, 0.02)
    M = p.N // 2
    W, Z = oracle.eigh(p.dense())
    Ds = [wl.derivative_1d(L) for L in shape]
    tau, j = od.gradient_densities(W, Z, shape, *Ds, T=1e12)
    ref = sum(np.sum(D * D, axis=1)[0] for D in Ds)
    assert np.abs(tau - ref).max() <= 1e-9 and np.abs(j).max() <= 1e-9
    tau, j = od.gradient_densities(W, Z, shape, *Ds, T=0.0)
    Ks = [wl.kinetic_1d(L) for L in shape]
    Kfull = (np.kron(np.kron(Ks[0], np.eye(shape[1])), np.eye(shape[2])) + np.kron(np.kron(np.eye(shape[0]), Ks[1]), np.eye(shape[2]))
             + np.kron(np.kron(np.eye(shape[0]), np.eye(shape[1])), Ks[2]))
    pos = W > 0
    Vp = Z[M:, pos]
    assert abs(tau.sum() - 4.0 * np.real(np.sum(np.conj(Vp) * (Kfull @ Vp)))) <= 1e-10
    Ec = float(np.median(W[pos]))
    t_c, j_c = od.gradient_densities(W, Z, shape, *Ds, T=0.0, Ec=Ec)
    keep = pos & (W < Ec)
    t_k, j_k = od.gradient_densities(W[keep], Z[:, keep], shape, *Ds, T=0.0)
    assert np.array_equal(t_c, t_k) and np.array_equal(j_c, j_k) and t_c.sum() < tau.sum()
