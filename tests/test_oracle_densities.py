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
