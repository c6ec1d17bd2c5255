"""Pins of oracle/tdslda.py (SURVEY.md 8(f)4: one TDSLDA step, PAPER.md:91 Eq. 5, :113-115 Eq. 8, :134 ABM).  CPU only.

Chosen so that a plausible mistake fails one of them: a wrong k-grid or sign in the kinetic term (plane waves, matrix
form), a transposed / conjugated block of H (matrix form, Hermiticity), a wrong ABM coefficient or history order (exact
polynomial quadrature, 5th-order convergence on a stationary state), a wrong sign of i (phase of a stationary state)."""
import numpy as np
import pytest

import oracle
from oracle import tdslda as td
from paper_2310_03341_b200 import workloads as wl


def _fields(shape, seed):
    rng = np.random.default_rng(seed)
    M = int(np.prod(shape))
    V = rng.uniform(-0.3, 0.3, M)
    Delta = 0.3 * np.exp(2j * np.pi * rng.uniform(size=M)) * rng.uniform(0.5, 1.0, M)
    return V, Delta


def test_kinetic_term_on_plane_waves():
    """Eq. 8: a plane wave exp(i k.r) with k on the grid is an eigenfunction of -1/2 lap with eigenvalue k^2/2, the
    Nyquist mode n = -L/2 included (k = -pi)."""
    shape = (4, 6, 8)
    ix, iy, iz = np.meshgrid(*[np.arange(L) for L in shape], indexing="ij")
    for n in [(0, 0, 0), (1, -2, 3), (-2, 3, -4), (1, 0, -4)]:
        k = [2 * np.pi * n[a] / shape[a] for a in range(3)]
        f = np.exp(1j * (k[0] * ix + k[1] * iy + k[2] * iz)).reshape(-1)
        out = td.kinetic(f, shape)
        assert np.abs(out - 0.5 * sum(kk * kk for kk in k) * f).max() <= 1e-13


@pytest.mark.parametrize("shape", [(4, 4, 6), (3, 5, 4)])
def test_apply_h_equals_the_dense_matrix_of_the_prologue_oracle(shape):
    """Eq. 5 applied through FFTs (this oracle) = the dense matrix of Eq. 5/7/8 assembled from Kronecker products
    (oracle/assemble.py, pinned separately) with the 1-D kinetic matrices of the input generator: two independent routes.
    (odd extents: the generator's matrix has no Nyquist mode, neither has the FFT grid)"""
    V, Delta = _fields(shape, 1)
    mu = 0.7
    M = int(np.prod(shape))
    rng = np.random.default_rng(2)
    Phi = rng.standard_normal((2 * M, 5)) + 1j * rng.standard_normal((2 * M, 5))
    H = oracle.assemble.assemble_bdg(*[wl.kinetic_1d(L) for L in shape], V, Delta, mu)
    assert np.abs(H - H.conj().T).max() == 0.0
    out = td.apply_h(Phi, shape, V, Delta, mu)
    assert np.abs(out - H @ Phi).max() <= 1e-12 * np.abs(H @ Phi).max()


def test_abm_coefficients_integrate_polynomials_exactly():
    """A 5-step Adams-Bashforth / 4-step Adams-Moulton pair of order 5 integrates y' = p(t), deg p <= 4, exactly; the
    coefficient sets sum to 1."""
    assert abs(td.AB5.sum() - 1.0) < 1e-15 and abs(td.AM4.sum() - 1.0) < 1e-15
    dt = 0.1
    for deg in range(5):
        f = lambda t: t ** deg
        exact = ((dt) ** (deg + 1) - 0.0) / (deg + 1)                    # integral over [0, dt]
        ab = dt * sum(c * f(-k * dt) for k, c in enumerate(td.AB5))
        am = dt * sum(c * f((1 - k) * dt) for k, c in enumerate(td.AM4))
        assert abs(ab - exact) <= 1e-15 and abs(am - exact) <= 1e-15
    # degree 5 is NOT exact (order 5, not 6): guards against accidentally using a longer formula
    f = lambda t: t ** 5
    assert abs(dt * sum(c * f(-k * dt) for k, c in enumerate(td.AB5)) - dt ** 6 / 6) > 1e-9


def _stationary_problem():
    shape = (4, 4, 4)
    p = wl.bdg_vortex_tangle(shape, 2, 1.0, wl.SEED_BASE + 41, 0.02)
    H = p.dense()
    E, Z = oracle.eigh(H)
    return shape, p, H, E, Z


def test_stationary_states_pick_up_the_phase_exp_minus_iEt_at_fifth_order():
    """With frozen fields an eigenvector of H evolves as exp(-i E t) phi (Eq. 5 -- the sign of i); the global error of
    the PECE scheme scales like dt^5.  g = 0 and the fields of H itself freeze the Hamiltonian."""
    shape, p, H, E, Z = _stationary_problem()
    M = int(np.prod(shape))
    cols = [M + 3, M + 10]                         # two positive-energy states
    Y0, E0 = Z[:, cols], E[cols]

    def run(dt, nsteps):
        # exact history f(t) = -i E exp(-i E t) phi at t = 0, -dt, ..., -4 dt
        F = [(-1j * E0 * np.exp(-1j * E0 * (-k * dt)))[None, :] * Y0 for k in range(5)]
        Y = Y0.copy()
        for _ in range(nsteps):
            # frozen Hamiltonian: pass Delta through a "functional" with g = 0 plus the fixed field
            Yp = Y + dt * sum(c * f for c, f in zip(td.AB5, F))
            fp = td.rhs(Yp, shape, p.V, p.Delta, p.mu)
            Y = Y + dt * (td.AM4[0] * fp + sum(c * f for c, f in zip(td.AM4[1:], F[:4])))
            F = [td.rhs(Y, shape, p.V, p.Delta, p.mu)] + F[:4]
        return Y

    errs = []
    for dt, n in ((0.02, 8), (0.01, 16)):
        Y = run(dt, n)
        exact = np.exp(-1j * E0 * dt * n)[None, :] * Y0
        errs.append(np.abs(Y - exact).max())
    assert errs[0] < 1e-6
    order = np.log2(errs[0] / errs[1])
    assert 4.5 <= order <= 6.5, (errs, order)


def test_abm5_step_with_the_toy_functional_is_consistent():
    """abm5_step (the function the GPU is compared with) on the nonlinear system Delta = g nu[phi]: history built by a
    fine classical Runge-Kutta integration backwards in time, result compared with the same integration forwards (an
    independent integrator); the states stay orthonormal (unitary evolution) and the returned pairing field is
    the one of the last evaluation."""
    shape, p, H, E, Z = _stationary_problem()
    pos = np.where(E > 0)[0]
    Y0, E0 = Z[:, pos], E[pos]
    g = -2.0
    dt = 0.005

    def f(Y):
        return td.rhs(Y, shape, p.V, td.pairing_field(Y, E0, g), p.mu)

    def rk4(Y, h, n):
        for _ in range(n):
            k1 = f(Y); k2 = f(Y + 0.5 * h * k1); k3 = f(Y + 0.5 * h * k2); k4 = f(Y + h * k3)
            Y = Y + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        return Y

    sub = 8
    hist = [Y0]
    for _ in range(4):
        hist.append(rk4(hist[-1], -dt / sub, sub))           # Y(-dt), ..., Y(-4 dt)
    F = [f(Y) for Y in hist]
    Y1, F1, D1 = td.abm5_step(Y0, F, dt, shape, p.V, p.mu, E0, g)
    assert len(F1) == 5 and F1[1] is F[0] and F1[4] is F[3]
    assert np.abs(D1 - td.pairing_field(Y1, E0, g)).max() == 0.0
    assert np.abs(F1[0] - f(Y1)).max() == 0.0
    Yr = rk4(Y0, dt / sub, sub)
    assert np.abs(Y1 - Yr).max() <= 1e-7, np.abs(Y1 - Yr).max()
    G = Y1.conj().T @ Y1
    assert np.abs(G - np.eye(G.shape[0])).max() <= 1e-7
    # and the step does something: the state moved by about dt |f|
    assert np.abs(Y1 - Y0).max() >= 0.2 * dt * np.abs(F[0]).max()
