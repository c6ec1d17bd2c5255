"""Oracle for one TDSLDA time step.  TEST INFRASTRUCTURE ONLY -- plain numpy, FP64; shares
nothing with the CUDA path.

What the paper fixes:
  * the equation of motion, Eq. 5:  i d/dt [u_n, v_n] = [[h, Delta], [Delta^*, -h^*]] [u_n, v_n], hbar = 1;
  * the kinetic term, Eq. 8:  -1/2 lap phi = F^-1( k^2/2 F(phi) ), k = 2 pi n / N per axis,
    n in {-N/2, ..., N/2 - 1}  (the unpaired Nyquist mode is kept: SURVEY.md 8(c) reading 10);
  * the integrator: "5th-order multistep Adams-Bashforth-Moulton predictor-corrector", h and Delta
    evaluated twice per step (predictor and corrector), "about 10 copies of the state".
Readings where the paper is silent:
  * the ABM coefficients are the textbook ones: 5-step Adams-Bashforth predictor and 4-step (5th order) Adams-Moulton
    corrector in PECE form (predict, evaluate, correct, evaluate);
  * h = -1/2 lap + V(r) - mu with a real local potential (the SLDA functional's A, B, C are not in the paper,
    SURVEY.md 2a A11); the pairing field follows the toy functional of the SCF test, Delta(r) = g nu(r) (Eq. 18b with a
    constant coupling), nu from Eq. 16d with occupation weights frozen at their initial values.
"""
from __future__ import annotations

import numpy as np

from . import densities as _dens

AB5 = np.array([1901.0, -2774.0, 2616.0, -1274.0, 251.0]) / 720.0      # f_n, f_{n-1}, ..., f_{n-4}
AM4 = np.array([251.0, 646.0, -264.0, 106.0, -19.0]) / 720.0           # f_{n+1}, f_n, ..., f_{n-3}


def k2_half(shape):
    """k^2/2 on the FFT grid of `shape`: k = 2 pi n / L, n = -L/2 .. L/2-1 per axis."""
    ks = []
    for L in shape:
        n = np.fft.fftfreq(L, d=1.0 / L)                 # 0, 1, ..., L/2-1, -L/2, ..., -1
        ks.append(2.0 * np.pi * n / L)
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    return 0.5 * (KX ** 2 + KY ** 2 + KZ ** 2)


def kinetic(f, shape):
    """Eq. 8: -1/2 lap f = F^-1(k^2/2 F(f)) for one field on the grid (row-major r = (ix ny + iy) nz + iz)."""
    g = np.fft.fftn(f.reshape(shape))
    return np.fft.ifftn(k2_half(shape) * g).reshape(-1)


def apply_h(Phi, shape, V, Delta, mu):
    """H Phi for the columns of Phi (2M x ncols): Eq. 5 with h = -1/2 lap + V - mu (real h: h^* = h)."""
    M = int(np.prod(shape))
    Phi = np.asarray(Phi, dtype=np.complex128)
    out = np.empty_like(Phi)
    for j in range(Phi.shape[1]):
        u, v = Phi[:M, j], Phi[M:, j]
        hu = kinetic(u, shape) + (V - mu) * u
        hv = kinetic(v, shape) + (V - mu) * v
        out[:M, j] = hu + Delta * v
        out[M:, j] = np.conj(Delta) * u - hv
    return out


def rhs(Phi, shape, V, Delta, mu):
    """d Phi / dt = -i H Phi  (Eq. 5, hbar = 1)."""
    return -1j * apply_h(Phi, shape, V, Delta, mu)


def pairing_field(Phi, E0, g, T=0.0, Ec=np.inf):
    """Delta = g nu, nu from Eq. 16d (oracle/densities.py) with the weights of the initial energies E0."""
    _, nu = _dens.densities(E0, Phi, T=T, Ec=Ec)
    return g * nu


def abm5_step(Y, F, dt, shape, V, mu, E0, g, T=0.0, Ec=np.inf):
    """One PECE step.  Y: state (2M x ncols) at t_n; F: list of the 5 derivatives [f_n, f_{n-1}, ..., f_{n-4}].
    Returns (Y_{n+1}, [f_{n+1}, f_n, ..., f_{n-3}], Delta used in the last evaluation)."""
    Yp = Y + dt * sum(c * f for c, f in zip(AB5, F))                         # P
    Dp = pairing_field(Yp, E0, g, T, Ec)
    fp = rhs(Yp, shape, V, Dp, mu)                                           # E
    Yc = Y + dt * (AM4[0] * fp + sum(c * f for c, f in zip(AM4[1:], F[:4])))  # C
    Dc = pairing_field(Yc, E0, g, T, Ec)
    fc = rhs(Yc, shape, V, Dc, mu)                                           # E
    return Yc, [fc] + list(F[:4]), Dc
