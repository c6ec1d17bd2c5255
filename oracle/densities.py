"""CPU oracle of the SCF epilogue: local densities from the quasiparticle states.
TEST INFRASTRUCTURE ONLY -- shares nothing with the CUDA path.

PAPER.md:300-311, Eq. (16a), (16d), (17), written out as they stand, in FP64:

    n(r)  = 2 sum_{0 < E_n < E_c} ( |v_n(r)|^2 f_T(-E_n) + |u_n(r)|^2 f_T(E_n) )          (16a)
    nu(r) =   sum_{0 < E_n < E_c} u_n(r) conj(v_n(r)) ( f_T(-E_n) - f_T(E_n) )             (16d)
    f_T(E) = 1 / (1 + exp(E / T)),   T = 0:  f_T(E) = 1 for E < 0, 0 for E > 0            (17)

phi_n = [u_n, v_n]^T is column n of Z: rows [0, M) hold u_n(r), rows [M, 2M) hold v_n(r) (matrix index
s * M + r); dx = 1, so sum_r |u_n|^2 + |v_n|^2 = 1.  The kinetic and current densities
(16b, 16c) need gradients and are not part of this row.
"""
from __future__ import annotations

import numpy as np


def fermi(E, T):
    """Eq. (17).  T = 0 is the step function (f(0) = 1/2 is never used: the sums exclude E = 0)."""
    E = np.asarray(E, dtype=np.float64)
    if T == 0.0:
        return np.where(E < 0.0, 1.0, np.where(E > 0.0, 0.0, 0.5))
    x = E / T
    out = np.empty_like(x)
    pos = x >= 0
    out[pos] = np.exp(-x[pos]) / (1.0 + np.exp(-x[pos]))      # overflow-free forms of 1 / (1 + e^x)
    out[~pos] = 1.0 / (1.0 + np.exp(x[~pos]))
    return out


def densities(E, Z, T=0.0, Ec=np.inf, points=None):
    """E: energies of the columns of Z (any order, any sign); Z: (2M, ncols) complex.  Returns
    (n, nu) on all M grid points, or on `points` only (the oracle then touches 2 len(points) rows of Z)."""
    E = np.asarray(E, dtype=np.float64)
    Z = np.asarray(Z)
    M = Z.shape[0] // 2
    rows = np.arange(M) if points is None else np.asarray(points)
    n = np.zeros(rows.shape[0], dtype=np.float64)
    nu = np.zeros(rows.shape[0], dtype=np.complex128)
    for j in range(Z.shape[1]):                     # state by state, in the order of Eq. (16)
        if not (0.0 < E[j] < Ec):
            continue
        fm, fp = float(fermi(-E[j], T)), float(fermi(E[j], T))
        u = Z[rows, j]
        v = Z[M + rows, j]
        n += 2.0 * (np.abs(v) ** 2 * fm + np.abs(u) ** 2 * fp)
        nu += u * np.conj(v) * (fm - fp)
    return n, nu


def particle_hole_map(E, Z):
    """Positive-energy states from negative-energy ones: H = [[h, D], [D^*, -h^*]] with diagonal D has
    S H^* S^-1 = -H, S = [[0, -I], [I, 0]] (SURVEY.md 8(c) reading 3), so phi = [u, v] with energy E < 0 gives
    [-v^*, u^*] with energy -E > 0.  Returns (-E, mapped Z) column by column; the densities of the negative
    branch are `densities(*particle_hole_map(E, Z), ...)`, i.e. Eq. (16) as written on the mapped states."""
    E = np.asarray(E, dtype=np.float64)
    Z = np.asarray(Z)
    M = Z.shape[0] // 2
    Zp = np.empty_like(Z)
    Zp[:M] = -np.conj(Z[M:])
    Zp[M:] = np.conj(Z[:M])
    return -E, Zp


def gradient_densities(E, Z, shape, Dx, Dy, Dz, T=0.0, Ec=np.inf):
    """Kinetic and current densities, Eq. (16b), (16c), written out state by state in FP64:

        tau(r) = 2 sum_{0 < E_n < E_c} ( |grad v_n|^2 f_T(-E_n) + |grad u_n|^2 f_T(E_n) )                  (16b)
        j(r)   = 2 sum_{0 < E_n < E_c} Im( v_n grad v_n^* f_T(-E_n) - u_n grad u_n^* f_T(E_n) )             (16c)

    Reading: Eq. 16b prints the range "0 <= E_n <= E_r"; the range of (16a, c, d) is used for all four.
    The gradient is applied along each axis through a dense real 1-D matrix (inputs Dx, Dy, Dz; the spectral
    derivative of PAPER.md:113-115 in matrix form): (d_x u)(ix, iy, iz) = sum_i' Dx[ix, i'] u(i', iy, iz), etc.,
    on the grid r = (ix ny + iy) nz + iz.  Returns tau (M,) and j (3, M)."""
    E = np.asarray(E, dtype=np.float64)
    Z = np.asarray(Z)
    nx, ny, nz = shape
    M = nx * ny * nz
    D = [np.asarray(Dx, dtype=np.float64), np.asarray(Dy, dtype=np.float64), np.asarray(Dz, dtype=np.float64)]
    tau = np.zeros(M, dtype=np.float64)
    j = np.zeros((3, M), dtype=np.float64)

    def grad(w):
        w = w.reshape(nx, ny, nz)
        return [np.einsum("ai,ijk->ajk", D[0], w).reshape(M),
                np.einsum("bj,ijk->ibk", D[1], w).reshape(M),
                np.einsum("ck,ijk->ijc", D[2], w).reshape(M)]

    for c in range(Z.shape[1]):
        if not (0.0 < E[c] < Ec):
            continue
        fm, fp = float(fermi(-E[c], T)), float(fermi(E[c], T))
        u, v = Z[:M, c], Z[M:, c]
        gu, gv = grad(u), grad(v)
        for a in range(3):
            tau += 2.0 * (np.abs(gv[a]) ** 2 * fm + np.abs(gu[a]) ** 2 * fp)
            j[a] += 2.0 * np.imag(v * np.conj(gv[a]) * fm - u * np.conj(gu[a]) * fp)
    return tau, j
