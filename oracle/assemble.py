"""CPU oracle of the SCF prologue: the dense BdG matrix from its fields.
TEST INFRASTRUCTURE ONLY -- shares nothing with the CUDA path.

PAPER.md:103-107 (Eq. 5 / 7): H = [[h, Delta], [Delta^*, -h^*]], h = -nabla^2/2 + V - mu, with the kinetic term
applied spectrally along each axis (Eq. 8) and the matrix kept DENSE.  On the grid
r = (ix Ny + iy) Nz + iz the definition written out with Kronecker products is

    T = Kx (x) Iy (x) Iz  +  Ix (x) Ky (x) Iz  +  Ix (x) Iy (x) Kz
    h = T + diag(V) - mu I            (evaluated in this order: ((Kx + Ky) + Kz + V) - mu on the diagonal)
    H = [[h, diag(Delta)], [diag(Delta)^*, -h^*]],      matrix index = s M + r,  s = 0 (u), 1 (v).

The 1-D matrices Kx, Ky, Kz are inputs (any real symmetric DVR of -d^2/2).
"""
from __future__ import annotations

import numpy as np


def assemble_bdg(Kx, Ky, Kz, V, Delta, mu, sign=1.0):
    Kx, Ky, Kz = (np.asarray(K, dtype=np.float64) for K in (Kx, Ky, Kz))
    nx, ny, nz = Kx.shape[0], Ky.shape[0], Kz.shape[0]
    M = nx * ny * nz
    V = np.asarray(V, dtype=np.float64).reshape(M)
    Delta = np.asarray(Delta, dtype=np.complex128).reshape(M)
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    T = np.kron(np.kron(Kx, Iy), Iz) + np.kron(np.kron(Ix, Ky), Iz)
    T = T + np.kron(np.kron(Ix, Iy), Kz)
    h = T + np.diag(V)
    h = h - mu * np.eye(M)
    H = np.zeros((2 * M, 2 * M), dtype=np.complex128)
    H[:M, :M] = h
    H[M:, M:] = -np.conj(h)
    H[:M, M:] = np.diag(Delta)
    H[M:, :M] = np.diag(np.conj(Delta))
    return sign * H
