"""Seeded synthetic inputs (BASELINE.json `configs`, recipe fixed in SURVEY.md 8(d)).

This module holds NONE of the eigensolver's arithmetic: it only builds the test
matrices.  It is the one module shared by the oracle-side tests and the CUDA-side
tests / bench (both sides must see the same seeded inputs).

The matrices stand in for the paper's production SLDA Hamiltonians (PAPER.md:144,
:166), which cannot be rebuilt here: they keep the structure that matters for the
eigensolver -- the BdG block form of Eq. 7, the spectral kinetic term
of Eq. 8 on the grid k = 2 pi n / N, n in {-N/2 .. N/2-1} stored as
a DENSE matrix ("dense diagonalization"), a diagonal complex pairing
field with vortex phase windings, and the +/- symmetric spectrum.

Conventions: grid Nx x Ny x Nz, dx = 1, hbar = m = 1; point index
r = (ix*Ny + iy)*Nz + iz; coordinates centred on half-integers x = ix - (Nx-1)/2
(no grid point on a vortex axis); matrix index = s*Nxyz + r, s = 0 (u), 1 (v);
N = 2*Nxyz.  RNG: numpy default_rng(PCG64), seed = SEED_BASE + config index; draw
order: noise field first (row-major r), then per vortex line position (3 uniforms in
the box) and direction (3 normalised Gaussians); signs alternate +,-,+,... (not drawn).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

SEED_BASE = 23100334100


# --------------------------------------------------------------------------- kinetic term
def kinetic_1d(L: int) -> np.ndarray:
    """K_L[i,j] = (1/L) sum_{n=-L/2}^{L/2-1} 0.5 (2 pi n / L)^2 cos(2 pi n (i-j) / L).

    Dense-matrix form of Eq. 8 along one axis; real symmetric
    circulant; the unpaired Nyquist mode n = -L/2 is kept (SURVEY.md 8(c) reading 10).
    """
    n = np.arange(-(L // 2), L - L // 2)
    k = 2.0 * np.pi * n / L
    diff = np.arange(L)[:, None] - np.arange(L)[None, :]
    K = np.zeros((L, L))
    for kk, nn in zip(k, n):
        K += 0.5 * kk * kk * np.cos(2.0 * np.pi * nn * diff / L)
    return K / L


def derivative_1d(L: int) -> np.ndarray:
    """D_L[i,j] = (1/L) sum_n (i k_n) exp(i k_n (i-j)) = -(1/L) sum_n k_n sin(k_n (i-j)), k_n = 2 pi n / L.

    Dense-matrix form of the spectral first derivative on the grid of PAPER.md:113-115; real antisymmetric circulant.
    The unpaired Nyquist mode n = -L/2 (even L) has no real first derivative on the grid and is dropped, the usual
    convention; D exp(i k x) = i k exp(i k x) for every other grid wave number.  An input of eigh_gradient_densities.
    """
    n = np.arange(-(L // 2), L - L // 2)
    if L % 2 == 0:
        n = n[1:]
    k = 2.0 * np.pi * n / L
    diff = np.arange(L)[:, None] - np.arange(L)[None, :]
    D = np.zeros((L, L))
    for kk in k:
        D -= kk * np.sin(kk * diff)
    return D / L


def grid_coords(shape: Tuple[int, int, int]):
    Nx, Ny, Nz = shape
    x = np.arange(Nx) - (Nx - 1) / 2.0
    y = np.arange(Ny) - (Ny - 1) / 2.0
    z = np.arange(Nz) - (Nz - 1) / 2.0
    X, Y, Z = np.meshgrid(x, y, z, indexing="ij")
    return X.reshape(-1), Y.reshape(-1), Z.reshape(-1)


# --------------------------------------------------------------------------- BdG assembly
@dataclass
class BdGProblem:
    """A BdG Hamiltonian H = [[h, diag(Delta)], [diag(Delta)^*, -h]], h = T + diag(V) - mu,
    kept as its fields; dense() / dense_torch() materialise the N x N complex128 matrix."""
    name: str
    shape: Tuple[int, int, int]
    mu: float
    V: np.ndarray            # real potential, Nxyz
    Delta: np.ndarray        # complex pairing field, Nxyz
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return 2 * int(np.prod(self.shape))

    def _h_triplets(self):
        """COO triplets (rows, cols, vals) of h = T + diag(V) - mu (real)."""
        Nx, Ny, Nz = self.shape
        nxyz = Nx * Ny * Nz
        idx = np.arange(nxyz).reshape(Nx, Ny, Nz)
        rows, cols, vals = [], [], []
        Kx, Ky, Kz = kinetic_1d(Nx), kinetic_1d(Ny), kinetic_1d(Nz)
        # x axis: (ix,iy,iz) <- (jx,iy,iz)
        r = np.broadcast_to(idx[:, None, :, :], (Nx, Nx, Ny, Nz))
        c = np.broadcast_to(idx[None, :, :, :], (Nx, Nx, Ny, Nz))
        v = np.broadcast_to(Kx[:, :, None, None], (Nx, Nx, Ny, Nz))
        rows.append(r.reshape(-1)); cols.append(c.reshape(-1)); vals.append(v.reshape(-1))
        # y axis: (ix,iy,iz) <- (ix,jy,iz)
        r = np.broadcast_to(idx[:, :, None, :], (Nx, Ny, Ny, Nz))
        c = np.broadcast_to(idx[:, None, :, :], (Nx, Ny, Ny, Nz))
        v = np.broadcast_to(Ky[None, :, :, None], (Nx, Ny, Ny, Nz))
        rows.append(r.reshape(-1)); cols.append(c.reshape(-1)); vals.append(v.reshape(-1))
        # z axis: (ix,iy,iz) <- (ix,iy,jz)
        r = np.broadcast_to(idx[:, :, :, None], (Nx, Ny, Nz, Nz))
        c = np.broadcast_to(idx[:, :, None, :], (Nx, Ny, Nz, Nz))
        v = np.broadcast_to(Kz[None, None, :, :], (Nx, Ny, Nz, Nz))
        rows.append(r.reshape(-1)); cols.append(c.reshape(-1)); vals.append(v.reshape(-1))
        # diagonal: V - mu
        d = np.arange(nxyz)
        rows.append(d); cols.append(d); vals.append(self.V - self.mu)
        return (np.concatenate(rows), np.concatenate(cols),
                np.ascontiguousarray(np.concatenate(vals), dtype=np.float64))

    def dense(self) -> np.ndarray:
        """Host assembly (numpy), complex128, Fortran order."""
        n = self.N // 2
        r, c, v = self._h_triplets()
        h = np.zeros((n, n))
        np.add.at(h, (r, c), v)
        H = np.zeros((2 * n, 2 * n), dtype=np.complex128, order="F")
        H[:n, :n] = h
        H[n:, n:] = -h
        i = np.arange(n)
        H[i, n + i] = self.Delta
        H[n + i, i] = np.conj(self.Delta)
        return H

    def dense_torch(self, device="cuda", out=None, sign: float = 1.0):
        """Device assembly (torch used for memory plumbing only): returns an N x N complex128
        tensor whose STORAGE is column-major (tensor.t() is contiguous).  sign=-1 gives -H."""
        import torch
        n = self.N // 2
        N = 2 * n
        r, c, v = self._h_triplets()
        if out is None:
            out = torch.zeros((N, N), dtype=torch.complex128, device=device)
        else:
            assert out.shape == (N, N) and out.dtype == torch.complex128
            out.zero_()
        # `out` is row-major storage of H^T, i.e. column-major storage of H: write H^T entries.
        Ht = out
        rt = torch.from_numpy(r).to(device)
        ct = torch.from_numpy(c).to(device)
        vt = torch.from_numpy(v).to(device).to(torch.complex128) * sign
        Ht.index_put_((ct, rt), vt, accumulate=True)                  # h block (transposed)
        Ht.index_put_((ct + n, rt + n), -vt, accumulate=True)         # -h block
        i = torch.arange(n, device=device)
        D = torch.from_numpy(np.ascontiguousarray(self.Delta)).to(device) * sign
        Ht[n + i, i] = D                   # H[i, n+i] = Delta  -> H^T[n+i, i]
        Ht[i, n + i] = torch.conj(D)       # H[n+i, i] = Delta^* -> H^T[i, n+i]
        return out.t()                      # logical H, column-major storage


def _vortex_lines_delta(shape, n_lines, rng, amp=0.3):
    """Delta = amp * prod_j tanh(d_j/2) exp(i s_j phi_j) over straight vortex lines
    (SURVEY.md 8(d), config 3): line j through p_j with unit direction t_j;
    d_j = distance to the line; frame e1 = normalise(t x a), a = z unless |t.z| > 0.9
    then a = x, e2 = t x e1; phi_j = atan2((r-p).e2, (r-p).e1); s_j = +,-,+,..."""
    Nx, Ny, Nz = shape
    X, Y, Z = grid_coords(shape)
    R = np.stack([X, Y, Z], axis=1)
    Delta = np.full(X.shape, amp, dtype=np.complex128)
    lines = []
    for j in range(n_lines):
        p = (rng.random(3) - 0.5) * np.array([Nx, Ny, Nz], dtype=np.float64)
        t = rng.standard_normal(3)
        t /= np.linalg.norm(t)
        s = 1.0 if j % 2 == 0 else -1.0
        a = np.array([0.0, 0.0, 1.0]) if abs(t[2]) <= 0.9 else np.array([1.0, 0.0, 0.0])
        e1 = np.cross(t, a)
        e1 /= np.linalg.norm(e1)
        e2 = np.cross(t, e1)
        q = R - p[None, :]
        q_perp = q - (q @ t)[:, None] * t[None, :]
        dj = np.linalg.norm(q_perp, axis=1)
        phi = np.arctan2(q @ e2, q @ e1)
        Delta *= np.tanh(dj / 2.0) * np.exp(1j * s * phi)
        lines.append((p, t, s))
    return Delta, lines


def bdg_uniform(shape=(8, 8, 8), mu=0.5, delta=0.2) -> BdGProblem:
    """Config 0: uniform real pairing on a periodic lattice, V = 0."""
    nxyz = int(np.prod(shape))
    return BdGProblem("bdg_uniform", tuple(shape), mu, np.zeros(nxyz),
                      np.full(nxyz, delta, dtype=np.complex128))


def bdg_single_vortex(shape=(16, 16, 16), mu=1.0, seed=SEED_BASE + 2, noise=0.01,
                      omega=0.05, amp=0.3) -> BdGProblem:
    """Config 2: one vortex line along z through the box centre, harmonic trap in rho
    plus seeded uniform noise: V = 0.5 omega^2 rho^2 + U(-noise, noise);
    Delta = amp tanh(rho/2) exp(i phi), phi = atan2(y, x)."""
    rng = np.random.default_rng(seed)
    X, Y, Z = grid_coords(shape)
    nxyz = X.shape[0]
    nz = rng.uniform(-noise, noise, nxyz)
    rho = np.hypot(X, Y)
    V = 0.5 * omega * omega * rho * rho + nz
    Delta = amp * np.tanh(rho / 2.0) * np.exp(1j * np.arctan2(Y, X))
    return BdGProblem("bdg_single_vortex", tuple(shape), mu, V, Delta)


def bdg_vortex_tangle(shape=(24, 24, 24), n_lines=6, mu=1.0, seed=SEED_BASE + 3,
                      noise=0.02, amp=0.3) -> BdGProblem:
    """Configs 3 and 4: product of straight vortex lines at seeded positions/orientations,
    seeded noise potential."""
    rng = np.random.default_rng(seed)
    nxyz = int(np.prod(shape))
    V = rng.uniform(-noise, noise, nxyz)
    Delta, lines = _vortex_lines_delta(tuple(shape), n_lines, rng, amp)
    return BdGProblem("bdg_vortex_tangle", tuple(shape), mu, V, Delta, meta={"lines": lines})


# --------------------------------------------------------------------------- config 1
def clustered_spectrum(N: int, rng, frac=0.1, cluster=10, width=1e-12) -> np.ndarray:
    """lambda for config 1 (SURVEY.md 8(c) reading 12): floor(frac*N) values in clusters of
    `cluster` (+ one remainder cluster), centres U[-1,1], members = centre +
    U(-width/2, width/2); the others U[-1,1].  Returned UNSORTED (cluster values first)."""
    ncl = int(np.floor(frac * N))
    nfull, rem = divmod(ncl, cluster)
    sizes = [cluster] * nfull + ([rem] if rem else [])
    centres = rng.uniform(-1.0, 1.0, len(sizes))
    offs = rng.uniform(-0.5 * width, 0.5 * width, ncl)
    lam_c = np.repeat(centres, sizes) + offs
    lam_o = rng.uniform(-1.0, 1.0, N - ncl)
    return np.concatenate([lam_c, lam_o])


def random_hermitian_clustered(N=4096, seed=SEED_BASE + 1):
    """Config 1: A = Q diag(lambda) Q^H, Q from the QR of a seeded complex Gaussian matrix,
    then A <- (A + A^H)/2.  Returns (A [complex128, Fortran order], lambda sorted ascending)."""
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))
    lam = clustered_spectrum(N, rng)
    Q, _ = np.linalg.qr(G)
    A = (Q * lam[None, :]) @ Q.conj().T
    A = 0.5 * (A + A.conj().T)
    return np.asfortranarray(A), np.sort(lam)


# --------------------------------------------------------------------------- registry
@dataclass
class Workload:
    index: int
    name: str
    N: int
    nev_runs: Tuple[int, ...]
    problem: Optional[BdGProblem] = None
    A_host: Optional[np.ndarray] = None
    lam_exact: Optional[np.ndarray] = None

    def dense(self) -> np.ndarray:
        return self.A_host if self.A_host is not None else self.problem.dense()

    def dense_torch(self, device="cuda", out=None, sign: float = 1.0):
        import torch
        if self.problem is not None:
            return self.problem.dense_torch(device, out=out, sign=sign)
        At = torch.from_numpy(np.ascontiguousarray(self.A_host.T)).to(device) * sign
        if out is not None:
            out.copy_(At)
            return out.t()
        return At.t()


def make_config(index: int) -> Workload:
    """The five BASELINE.json configs."""
    if index == 0:
        p = bdg_uniform((8, 8, 8), 0.5, 0.2)
        return Workload(0, "cfg0_bdg_uniform_8x8x8", p.N, (p.N,), problem=p)
    if index == 1:
        A, lam = random_hermitian_clustered(4096, SEED_BASE + 1)
        return Workload(1, "cfg1_random_clustered_4096", 4096, (4096,), A_host=A, lam_exact=lam)
    if index == 2:
        p = bdg_single_vortex((16, 16, 16), 1.0, SEED_BASE + 2)
        return Workload(2, "cfg2_bdg_single_vortex_16x16x16", p.N, (p.N,), problem=p)
    if index == 3:
        p = bdg_vortex_tangle((24, 24, 24), 6, 1.0, SEED_BASE + 3, 0.02)
        return Workload(3, "cfg3_bdg_vortex_tangle_24x24x24", p.N, (p.N, p.N // 2), problem=p)
    if index == 4:
        p = bdg_vortex_tangle((32, 32, 24), 10, 1.2, SEED_BASE + 4, 0.02)
        return Workload(4, "cfg4_bdg_vortex_tangle_32x32x24", p.N, (p.N, p.N // 2), problem=p)
    raise ValueError(f"no config {index}")
