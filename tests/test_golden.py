"""Stored expected values (tests/golden/, written by tests/golden/make_golden.py from oracle/ only, or printed in the
paper): CPU tests tie them to closed forms and to the paper's number; GPU tests compare the CUDA path with them."""
import os

import numpy as np
import pytest

from paper_2310_03341_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _config0_spectrum():
    rows = [l.split() for l in open(os.path.join(GOLD, "config0_spectrum.txt")) if not l.startswith("#")]
    vals = np.array([float(r[0]) for r in rows])
    mult = np.array([int(r[1]) for r in rows])
    return vals, mult


def _vortex_fields():
    E, F, sec = [], [], None
    for l in open(os.path.join(GOLD, "vortex_4x4x6_fields.txt")):
        if l.startswith("#"):
            continue
        l = l.strip()
        if l in ("E", "F"):
            sec = l
        elif sec == "E":
            E.append(float(l))
        else:
            t = l.split()
            F.append((float(t[1]), float(t[2]) + 1j * float(t[3])))
    return np.array(E), np.array([f[0] for f in F]), np.array([f[1] for f in F])


def test_config0_golden_is_the_closed_form():
    """64 distinct values, multiplicities summing to 1024, equal to +-sqrt((eps_k - mu)^2 + Delta^2)."""
    vals, mult = _config0_spectrum()
    assert vals.size == 64 and mult.sum() == 1024 and mult.max() == 48
    ks = [2 * np.pi * np.arange(-4, 4) / 8] * 3
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    E = np.sqrt((0.5 * (KX ** 2 + KY ** 2 + KZ ** 2).reshape(-1) - 0.5) ** 2 + 0.04)
    ref = np.sort(np.concatenate([-E, E]))
    assert np.abs(np.repeat(vals, mult) - ref).max() <= 1e-12 * np.abs(ref).max()


def test_paper_fraction_of_states_below_the_cutoff():
    """PAPER.md:35 / :127: N_qpwf ~ 0.5 N^3 states lie below E_c = pi^2 / 2.  With Delta -> 0 and mu = 0
    the quasiparticle energies are the kinetic energies |k|^2 / 2 on the grid of PAPER.md:113, so the number of columns
    the density sums keep (0 < E < E_c), as a fraction of the lattice points, must reproduce the printed 0.5 (pi/6 in the
    continuum) -- here through the oracle chain assemble -> eigenvalues -> the oracle's own cutoff rule."""
    import oracle
    from oracle import assemble as oa
    from oracle import densities as od
    printed = float([l.split()[1] for l in open(os.path.join(GOLD, "paper_nqpwf.txt")) if l.startswith("fraction_printed")][0])
    shape = (8, 8, 8)
    M = 512
    Ks = [wl.kinetic_1d(L) for L in shape]
    H = oa.assemble_bdg(*Ks, np.zeros(M), np.full(M, 1e-6), 0.0)
    E, Z = oracle.eigh(H)
    Ec = np.pi ** 2 / 2
    n_all, _ = od.densities(E, Z, T=1e12)                    # f = 1/2: n(r) = sum over kept states of |u|^2 + |v|^2
    n_cut, _ = od.densities(E, Z, T=1e12, Ec=Ec)
    kept = n_cut.sum() / n_all.sum() * M                     # number of kept states (each is normalised)
    assert abs(kept - np.count_nonzero((E > 0) & (E < Ec))) <= 1e-8
    assert abs(kept / M - printed) <= 0.05
    assert abs(kept / M - np.pi / 6) <= 0.05                 # 251 of 512 on the 8^3 lattice


def test_vortex_golden_is_consistent():
    """Particle-hole symmetric spectrum, n in [0, 2], and the stored fields are what the oracle gives today."""
    import oracle
    from oracle import assemble as oa
    from oracle import densities as od
    E, n, nu = _vortex_fields()
    assert E.size == 192 and n.size == 96
    assert np.abs(E + E[::-1]).max() <= 1e-12 * np.abs(E).max()
    assert n.min() >= 0 and n.max() <= 2
    q = wl.bdg_vortex_tangle((4, 4, 6), 3, 1.0, wl.SEED_BASE + 3, 0.02)
    H = oa.assemble_bdg(*[wl.kinetic_1d(L) for L in q.shape], q.V, q.Delta, q.mu)
    E2, Z2 = oracle.eigh(H)
    n2, nu2 = od.densities(E2, Z2, T=0.05, Ec=6.0)
    assert np.abs(E2 - E).max() <= 1e-13 * np.abs(E).max()
    assert np.abs(n2 - n).max() <= 1e-13 and np.abs(nu2 - nu).max() <= 1e-13


@pytest.mark.gpu
def test_gpu_config0_against_golden():
    import torch
    from paper_2310_03341_b200 import binding
    vals, mult = _config0_spectrum()
    p = wl.bdg_uniform((8, 8, 8), 0.5, 0.2)
    eng = binding.Eigh(p.N)
    At = torch.from_numpy(np.ascontiguousarray(p.dense().T)).cuda()
    W, _ = eng.solve(At)
    torch.cuda.synchronize()
    eng.close()
    ref = np.repeat(vals, mult)
    assert np.abs(W.cpu().numpy() - ref).max() <= 1e-11 * np.abs(ref).max()


@pytest.mark.gpu
def test_gpu_scf_chain_against_golden():
    import torch
    from paper_2310_03341_b200 import binding
    E, n, nu = _vortex_fields()
    q = wl.bdg_vortex_tangle((4, 4, 6), 3, 1.0, wl.SEED_BASE + 3, 0.02)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()   # noqa: E731
    eng = binding.Eigh(q.N)
    Ks = [dev(wl.kinetic_1d(L)) for L in q.shape]
    At = eng.assemble_bdg(q.shape, *Ks, dev(q.V), dev(q.Delta), q.mu)
    W, Zt = eng.solve(At)
    n_g, nu_g = eng.densities(W, Zt, T=0.05, Ec=6.0)
    torch.cuda.synchronize()
    eng.close()
    assert np.abs(W.cpu().numpy() - E).max() <= 1e-11 * np.abs(E).max()
    assert np.abs(n_g.cpu().numpy() - n).max() <= 1e-10
    assert np.abs(nu_g.cpu().numpy() - nu).max() <= 1e-10
