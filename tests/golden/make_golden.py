"""Writes the stored expected values under tests/golden/ -- calls ONLY oracle/ and the seeded input generators.

    python tests/golden/make_golden.py

config0_spectrum.txt      eigenvalues of BASELINE.json config 0 (uniform-pairing BdG, 8x8x8, N = 1024) by oracle.eigh
                          (Householder tridiagonalisation + implicit QL), distinct values with multiplicities.
vortex_4x4x6_fields.txt   E_n, n(r), nu(r) of the 4x4x6 vortex-tangle problem at T = 0.05, E_c = 6 by the oracle chain
                          assemble_bdg -> eigh -> densities (PAPER.md:103-107 Eq. 5/7, :300-311 Eq. 16a/16d/17).
paper_nqpwf.txt is NOT written here: it holds a number printed in the paper.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from oracle import assemble as oa  # noqa: E402
from oracle import densities as od  # noqa: E402
from paper_2310_03341_b200 import workloads as wl  # noqa: E402


def main():
    p = wl.bdg_uniform((8, 8, 8), 0.5, 0.2)
    W = oracle.eigh(p.dense(), vectors=False)
    groups = []
    for x in W:
        if groups and abs(x - groups[-1][0] / groups[-1][1]) <= 1e-9:
            groups[-1][0] += x
            groups[-1][1] += 1
        else:
            groups.append([x, 1])
    with open(os.path.join(HERE, "config0_spectrum.txt"), "w") as f:
        f.write("# config 0 (BASELINE.json): BdG uniform pairing, 8x8x8, mu = 0.5, Delta = 0.2, N = 1024\n")
        f.write("# written by tests/golden/make_golden.py from oracle.eigh; columns: mean eigenvalue of the shell, multiplicity\n")
        for s, m in groups:
            f.write(f"{s / m:.17e} {m}\n")

    q = wl.bdg_vortex_tangle((4, 4, 6), 3, 1.0, wl.SEED_BASE + 3, 0.02)
    Ks = [wl.kinetic_1d(L) for L in q.shape]
    H = oa.assemble_bdg(*Ks, q.V, q.Delta, q.mu)
    E, Z = oracle.eigh(H)
    n, nu = od.densities(E, Z, T=0.05, Ec=6.0)
    with open(os.path.join(HERE, "vortex_4x4x6_fields.txt"), "w") as f:
        f.write("# bdg_vortex_tangle((4,4,6), 3 lines, mu = 1.0, seed = SEED_BASE + 3, noise 0.02): oracle chain\n")
        f.write("# assemble_bdg -> eigh -> densities(T = 0.05, Ec = 6); written by tests/golden/make_golden.py\n")
        f.write("# section E: 192 eigenvalues; section F: r, n(r), Re nu(r), Im nu(r) for the 96 grid points\n")
        f.write("E\n")
        for x in E:
            f.write(f"{x:.17e}\n")
        f.write("F\n")
        for r in range(n.size):
            f.write(f"{r} {n[r]:.17e} {nu[r].real:.17e} {nu[r].imag:.17e}\n")


if __name__ == "__main__":
    main()
