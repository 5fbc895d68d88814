"""Writes tests/golden/ed_energies.txt.  Calls only oracle/ (never the CUDA path)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from oracle import fock, lattice  # noqa: E402

rows = []
for L, N in ((3, 4), (3, 5), (4, 8)):
    T, V, mc = lattice.spinless_tV(L, 1.0, 0.4, 0.8)
    rows.append((f"spinless_{L}x{L}_N{N}", fock.ground_energy(T, V, mc, (N,))))
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "ed_energies.txt"), "w") as f:
    f.write("# name | E0 | Eq. (3) PAPER.md:70, t=1 t'=0.4 V=0.8 (PAPER.md:34), torus, snake order; oracle.fock.ground_energy\n")
    for name, e in rows:
        f.write(f"{name} | {e:.12f}\n")
print(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "ed_energies.txt")).read())
