"""Writes tests/golden/hydrogen_energies.txt from the closed-form Dirac-Coulomb (Sommerfeld) levels

    E_{n,kappa} = c^2 [ (1 + (Z alpha / (n - |kappa| + sqrt(kappa^2 - Z^2 alpha^2)))^2)^(-1/2) - 1 ],  alpha = 1/c,

energies relative to the rest energy as in PAPER.md:79-81 (beta shifted by -c^2); for 1s1/2 this is
c^2 (sqrt(1 - (Z/c)^2) - 1) quoted in BASELINE.json north_star.  40-digit decimal arithmetic; calls
nothing from oracle/ or the CUDA package.  Run:  python tests/golden/make_hydrogen_energies.py
"""
from decimal import Decimal, getcontext
import os

getcontext().prec = 40
C = Decimal("137.035999084")
Z = Decimal(1)


def level(n: int, kappa: int) -> Decimal:
    za = Z / C
    gam = (Decimal(kappa * kappa) - za * za).sqrt()
    den = Decimal(n - abs(kappa)) + gam
    return C * C * (1 / (1 + (za / den) ** 2).sqrt() - 1)


LEVELS = [("1s1/2", 1, -1), ("2s1/2", 2, -1), ("2p1/2", 2, 1), ("2p3/2", 2, -2), ("3s1/2", 3, -1),
          ("3p1/2", 3, 1), ("3p3/2", 3, -2), ("3d3/2", 3, 2), ("3d5/2", 3, -3), ("4f5/2", 4, 3),
          ("4f7/2", 4, -4), ("5g7/2", 5, 4)]

if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "hydrogen_energies.txt")
    with open(out, "w") as f:
        f.write("# Closed-form Dirac hydrogen levels (a.u., rest energy removed), Z=1, c=137.035999084\n")
        f.write("# source: Sommerfeld fine-structure formula; written by make_hydrogen_energies.py\n")
        f.write("# label n kappa energy\n")
        for lab, n, k in LEVELS:
            f.write(f"{lab} {n} {k} {level(n, k):.25f}\n")
    print(open(out).read())
