#!/usr/bin/env python
"""Writes tests/golden/vg_table.txt: values of the exchange kernel v(G) in 40-digit decimal arithmetic.

Formulas (BASELINE.json north_star; "kernel for the (possibly screened) electron-electron interaction",
PAPER.md:61 "Poisson-like equations"; readings Q2/Q3 of DESIGN.md):
    bare Coulomb : v(G) = 4 pi / |G|^2,                                  v(0) = 0
    HSE-screened : v(G) = 4 pi / |G|^2 * (1 - exp(-|G|^2 / (4 omega^2))),  v(0) = pi / omega^2   (the G -> 0 limit)
with G = 2 pi (m0/L0, m1/L1, m2/L2) for an orthorhombic cell.  Pure Python `decimal`; uses nothing from oracle/ or the
CUDA path, so the table pins both.  Run from the repo root:  python tests/golden/make_vg_table.py
"""
import os
from decimal import Decimal as D, getcontext

getcontext().prec = 50
PI = D("3.14159265358979323846264338327950288419716939937510")
OMEGA = D("0.106")                      # bohr^-1 (BASELINE.json configs)
CELLS = {"Si8": ("10.26", "10.26", "10.26"), "Si1536": ("82.08", "82.08", "30.78"), "Si1536p": ("82.08", "61.56", "41.04")}
MS = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 1), (-1, 2, 0), (3, -2, 1), (7, 0, -7), (-8, 5, 3), (0, -8, 8)]


def v(kernel, L, m):
    g2 = sum((2 * PI * D(mi) / D(Li)) ** 2 for mi, Li in zip(m, L))
    if g2 == 0:
        return D(0) if kernel == "coulomb" else PI / OMEGA ** 2
    val = 4 * PI / g2
    if kernel == "hse":
        val *= 1 - (-g2 / (4 * OMEGA ** 2)).exp()
    return val


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "vg_table.txt")
    with open(out, "w") as f:
        f.write("# kernel cell L0 L1 L2 m0 m1 m2 v(G)   [bohr, bohr^2]; written by tests/golden/make_vg_table.py (40 digits)\n")
        for kernel in ("coulomb", "hse"):
            for name, L in CELLS.items():
                for m in MS:
                    f.write(f"{kernel} {name} {L[0]} {L[1]} {L[2]} {m[0]} {m[1]} {m[2]} {v(kernel, L, m):.40E}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
