"""Writes tests/golden/G1.txt and G2.txt from DENSE matrix exponentials (scipy), not from any
pair-rotation code: the expected values are fixed by the mathematics of PAPER.md:61-89 under the
readings in DESIGN.md, independent of both the oracle and the CUDA path.

  G1: 4x4 closed, no potential, theta = 0.3, 3 steps, psi0 = delta at (x=1, y=2)
  G2: 4x4 periodic, V(x,y) = 0.1*(x + 2y), dt = 1, theta = 0.3, 3 steps, same delta
(the two worked examples of SURVEY.md 8(c); the paper itself prints no numerical example).

Run:  python tests/golden/make_golden.py
"""
from __future__ import annotations

import sys
from pathlib import Path

import numpy as np

sys.path.insert(0, str(Path(__file__).resolve().parents[1]))
from dense_ref import step_unitary  # noqa: E402

HERE = Path(__file__).resolve().parent


def _write(name, header, re, im):
    with open(HERE / name, "w") as f:
        f.write(header)
        f.write("# rows are y = 0..3, columns x = 0..3; first block Re, second block Im\n")
        for plane in (re, im):
            for row in plane:
                f.write(" ".join(f"{v:+.17e}" for v in row) + "\n")


def main():
    nx = ny = 4
    theta = 0.3
    psi0 = np.zeros(nx * ny, dtype=complex)
    psi0[2 * nx + 1] = 1.0

    U = step_unitary(nx, ny, False, theta)
    psi = np.linalg.matrix_power(U, 3) @ psi0
    _write("G1.txt",
           "# G1: 4x4 closed, pot NULL, theta=0.3, 3 steps, delta at (x=1,y=2). SURVEY.md 8(c);\n"
           "# dense product of expm(i*theta*A_part), PAPER.md:71-89 (Eq. 3).\n",
           psi.real.reshape(ny, nx), psi.imag.reshape(ny, nx))

    y, x = np.mgrid[0:ny, 0:nx]
    V = 0.1 * (x + 2 * y)
    U = step_unitary(nx, ny, True, theta, V=V, dt=1.0)
    psi = np.linalg.matrix_power(U, 3) @ psi0
    _write("G2.txt",
           "# G2: 4x4 periodic, V=0.1*(x+2y), dt=1, theta=0.3, 3 steps, delta at (x=1,y=2).\n"
           "# dense product with diag(exp(-iV)) at the centre, PAPER.md:65-69, 85-89.\n",
           psi.real.reshape(ny, nx), psi.imag.reshape(ny, nx))


if __name__ == "__main__":
    main()
