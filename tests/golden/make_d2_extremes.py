#!/usr/bin/env python
"""Regenerates the numbers of tests/golden/d2_extremes.txt WITHOUT the oracle (numpy only), so that the
file pins oracle/wz_oracle.cpp:orc_dslash_d2_extremes from outside.

    python tests/golden/make_d2_extremes.py          # prints the table rows

d^2(p) = Dslash(p)^dag Dslash(p) over the antiperiodic-time momentum lattice, two routes:
  (1) every momentum: the scalar form that follows from PAPER.md:210-225 Eq. (3.1), (3.3) and 382-390
      Eq. (4.1)-(4.2):  S2 = sum sin^2 p,  Mw = 1 - 2 sum sin^2(p/2),  s = sqrt(Mw^2 + S2),
      d^2 = S2 / (1/2 + Mw/(2s))^2 / s^2   [= |D1|^2 / (1 - D2/2)^2, straight from the two printed symbols];
  (2) at the two extremal momenta only: Eq. (2.9) and 170-178 Eq. (2.19)-(2.20) by 4x4 matrix
      algebra (A = 1 - D_W on a plane wave, D = 1 - A (A^dag A)^(-1/2), Dslash = (1 - D/2)^(-1) D), as a
      cross-check of route (1).
"""
import numpy as np

LATTICES = [(4, 4, 4, 4), (8, 8, 8, 8), (16, 16, 16, 16), (32, 32, 32, 32), (48, 24, 24, 24), (64, 64, 64, 64)]


def gammas():
    s = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]], complex), np.array([[1, 0], [0, -1]], complex)]
    z, one = np.zeros((2, 2), complex), np.eye(2, dtype=complex)
    return [np.block([[z, one], [one, z]])] + [np.block([[z, 1j * k], [-1j * k, z]]) for k in s]


def d2_matrix(p):
    g = gammas()
    A = np.eye(4, dtype=complex)
    for mu in range(4):
        fwd, bwd = np.exp(1j * p[mu]) - 1.0, 1.0 - np.exp(-1j * p[mu])
        A -= g[mu] * 0.5 * (fwd + bwd) - np.eye(4) * 0.5 * (bwd * fwd)
    w, v = np.linalg.eigh(A.conj().T @ A)
    D = np.eye(4) - A @ (v @ np.diag(w ** -0.5) @ v.conj().T)
    Ds = np.linalg.solve(np.eye(4) - 0.5 * D, D)
    return float(np.linalg.eigvalsh(Ds.conj().T @ Ds).max())


def main():
    for dims in LATTICES:
        p = [2 * np.pi * (np.arange(L) + (0.5 if mu == 0 else 0.0)) / L for mu, L in enumerate(dims)]
        P = np.meshgrid(*p, indexing="ij", sparse=True)
        S2 = sum(np.sin(x) ** 2 for x in P)
        Mw = 1.0 - 2.0 * sum(np.sin(x / 2) ** 2 for x in P)
        s = np.sqrt(Mw ** 2 + S2)
        half = 0.5 + Mw / (2 * s)                      # (1 - D2/2)(p), Eq. (3.1); its zeros sit at the would-be
        with np.errstate(divide="ignore", invalid="ignore"):   # doublers, which the half-integer p0 avoids
            d2 = S2 / s ** 2 / half ** 2
        lo, hi = float(np.nanmin(d2)), float(np.nanmax(d2))
        ilo, ihi = np.unravel_index(np.nanargmin(d2), d2.shape), np.unravel_index(np.nanargmax(d2), d2.shape)
        for val, idx in ((lo, ilo), (hi, ihi)):
            pm = [p[mu][idx[mu]] for mu in range(4)]
            assert abs(d2_matrix(pm) - val) <= 1e-7 * val, (dims, val, d2_matrix(pm))
        print("%d %d %d %d %.5g %.6g" % (dims + (lo, hi)))


if __name__ == "__main__":
    main()
