"""Dense position-space route to the fermion matrix (oracle route O3; tiny lattices only).

TEST INFRASTRUCTURE ONLY.  No Fourier transform appears anywhere in this file:
the operator is assembled from difference matrices exactly as PAPER.md:89-98
Eq. (2.9) and 170-178 Eq. (2.19)-(2.20) write it, with numpy.linalg as the
library primitive for the matrix inverse square root, the inverse and the solve.
It exists to pin oracle/wz_oracle.cpp's momentum route (which uses the FFT trick
of PAPER.md:896 and the closed-form symbol) on 2^4 and 4^4 lattices.

Vector index = spin * V + site, site = ((x0*L1 + x1)*L2 + x2)*L3 + x3.
"""
from __future__ import annotations

import numpy as np


def gammas():
    """PAPER.md:43-47 Eq. (2.2), typed independently of wz_oracle.cpp."""
    s1 = np.array([[0, 1], [1, 0]], dtype=complex)
    s2 = np.array([[0, -1j], [1j, 0]], dtype=complex)
    s3 = np.array([[1, 0], [0, -1]], dtype=complex)
    z = np.zeros((2, 2), dtype=complex)
    one = np.eye(2, dtype=complex)
    g0 = np.block([[z, one], [one, z]])
    gi = [np.block([[z, 1j * s], [-1j * s, z]]) for s in (s1, s2, s3)]
    g5 = np.diag([-1.0, -1.0, 1.0, 1.0]).astype(complex)
    return [g0] + gi, g5


def difference_matrices(dims):
    """Forward (d) and backward (d*) difference matrices per axis, V x V.

    (d psi)(x) = psi(x + mu) - psi(x), (d* psi)(x) = psi(x) - psi(x - mu);
    the fermion is antiperiodic in time, periodic in space:
    psi(x0 = T) = -psi(x0 = 0).
    """
    dims = tuple(int(d) for d in dims)
    V = int(np.prod(dims))
    idx = np.arange(V).reshape(dims)
    fwd, bwd = [], []
    for mu in range(4):
        F = -np.eye(V)
        B = np.eye(V)
        for x in np.ndindex(*dims):
            here = idx[x]
            xp = list(x)
            xp[mu] += 1
            sign = 1.0
            if xp[mu] == dims[mu]:
                xp[mu] = 0
                sign = -1.0 if mu == 0 else 1.0
            F[here, idx[tuple(xp)]] += sign
            xm = list(x)
            xm[mu] -= 1
            sign = 1.0
            if xm[mu] < 0:
                xm[mu] = dims[mu] - 1
                sign = -1.0 if mu == 0 else 1.0
            B[here, idx[tuple(xm)]] -= sign
        fwd.append(F)
        bwd.append(B)
    return fwd, bwd


def overlap_pieces(dims, rho=1.0):
    """A, D, D1, D2 of Eq. (2.9) as dense 4V x 4V matrices (a = 1).

    D_W = 1/2 gamma_mu (d*_mu + d_mu) - 1/2 d*_mu d_mu   (Wilson sign: DESIGN.md reading G1)
    A = rho - D_W;  D = rho (1 - A (A^dag A)^(-1/2))     (rho: reading G2)
    D1 = 1/2 gamma_mu (d* + d) (A^dag A)^(-1/2) * rho,  D2 = rho [1 - (rho + 1/2 d* d)(A^dag A)^(-1/2)].
    """
    gam, _ = gammas()
    fwd, bwd = difference_matrices(dims)
    V = fwd[0].shape[0]
    one4 = np.eye(4)
    nabla = sum(np.kron(gam[mu], 0.5 * (bwd[mu] + fwd[mu])) for mu in range(4))
    lap = sum(bwd[mu] @ fwd[mu] for mu in range(4))
    DW = nabla - 0.5 * np.kron(one4, lap)
    A = rho * np.eye(4 * V) - DW
    AdA = A.conj().T @ A
    evals, evecs = np.linalg.eigh(AdA)
    inv_sqrt = (evecs * (1.0 / np.sqrt(evals))) @ evecs.conj().T
    D = rho * (np.eye(4 * V) - A @ inv_sqrt)
    D1 = rho * nabla @ inv_sqrt
    D2 = rho * (np.eye(4 * V) - np.kron(one4, rho * np.eye(V) + 0.5 * lap) @ inv_sqrt)
    return A, D, D1, D2


def dslash_dense(dims, rho=1.0):
    """Dslash = (1 - D2/2rho)^(-1) D1 (Eq. 2.19), and the right side of Eq. (2.20)."""
    _, D, D1, D2 = overlap_pieces(dims, rho)
    n = D.shape[0]
    lhs = np.linalg.solve(np.eye(n) - D2 / (2.0 * rho), D1)
    rhs = np.linalg.solve(np.eye(n) - D / (2.0 * rho), D)
    return lhs, rhs


def fermion_matrix_dense(dims, phi, m, g, rho=1.0):
    """M of Eq. (2.19): Dslash + m P+ + m* P- + 2 g phi P+ + 2 g* phi* P-."""
    dslash, _ = dslash_dense(dims, rho)
    V = int(np.prod(dims))
    w = complex(m) + 2.0 * complex(g) * np.asarray(phi, dtype=complex).reshape(V)
    _, g5 = gammas()
    Pp = 0.5 * (np.eye(4) + g5)
    Pm = 0.5 * (np.eye(4) - g5)
    M = dslash + np.kron(Pp, np.diag(w)) + np.kron(Pm, np.diag(w.conj()))
    return M


def solve_normal_equations(M, b):
    """x = (M^dag M)^(-1) b by Cholesky (M^dag M is Hermitian positive definite)."""
    A = M.conj().T @ M
    Lc = np.linalg.cholesky(A)
    y = np.linalg.solve(Lc, np.asarray(b, dtype=complex).reshape(-1))
    return np.linalg.solve(Lc.conj().T, y)
