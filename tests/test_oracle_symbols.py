"""Pins for the momentum-space symbols (PAPER.md identities T1-T10)."""
import os

import numpy as np
import pytest

from oracle import dense_route

HERE = os.path.dirname(os.path.abspath(__file__))


def _momenta(dims, count, seed):
    """Random lattice momenta with half-integer time component."""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(count):
        n = [rng.integers(0, d) for d in dims]
        out.append(np.array([2 * np.pi * (n[0] + 0.5) / dims[0]] + [2 * np.pi * n[i] / dims[i] for i in (1, 2, 3)]))
    return out


def test_gamma_algebra(orc):
    gam = [orc.gamma(mu) for mu in range(4)]
    g5 = orc.gamma(5)
    ref, ref5 = dense_route.gammas()       # typed independently from Eq. (2.2)
    for mu in range(4):
        assert np.array_equal(gam[mu], ref[mu])
        assert np.allclose(gam[mu], gam[mu].conj().T)
        assert np.allclose(gam[mu] @ g5 + g5 @ gam[mu], 0)
        for nu in range(4):
            assert np.allclose(gam[mu] @ gam[nu] + gam[nu] @ gam[mu], 2 * np.eye(4) * (mu == nu))
    assert np.array_equal(g5, ref5)
    assert np.allclose(np.diag(g5), [-1, -1, 1, 1])


@pytest.mark.parametrize("rho", [1.0, 0.7, 1.4])
def test_symbol_identities(orc, rho):
    g5 = orc.gamma(5)
    gam = [orc.gamma(mu) for mu in range(4)]
    one = np.eye(4)
    for p in _momenta((8, 6, 4, 16), 40, 7) + [np.array([0.3, -1.1, 2.9, 0.05])]:
        D, D1, D2 = orc.overlap_D_symbol(p, rho)
        ds = orc.dslash_symbol(p, rho)
        sn = np.sin(p)
        Mw = rho - 2 * (np.sin(p / 2) ** 2).sum()
        s = np.sqrt(Mw ** 2 + (sn ** 2).sum())
        X = sum(gam[mu] * sn[mu] for mu in range(4))
        # T1, Eq. (3.1): (1 - D2/2rho)(p) = 1/2 + Mw/(2s)
        assert np.allclose(one - D2 / (2 * rho), (0.5 + Mw / (2 * s)) * one, atol=1e-13)
        # T2, Eq. (3.3) with the sign of reading G3: D1(p) = + i rho X / s on exp(+ipx)
        assert np.allclose(D1, 1j * rho * X / s, atol=1e-13)
        # Ginsparg-Wilson:  gamma5 D + D gamma5 = (1/rho) D gamma5 D
        assert np.allclose(g5 @ D + D @ g5, D @ g5 @ D / rho, atol=1e-12)
        # T4, Eq. (3.6)/(2.18):  D1^2 - D2^2 = -2 rho D2,  D^dag D = 2 rho D2
        assert np.allclose(D1 @ D1 - D2 @ D2, -2 * rho * D2, atol=1e-12)
        assert np.allclose(D.conj().T @ D, 2 * rho * D2, atol=1e-12)
        # definition of Dslash, Eq. (2.19), and identity T5, Eq. (2.20)
        lhs = np.linalg.solve(one - D2 / (2 * rho), D1)
        rhs = np.linalg.solve(one - D / (2 * rho), D)
        scale = np.abs(lhs).max()
        assert np.abs(ds - lhs).max() <= 1e-12 * scale
        assert np.abs(ds - rhs).max() <= 1e-11 * scale
        # T3, Eq. (3.4): anticommutes with gamma5; anti-Hermitian; Dslash^dag Dslash scalar
        assert np.abs(ds @ g5 + g5 @ ds).max() <= 1e-13 * scale
        assert np.abs(ds + ds.conj().T).max() <= 1e-13 * scale
        d2 = (ds.conj().T @ ds)[0, 0].real
        assert np.abs(ds.conj().T @ ds - d2 * one).max() <= 1e-12 * d2
        # T6, Eq. (3.5) and T7, Eq. (7.11), for a complex mass
        m = 0.3 - 0.2j
        Pp, Pm = (one + g5) / 2, (one - g5) / 2
        M0 = ds + m * Pp + np.conj(m) * Pm
        left = (-D1 + (one - D2 / (2 * rho)) @ (np.conj(m) * Pp + m * Pm)) @ M0
        right = 2 * D2 / rho * rho + abs(m) ** 2 * (one - D2 / (2 * rho))
        if rho == 1.0:
            assert np.abs(left - right).max() <= 1e-11 * max(1.0, np.abs(right).max())
        assert np.abs(M0.conj().T @ M0 - (d2 + abs(m) ** 2) * one).max() <= 1e-12 * (d2 + 1)
        assert np.abs(np.linalg.inv(M0) - M0.conj().T / (d2 + abs(m) ** 2)).max() <= 1e-11 * np.abs(np.linalg.inv(M0)).max()


def test_small_momentum_limit(orc):
    # T10, Eq. (3.18): D1 -> gamma.d, i.e. Dslash(p) -> i gamma.p
    gam = [orc.gamma(mu) for mu in range(4)]
    p = 1e-4 * np.array([0.3, -0.7, 0.2, 0.5])
    ds = orc.dslash_symbol(p, 1.0)
    want = 1j * sum(gam[mu] * p[mu] for mu in range(4))
    assert np.abs(ds - want).max() <= 1e-8 * np.abs(want).max()


def test_stable_branch_near_doublers(orc):
    # for Mw < 0 the closed form 2 rho/(s + Mw) cancels; the oracle's value must
    # agree with extended-precision evaluation of the same formula.
    for p in [np.array([np.pi - 1e-3, 0.0, 0.0, 0.0]), np.array([np.pi - 0.05, np.pi, 0.1, 0.0]),
              np.array([np.pi * 63 / 64, np.pi, np.pi, np.pi])]:
        pl = p.astype(np.longdouble)
        S2 = (np.sin(pl) ** 2).sum()
        Mw = 1 - 2 * (np.sin(pl / 2) ** 2).sum()
        s = np.sqrt(Mw * Mw + S2)
        c = 2 * (s - Mw) / S2
        d2 = float(c * c * S2)
        ds = orc.dslash_symbol(p, 1.0)
        got = (ds.conj().T @ ds)[0, 0].real
        assert abs(got - d2) <= 1e-13 * d2


def test_dslash_finite_on_apbc_lattice_and_golden_extremes(orc):
    # T8/T9 and pin P8 (tests/golden/d2_extremes.txt)
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "d2_extremes.txt")) if l.strip() and l[0] != "#"]
    for row in rows:
        dims = tuple(int(v) for v in row[:4])
        lo, hi = orc.d2_extremes(dims, 1.0, True)
        assert abs(lo - float(row[4])) <= 5e-5 * float(row[4])  # 5 significant figures
        assert abs(hi - float(row[5])) <= 5e-5 * float(row[5])
        # closed form of the minimum: p = (pi/T, 0, 0, 0)
        T = dims[0]
        sp = np.sin(np.pi / T)
        Mw = 1 - 2 * np.sin(np.pi / (2 * T)) ** 2
        s = np.sqrt(Mw ** 2 + sp ** 2)
        assert abs(lo - (2 * sp / (s + Mw)) ** 2) <= 1e-12
        assert 0.5 * (28 * T / np.pi) ** 2 < hi < 1.5 * (28 * T / np.pi) ** 2
