"""Pins for the oracle's fermion matrix.  CPU only."""
import numpy as np
import pytest

from oracle import dense_route
from paper_1005_3276_b200 import inputs


def _rand(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def _shift(psi, mu, step):
    """psi(x + step*mu) with the antiperiodic sign across the time wrap."""
    out = np.roll(psi, -step, axis=1 + mu)
    if mu == 0:
        T = psi.shape[1]
        idx = [slice(None)] * psi.ndim
        idx[1] = slice(T - 1, T) if step > 0 else slice(0, 1)
        out[tuple(idx)] *= -1
    return out


def test_stencil_identities(orc):
    # P2: F^-1[i sin p_mu F psi] = (psi(x+mu) - psi(x-mu))/2 ; F^-1[2 sum sin^2(p/2) F psi] = -1/2 lap psi
    dims = (4, 6, 4, 8)
    psi = _rand((4,) + dims, 11)
    f = orc.dft4d(psi, +1, True, "naive")
    n = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    p = [2 * np.pi * (n[0] + 0.5) / dims[0]] + [2 * np.pi * n[i] / dims[i] for i in (1, 2, 3)]
    for mu in range(4):
        got = orc.dft4d(1j * np.sin(p[mu]) * f, -1, True, "naive")
        want = 0.5 * (_shift(psi, mu, +1) - _shift(psi, mu, -1))
        assert np.abs(got - want).max() <= 1e-13
    got = orc.dft4d(2 * sum(np.sin(p[mu] / 2) ** 2 for mu in range(4)) * f, -1, True, "naive")
    want = -0.5 * sum(_shift(psi, mu, +1) + _shift(psi, mu, -1) - 2 * psi for mu in range(4))
    assert np.abs(got - want).max() <= 1e-13


def _momentum_route_matrix(orc, dims, phi, m, g, rho, dagger=False):
    V = int(np.prod(dims))
    cols = []
    for j in range(4 * V):
        e = np.zeros(4 * V, complex)
        e[j] = 1.0
        cols.append(orc.apply_M(phi, e.reshape((4,) + dims), m, g, rho, dagger, "naive").reshape(-1))
    return np.array(cols).T


@pytest.mark.parametrize("dims,rho", [((2, 2, 2, 2), 1.0), ((2, 2, 2, 2), 1.3), ((4, 2, 2, 4), 1.0)])
def test_dense_route_matches_momentum_route_small(orc, dims, rho):
    phi = inputs.make_phi(9, dims, 0.4)
    m, g = 0.2 + 0.1j, 0.5 - 0.3j
    M_dense = dense_route.fermion_matrix_dense(dims, phi, m, g, rho)
    M_mom = _momentum_route_matrix(orc, dims, phi, m, g, rho)
    assert np.abs(M_dense - M_mom).max() <= 1e-11 * np.abs(M_dense).max()
    Md_mom = _momentum_route_matrix(orc, dims, phi, m, g, rho, dagger=True)
    assert np.abs(M_dense.conj().T - Md_mom).max() <= 1e-11 * np.abs(M_dense).max()


def test_dense_route_4444_and_eq_2_20(orc):
    # P4 on the 4^4 lattice of config 1 (dimension 1024): apply to random vectors instead of all
    # unit vectors, and check Eq. (2.20) between the two dense forms of Dslash.
    dims = (4, 4, 4, 4)
    cfg = inputs.CONFIGS[1]
    phi = inputs.make_phi(cfg["seed"], dims, cfg["sigma"])
    lhs, rhs = dense_route.dslash_dense(dims, 1.0)
    assert np.abs(lhs - rhs).max() <= 1e-10 * np.abs(lhs).max()
    M = dense_route.fermion_matrix_dense(dims, phi, cfg["m"], cfg["g"], 1.0)
    for seed in (1, 2):
        v = _rand((4,) + dims, seed)
        want = (M @ v.reshape(-1)).reshape(v.shape)
        got = orc.apply_M(phi, v, cfg["m"], cfg["g"], 1.0, False, "naive")
        assert np.linalg.norm(got - want) <= 1e-11 * np.linalg.norm(want)
        want = (M.conj().T @ (M @ v.reshape(-1))).reshape(v.shape)
        got = orc.apply_MdagM(phi, v, cfg["m"], cfg["g"], 1.0, "naive")
        assert np.linalg.norm(got - want) <= 1e-11 * np.linalg.norm(want)
    # the solve: Cholesky on the dense normal equations vs the oracle's CG
    b = inputs.make_source(cfg["seed"], 0, dims)
    x_direct = dense_route.solve_normal_equations(M, b).reshape(b.shape)
    x_cg, info = orc.cg(phi, b, cfg["m"], cfg["g"], 1.0, 1e-12, 5000, "naive")
    assert info.converged
    evals = np.linalg.eigvalsh(M.conj().T @ M)
    kappa = evals[-1] / evals[0]
    assert np.linalg.norm(x_cg - x_direct) <= kappa * 1e-12 * np.linalg.norm(x_direct)
    assert evals[0] > 0


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 6, 16)])
def test_constant_phi_closed_form(orc, dims):
    # P5 (Eq. 7.11 generalised): phi = phi0 => M^dag M = d^2(p) + |w|^2
    m, g, phi0 = 0.1 + 0.05j, 0.7, 0.3 - 0.2j
    w = m + 2 * g * phi0
    phi = np.full(dims, phi0, complex)
    b = _rand((4,) + dims, 5)
    n = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    p = [2 * np.pi * (n[0] + 0.5) / dims[0]] + [2 * np.pi * n[i] / dims[i] for i in (1, 2, 3)]
    S2 = sum(np.sin(q) ** 2 for q in p)
    Mw = 1 - 2 * sum(np.sin(q / 2) ** 2 for q in p)
    d2 = (2 / (np.sqrt(Mw ** 2 + S2) + Mw)) ** 2 * S2
    bt = np.fft.fftn(b * np.exp(-1j * np.pi * np.arange(dims[0]) / dims[0])[None, :, None, None, None], axes=(1, 2, 3, 4))
    want = np.fft.ifftn(bt * (d2 + abs(w) ** 2), axes=(1, 2, 3, 4)) * np.exp(1j * np.pi * np.arange(dims[0]) / dims[0])[None, :, None, None, None]
    got = orc.apply_MdagM(phi, b, m, g, 1.0, "naive")
    assert np.linalg.norm(got - want) <= 1e-11 * np.linalg.norm(want)
    xw = np.fft.ifftn(bt / (d2 + abs(w) ** 2), axes=(1, 2, 3, 4)) * np.exp(1j * np.pi * np.arange(dims[0]) / dims[0])[None, :, None, None, None]
    x, info = orc.cg(phi, b, m, g, 1.0, 1e-13, 20000, "naive")
    assert info.converged
    assert np.linalg.norm(x - xw) <= 1e-9 * np.linalg.norm(xw)


def test_adjoint_hermiticity_positivity_gamma5(orc):
    # P6, P7
    dims = (4, 8, 4, 16)
    phi = inputs.make_phi(3, dims, 0.5)
    m, g = 0.05 + 0.02j, 1.0 + 0.4j
    u, v = _rand((4,) + dims, 1), _rand((4,) + dims, 2)
    for method in ("naive", "radix2"):
        Mv = orc.apply_M(phi, v, m, g, 1.0, False, method)
        Mdu = orc.apply_M(phi, u, m, g, 1.0, True, method)
        assert abs(np.vdot(u, Mv) - np.vdot(Mdu, v)) <= 1e-13 * abs(np.vdot(u, Mv)) + 1e-10
        Av = orc.apply_MdagM(phi, v, m, g, 1.0, method)
        Au = orc.apply_MdagM(phi, u, m, g, 1.0, method)
        assert abs(np.vdot(u, Av) - np.vdot(Au, v)) <= 1e-12 * abs(np.vdot(u, Av))
        assert abs(np.vdot(v, Av) - np.vdot(Mv, Mv)) <= 1e-12 * np.vdot(Mv, Mv).real
        assert np.vdot(v, Av).real > 0
    a = orc.apply_M(phi, v, m, g, 1.0, False, "naive")
    b = orc.apply_M(phi, v, m, g, 1.0, False, "radix2")
    assert np.linalg.norm(a - b) <= 1e-13 * np.linalg.norm(a)
    # real m, g and real phi: gamma5 M gamma5 = M^dag
    g5 = np.array([-1, -1, 1, 1]).reshape(4, 1, 1, 1, 1)
    phir = phi.real.astype(complex)
    left = g5 * orc.apply_M(phir, g5 * v, 0.05, 1.0, 1.0, False, "naive")
    right = orc.apply_M(phir, v, 0.05, 1.0, 1.0, True, "naive")
    assert np.linalg.norm(left - right) <= 1e-13 * np.linalg.norm(right)


def test_point_source_locality_probe(orc):
    # P9, Eq. 3.9-3.11 and the Fig. 1 caption: f(0) = 0, even r below odd r.
    dims = (16, 16, 16, 16)                                   # the lattice of Fig. 1
    eta = np.zeros((4,) + dims, complex)
    eta[2, 0, 0, 0, 0] = 1.0
    psi = orc.apply_M(np.zeros(dims, complex), eta, 0.0, 0.0, 1.0, False, "radix2")   # m = g = 0: M = Dslash
    nrm = np.sqrt((np.abs(psi) ** 2).sum(axis=0))
    assert nrm[0, 0, 0, 0] <= 1e-13
    x = np.meshgrid(*[np.minimum(np.arange(d), d - np.arange(d)) for d in dims], indexing="ij")
    r = sum(x)
    f = np.array([0.0] + [nrm[r == k].max() for k in range(1, 33)])   # f[r], r = 0..32
    assert f[1] == f.max()
    for k in range(4, 32, 2):                                  # even r lower than both odd neighbours
        assert f[k] < f[k - 1] and f[k] < f[k + 1]
    # long tail: far from exponential -- the last decade of r loses less than a factor 2
    assert f[31] > 0.5 * f[21]
