"""Pins of the oracle's preconditioned shifted solve and of the rational sum
(Eq. 7.6-7.7, 927-933 Eq. 7.13-7.14, 948 cutoff rule)."""
import numpy as np

from paper_1005_3276_b200 import inputs


def rel(a, ref):
    return float(np.linalg.norm((a - ref).ravel()) / np.linalg.norm(ref.ravel()))


def _dense_A(dims, phi, m, g):
    from oracle import dense_route

    M = dense_route.fermion_matrix_dense(dims, phi, m, g, 1.0)
    return M.conj().T @ M


def test_shift_pc_solution_equals_dense_solve(orc):
    """Eq. 7.14 is Eq. 7.13 in other variables: its x = M0^-1 xtilde must solve (M^dag M + sigma) x = b.
    Dense position-space route (no Fourier transform anywhere), sigma below and above the cutoff."""
    dims = (4, 4, 4, 4)
    phi = inputs.make_phi(1, dims, 0.3)
    b = inputs.make_source(1, 0, dims)
    for m, g in ((1.0, 0.2), (0.1 + 0.05j, 0.5 - 0.1j)):
        A = _dense_A(dims, phi, m, g)
        for sigma in (0.0, 0.3, 25.0, 400.0):
            x, info = orc.cg_shift_pc(phi, b, m, g, sigma, 1.0, 1e-12, 5000)
            xd = np.linalg.solve(A + sigma * np.eye(A.shape[0]), b.reshape(-1)).reshape(b.shape)
            assert info.converged and rel(x, xd) < 1e-9, (m, g, sigma, rel(x, xd))
            assert info.rel_residual_true < 1e-9


def test_shift_zero_is_the_preconditioned_solve(orc):
    dims = (8, 4, 4, 4)
    phi = inputs.make_phi(2, dims, 0.3)
    b = inputs.make_source(2, 0, dims)
    x0, i0 = orc.cg_pc(phi, b, 1.0, 0.2, 1.0, 1e-12, 500)
    x1, i1 = orc.cg_shift_pc(phi, b, 1.0, 0.2, 0.0, 1.0, 1e-12, 500)
    assert i0.iterations == i1.iterations and rel(x1, x0) < 1e-13


def test_free_field_converges_in_one_iteration_at_any_shift(orc):
    """g = 0: Mtilde = 1 and (M0^-1)^dag M0^-1 = 1/(d^2(p) + |m|^2) is momentum-diagonal, so the operator
    of Eq. 7.14 is 1 + sigma/(d^2 + |m|^2).  With sigma = 0 it is the identity: CG stops after ONE step;
    with sigma > 0 it is not a multiple of the identity and needs more -- the 'degradation of the
    speedup for larger beta_i' of PAPER.md:948."""
    dims = (8, 4, 4, 4)
    phi = inputs.make_phi(3, dims, 0.3)
    b = inputs.make_source(3, 0, dims)
    _, i0 = orc.cg_shift_pc(phi, b, 1.0, 0.0, 0.0, 1.0, 1e-12, 100)
    _, i1 = orc.cg_shift_pc(phi, b, 1.0, 0.0, 5.0, 1.0, 1e-12, 100)
    assert i0.iterations == 1 and i1.iterations > 1


def test_cutoff_regime_of_table_VII(orc):
    """PAPER.md:948-950 (m = 1, g = 0.1, Table VII): with preconditioning up to beta = 100 and plain CG
    above, every one of the d = 20 problems stays under 100 iterations at 1e-6 (the paper's single-precision
    criterion) and under 200 at 1e-12; preconditioning wins at small beta, plain CG at very large beta."""
    dims = (8, 4, 4, 4)
    phi = inputs.make_phi(4, dims, 0.3)
    b = inputs.make_source(4, 0, dims)
    _, _, betas = inputs.rational_ladder(20, 1e-2, 1e3)
    for tol, cap in ((1e-6, 100), (1e-12, 200)):
        for beta in betas:
            if beta <= 100.0:
                _, info = orc.cg_shift_pc(phi, b, 1.0, 0.1, float(beta), 1.0, tol, 1000)
            else:
                _, info = orc.cg_shift(phi, b, 1.0, 0.1, float(beta), 1.0, tol, 1000)
            assert info.converged and info.iterations < cap, (tol, beta, info.iterations)
    small, large = float(betas[0]), float(betas[-1])
    assert orc.cg_shift_pc(phi, b, 1.0, 0.1, small, 1.0, 1e-6, 5000)[1].iterations < \
        orc.cg_shift(phi, b, 1.0, 0.1, small, 1.0, 1e-6, 5000)[1].iterations
    assert orc.cg_shift(phi, b, 1.0, 0.1, large, 1.0, 1e-6, 5000)[1].iterations <= \
        orc.cg_shift_pc(phi, b, 1.0, 0.1, large, 1.0, 1e-6, 5000)[1].iterations


def test_rational_sum_partial_fraction_identity(orc):
    """1/((A + b1)(A + b2)) = [1/(A + b1) - 1/(A + b2)] / (b2 - b1): the two-term rational sum equals two
    solves in sequence (one below, one above the cutoff, so both branches of the rule are exercised)."""
    dims = (4, 4, 4, 4)
    phi = inputs.make_phi(5, dims, 0.3)
    eta = inputs.make_source(5, 0, dims)
    b1, b2 = 0.7, 150.0
    out, infos = orc.rational_apply(phi, eta, 1.0, 0.2, 0.0, [1 / (b2 - b1), -1 / (b2 - b1)], [b1, b2], 1.0, 1e-13, 5000)
    y, _ = orc.cg_shift(phi, eta, 1.0, 0.2, b2, 1.0, 1e-13, 5000)
    z, _ = orc.cg_shift(phi, y, 1.0, 0.2, b1, 1.0, 1e-13, 5000)
    assert len(infos) == 2 and all(i.converged for i in infos)
    assert rel(out, z) < 1e-10


def test_rational_sum_is_the_inverse_fourth_root(orc):
    """Eq. 7.6 with the synthetic ladder against (M^dag M)^(-1/4) eta from the dense eigen-decomposition:
    the error is bounded by the scalar approximation error over the spectrum."""
    dims = (4, 4, 4, 4)
    phi = inputs.make_phi(6, dims, 0.3)
    eta = inputs.make_source(6, 0, dims)
    A = _dense_A(dims, phi, 1.0, 0.2)
    lam, U = np.linalg.eigh(A)
    a0, al, be = inputs.rational_ladder(20, 0.5 * lam[0], 2.0 * lam[-1])
    scal = a0 + (al[None, :] / (lam[:, None] + be[None, :])).sum(axis=1)
    eps = float(np.max(np.abs(scal * lam ** 0.25 - 1.0)))
    assert eps < 0.03
    out, infos = orc.rational_apply(phi, eta, 1.0, 0.2, a0, al, be, 1.0, 1e-12, 5000)
    exact = (U @ (lam ** -0.25 * (U.conj().T @ eta.reshape(-1)))).reshape(eta.shape)
    assert rel(out, exact) <= 1.05 * eps
    # and exactly (to solver accuracy) the same rational function of the dense matrix
    dense = (U @ (scal * (U.conj().T @ eta.reshape(-1)))).reshape(eta.shape)
    assert rel(out, dense) < 1e-10
