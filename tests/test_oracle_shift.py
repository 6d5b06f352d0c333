"""Pins of the oracle's shifted solve (SURVEY 8(f) NEXT-2 first step; Eq. 7.13)."""
import numpy as np

from paper_1005_3276_b200 import inputs


def rel(a, ref):
    return float(np.linalg.norm((a - ref).ravel()) / np.linalg.norm(ref.ravel()))


def test_shifted_solution_equals_dense_solve(orc):
    from oracle import dense_route

    dims = (4, 4, 4, 4)
    cfg = inputs.CONFIGS[1]
    phi = inputs.make_phi(1, dims, cfg["sigma"])
    b = inputs.make_source(1, 0, dims)
    M = dense_route.fermion_matrix_dense(dims, phi, cfg["m"], cfg["g"], 1.0)
    A = M.conj().T @ M
    for sigma in (0.0, 0.3, 25.0):
        x, info = orc.cg_shift(phi, b, cfg["m"], cfg["g"], sigma, 1.0, 1e-12, 5000)
        xd = np.linalg.solve(A + sigma * np.eye(A.shape[0]), b.reshape(-1)).reshape(b.shape)
        assert info.converged and rel(x, xd) < 1e-9
        assert info.rel_residual_true < 1e-11


def test_shift_zero_is_plain_cg_and_large_shift_converges_fast(orc):
    """sigma = 0 reproduces orc_cg (up to the summation order of its OpenMP loops); 'for very large beta_i the problem
    without preconditioning converges rapidly'."""
    dims = (8, 4, 4, 4)
    phi = inputs.make_phi(2, dims, 0.3)
    b = inputs.make_source(2, 0, dims)
    x0, i0 = orc.cg(phi, b, 0.05, 1.0, 1.0, 1e-10, 5000)
    x1, i1 = orc.cg_shift(phi, b, 0.05, 1.0, 0.0, 1.0, 1e-10, 5000)
    assert abs(i0.iterations - i1.iterations) <= max(2, i0.iterations // 100) and rel(x1, x0) < 1e-6
    its = [orc.cg_shift(phi, b, 0.05, 1.0, s, 1.0, 1e-10, 5000)[1].iterations for s in (0.0, 1.0, 100.0, 1e4)]
    assert its[0] > its[1] > its[2] > its[3] and its[3] < 40


def test_c64ru_shifted_solution_equals_dense_solve(orc):
    """Reading G9's complex64 loop on the shifted system (what WZ_C64 plans are compared with)."""
    from oracle import dense_route

    dims = (4, 4, 4, 4)
    cfg = inputs.CONFIGS[1]
    phi = inputs.make_phi(1, dims, cfg["sigma"])
    b = inputs.make_source(1, 0, dims)
    M = dense_route.fermion_matrix_dense(dims, phi, cfg["m"], cfg["g"], 1.0)
    A = M.conj().T @ M
    for sigma in (0.0, 0.3, 25.0):
        X, info = orc.cg_c64ru(phi, b, cfg["m"], cfg["g"], 1.0, 1e-6, 5000, sigma=sigma)
        xd = np.linalg.solve(A + sigma * np.eye(A.shape[0]), b.reshape(-1)).reshape(b.shape)
        assert info.converged and info.reliable_updates >= 1 and info.rel_residual_true <= 1e-6
        res = rel((A @ X.reshape(-1) + sigma * X.reshape(-1)).reshape(b.shape), b)
        assert abs(res - info.rel_residual_true) < 1e-9 and rel(X, xd) < 1e-4


# ---- multi-shift CG (oracle O8; SURVEY 8(f) NEXT-2 "all shifts from one Krylov space") ----

def test_multishift_equals_dense_solves(orc):
    from oracle import dense_route

    dims = (4, 4, 4, 4)
    cfg = inputs.CONFIGS[1]
    phi = inputs.make_phi(1, dims, cfg["sigma"])
    b = inputs.make_source(1, 0, dims)
    M = dense_route.fermion_matrix_dense(dims, phi, cfg["m"], cfg["g"], 1.0)
    A = M.conj().T @ M
    sigmas = [0.0, 0.3, 25.0, 1e-3, 400.0]
    X, infos, mv = orc.cg_multishift(phi, b, cfg["m"], cfg["g"], sigmas, 1.0, 1e-12, 5000)
    for i, sigma in enumerate(sigmas):
        xd = np.linalg.solve(A + sigma * np.eye(A.shape[0]), b.reshape(-1)).reshape(b.shape)
        assert infos[i].converged and rel(X[i], xd) < 1e-9, (sigma, rel(X[i], xd))
        assert infos[i].rel_residual_true < 1e-11
        # the recursive |zeta| ||r|| is the residual of the shifted system (collinearity), not just a bound
        assert abs(infos[i].rel_residual_true - infos[i].rel_residual_recursive) <= 0.05 * infos[i].rel_residual_true + 2e-13
    assert mv == max(i.iterations for i in infos)


def test_multishift_follows_the_single_shift_iterations(orc):
    """In exact arithmetic shift i's iterate after n steps IS the n-th CG iterate of (A + sigma_i) x = b, so
    every shift freezes at the iteration count of its own single-shift solve (orc_cg_shift, pinned above
    against dense solves), and the solutions agree to kappa * tol; the smallest shift sets the matvec count."""
    dims = (8, 4, 4, 4)
    phi = inputs.make_phi(2, dims, 0.3)
    b = inputs.make_source(2, 0, dims)
    m, g, tol = 0.05, 1.0, 1e-10
    sigmas = [0.0, 0.01, 1.0, 100.0, 1e4]
    X, infos, mv = orc.cg_multishift(phi, b, m, g, sigmas, 1.0, tol, 5000)
    single = [orc.cg_shift(phi, b, m, g, s, 1.0, tol, 5000) for s in sigmas]
    for i, (xs, info_s) in enumerate(single):
        assert infos[i].converged
        assert abs(infos[i].iterations - info_s.iterations) <= max(2, info_s.iterations // 100), \
            (sigmas[i], infos[i].iterations, info_s.iterations)
        assert rel(X[i], xs) < 1e-6
        assert infos[i].rel_residual_true <= tol * 1.05
    assert mv == infos[0].iterations and infos[0].iterations > infos[2].iterations > infos[4].iterations
    # sigma = 0 alone is plain CG: zeta stays 1
    X0, i0, mv0 = orc.cg_multishift(phi, b, m, g, [0.0], 1.0, tol, 5000)
    x_cg, i_cg = orc.cg(phi, b, m, g, 1.0, tol, 5000)
    assert i0[0].iterations == i_cg.iterations and rel(X0[0], x_cg) < 1e-12


def test_multishift_rational_sum_equals_sequential_solves(orc):
    """Eq. (7.6): alpha_0 eta + sum alpha_i X_i from one multi-shift run against the oracle's
    one-solve-per-shift rational_apply (plain branch)."""
    dims = (4, 4, 4, 4)
    phi = inputs.make_phi(9, dims, 0.5)
    eta = inputs.make_source(9, 0, dims)
    a0, al, be = inputs.rational_ladder(8, 1e-2, 1e2)
    ref, _ = orc.rational_apply(phi, eta, 1.0, 0.1, a0, al, be, 1.0, 1e-12, 2000, pc_cutoff=-1.0)
    X, infos, _ = orc.cg_multishift(phi, eta, 1.0, 0.1, be, 1.0, 1e-12, 2000)
    out = a0 * eta + sum(a * x for a, x in zip(al, X))
    assert all(i.converged for i in infos) and rel(out, ref) < 1e-10
