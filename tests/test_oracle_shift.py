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
