"""ctypes binding of oracle/wz_oracle.cpp (the CPU oracle; test infrastructure only).

The arithmetic lives in wz_oracle.cpp, each function there cites the passage of
PAPER.md it follows.  This file only builds the shared object with g++ and
marshals numpy arrays.  All arrays are complex128 in the external layout
spinor = [spin][x0][x1][x2][x3], phi = [x0][x1][x2][x3].
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wz_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_wz.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (OpenMP) if the .so is missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC]
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


class _Info(ctypes.Structure):
    _fields_ = [("iterations", ctypes.c_int), ("reliable_updates", ctypes.c_int),
                ("converged", ctypes.c_int), ("rel_residual_recursive", ctypes.c_double),
                ("rel_residual_true", ctypes.c_double)]


@dataclass
class CGInfo:
    iterations: int
    reliable_updates: int
    converged: bool
    rel_residual_recursive: float
    rel_residual_true: float
    history: np.ndarray


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_set_threads.restype = ctypes.c_int
    return _lib


def set_threads(n: int = 0) -> int:
    """Set (n > 0) or query (n = 0) the OpenMP thread count the oracle uses."""
    return int(lib().orc_set_threads(int(n)))


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def _c2(z):
    z = complex(z)
    return (ctypes.c_double * 2)(z.real, z.imag)


def _method(dims, method):
    if method == "auto":
        pow2 = all(d & (d - 1) == 0 for d in dims)
        return 1 if (pow2 and max(dims) >= 16) else 0
    return {"naive": 0, "radix2": 1}[method]


def gamma(mu: int) -> np.ndarray:
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().orc_gamma(int(mu), _dp(out))
    return out


def dft4d(a: np.ndarray, direction: int, apbc: bool, method: str = "auto") -> np.ndarray:
    """4D DFT over the last four axes of `a` (any leading component axes)."""
    a = np.array(a, dtype=np.complex128, order="C", copy=True)
    dims = a.shape[-4:]
    ncomp = int(np.prod(a.shape[:-4], dtype=np.int64)) if a.ndim > 4 else 1
    rc = lib().orc_dft4d(_method(dims, method), int(direction), int(bool(apbc)), _dims(dims), _dp(a), ncomp)
    if rc:
        raise ValueError("radix-2 oracle FFT needs power-of-two extents")
    return a


def overlap_D_symbol(p, rho: float = 1.0):
    """(D, D1, D2) of Eq. (2.9) on the plane wave exp(+ipx), by 4x4 matrix algebra."""
    p = np.ascontiguousarray(p, dtype=np.float64)
    D, D1, D2 = (np.zeros((4, 4), dtype=np.complex128) for _ in range(3))
    rc = lib().orc_overlap_D_symbol(_dp(p), ctypes.c_double(rho), _dp(D), _dp(D1), _dp(D2))
    if rc:
        raise ArithmeticError("A^dag A is not proportional to the unit matrix")
    return D, D1, D2


def dslash_symbol(p, rho: float = 1.0) -> np.ndarray:
    """Dslash(p) = (1 - D2/2rho)^-1 D1 as the 4x4 matrix the oracle operator applies."""
    p = np.ascontiguousarray(p, dtype=np.float64)
    out = np.zeros((4, 4), dtype=np.complex128)
    lib().orc_dslash_symbol_p(_dp(p), ctypes.c_double(rho), _dp(out))
    return out


def d2_extremes(dims, rho: float = 1.0, apbc: bool = True):
    lo, hi = ctypes.c_double(), ctypes.c_double()
    lib().orc_dslash_d2_extremes(_dims(dims), ctypes.c_double(rho), int(apbc), ctypes.byref(lo), ctypes.byref(hi))
    return lo.value, hi.value


def apply_M(phi, psi, m, g, rho=1.0, dagger=False, method="auto") -> np.ndarray:
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    dims = phi.shape
    assert psi.shape == (4,) + tuple(dims)
    out = np.empty_like(psi)
    rc = lib().orc_apply_M(_method(dims, method), _dims(dims), _dp(phi), _c2(m), _c2(g),
                           ctypes.c_double(rho), int(bool(dagger)), _dp(psi), _dp(out))
    if rc:
        raise ValueError("oracle apply_M failed")
    return out


def apply_MdagM(phi, psi, m, g, rho=1.0, method="auto") -> np.ndarray:
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    dims = phi.shape
    assert psi.shape == (4,) + tuple(dims)
    out = np.empty_like(psi)
    rc = lib().orc_apply_MdagM(_method(dims, method), _dims(dims), _dp(phi), _c2(m), _c2(g),
                               ctypes.c_double(rho), _dp(psi), _dp(out))
    if rc:
        raise ValueError("oracle apply_MdagM failed")
    return out


def cg(phi, b, m, g, rho=1.0, tol=1e-10, max_iter=100000, method="auto"):
    """Textbook CG on M^dag M x = b in complex128.  Returns (x, CGInfo)."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    x = np.zeros_like(b)
    hist = np.zeros(max_iter + 1, dtype=np.float64)
    info = _Info()
    rc = lib().orc_cg(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(x), _c2(m), _c2(g),
                      ctypes.c_double(rho), ctypes.c_double(tol), int(max_iter), ctypes.byref(info), _dp(hist))
    if rc:
        raise ValueError("oracle cg failed")
    return x, CGInfo(info.iterations, info.reliable_updates, bool(info.converged),
                     info.rel_residual_recursive, info.rel_residual_true, hist[: info.iterations + 1].copy())


def cg_c64ru(phi, b, m, g, rho=1.0, tol=1e-6, max_iter=100000, delta=0.1, method="auto", sigma=0.0):
    """complex64-vector CG with reliable updates (oracle variant O4'); sigma: on the shifted
    system (M^dag M + sigma) x = b of Eq. (7.13).  Returns (X, CGInfo)."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    X = np.zeros_like(b)
    hist = np.zeros(max_iter + 1, dtype=np.float64)
    info = _Info()
    rc = lib().orc_cg_c64ru_shift(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(X), _c2(m), _c2(g),
                                  ctypes.c_double(rho), ctypes.c_double(sigma), ctypes.c_double(tol), int(max_iter),
                                  ctypes.c_double(delta), ctypes.byref(info), _dp(hist))
    if rc:
        raise ValueError("oracle cg_c64ru failed")
    return X, CGInfo(info.iterations, info.reliable_updates, bool(info.converged),
                     info.rel_residual_recursive, info.rel_residual_true, hist[: info.iterations + 1].copy())


def apply_M0inv(dims, psi, m, rho=1.0, dagger=False, method="auto") -> np.ndarray:
    """M0^-1 psi (Eq. 7.11) or its conjugate transpose; M0 = free (g = 0) fermion matrix."""
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    dims = tuple(int(d) for d in dims)
    assert psi.shape == (4,) + dims
    out = np.empty_like(psi)
    rc = lib().orc_apply_M0inv(_method(dims, method), _dims(dims), _c2(m), ctypes.c_double(rho),
                               int(bool(dagger)), _dp(psi), _dp(out))
    if rc:
        raise ValueError("oracle apply_M0inv failed")
    return out


def apply_Mtilde(phi, psi, m, g, rho=1.0, dagger=False, method="auto") -> np.ndarray:
    """Mtilde = M M0^-1 (Eq. 7.10) or its conjugate transpose."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    dims = phi.shape
    out = np.empty_like(psi)
    rc = lib().orc_apply_Mtilde(_method(dims, method), _dims(dims), _dp(phi), _c2(m), _c2(g),
                                ctypes.c_double(rho), int(bool(dagger)), _dp(psi), _dp(out))
    if rc:
        raise ValueError("oracle apply_Mtilde failed")
    return out


def cg_pc(phi, b, m, g, rho=1.0, tol=1e-10, max_iter=100000, method="auto"):
    """Preconditioned CG (Eq. 7.8-7.11) in complex128.  Returns (x, CGInfo)."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    x = np.zeros_like(b)
    hist = np.zeros(max_iter + 1, dtype=np.float64)
    info = _Info()
    rc = lib().orc_cg_pc(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(x), _c2(m), _c2(g),
                         ctypes.c_double(rho), ctypes.c_double(tol), int(max_iter), ctypes.byref(info), _dp(hist))
    if rc:
        raise ValueError("oracle cg_pc failed")
    return x, CGInfo(info.iterations, info.reliable_updates, bool(info.converged),
                     info.rel_residual_recursive, info.rel_residual_true, hist[: info.iterations + 1].copy())


def apply_Dslash(dims, psi, rho=1.0, method="auto") -> np.ndarray:
    """Dslash psi = (1 - D2/2)^-1 D1 psi: the fermion matrix of Eq. (2.19) at m = 0, g = 0."""
    dims = tuple(int(d) for d in dims)
    return apply_M(np.zeros(dims, dtype=np.complex128), psi, 0.0, 0.0, rho, False, method)


def locality_profile(dims, spin=0, rho=1.0, method="auto"):
    """PAPER.md:262-282, Eq. (3.9)-(3.11): psi = Dslash eta for a unit point source eta at the
    origin (spin component `spin`), f(r) = max{ ||psi(x)|| : ||x||_1 = r } with the taxi-driver
    distance of Eq. (3.10) and ||.|| the norm over the spinor index.  Returns (f, psi)."""
    dims = tuple(int(d) for d in dims)
    eta = np.zeros((4,) + dims, dtype=np.complex128)
    eta[(spin, 0, 0, 0, 0)] = 1.0
    psi = apply_Dslash(dims, eta, rho, method)
    nrm = np.sqrt((np.abs(psi) ** 2).sum(axis=0))
    dist = np.zeros(dims, dtype=np.int64)
    for mu, L in enumerate(dims):
        x = np.arange(L)
        d = np.minimum(x, L - x)                      # |x_mu| or |L_mu - x_mu|, the shorter one
        shape = [1, 1, 1, 1]
        shape[mu] = L
        dist = dist + d.reshape(shape)
    rmax = int(sum(L // 2 for L in dims))
    f = np.zeros(rmax + 1)
    for r in range(rmax + 1):
        sel = nrm[dist == r]
        f[r] = sel.max() if sel.size else 0.0
    return f, psi


def cg_shift(phi, b, m, g, sigma, rho=1.0, tol=1e-10, max_iter=100000, method="auto"):
    """Textbook CG on (M^dag M + sigma) x = b (Eq. 7.13) in complex128.  Returns (x, CGInfo)."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    x = np.zeros_like(b)
    hist = np.zeros(max_iter + 1, dtype=np.float64)
    info = _Info()
    rc = lib().orc_cg_shift(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(x), _c2(m), _c2(g),
                            ctypes.c_double(rho), ctypes.c_double(sigma), ctypes.c_double(tol), int(max_iter),
                            ctypes.byref(info), _dp(hist))
    if rc:
        raise ValueError("oracle cg_shift failed")
    return x, CGInfo(info.iterations, info.reliable_updates, bool(info.converged),
                     info.rel_residual_recursive, info.rel_residual_true, hist[: info.iterations + 1].copy())


def cg_shift_pc(phi, b, m, g, sigma, rho=1.0, tol=1e-10, max_iter=100000, method="auto"):
    """Textbook CG on the preconditioned shifted system of Eq. (7.14),
    (Mtilde^dag Mtilde + sigma (M0^-1)^dag M0^-1) xtilde = (M0^-1)^dag b, x = M0^-1 xtilde.
    Returns (x, CGInfo); rel_residual_true refers to (M^dag M + sigma) x = b."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    x = np.zeros_like(b)
    hist = np.zeros(max_iter + 1, dtype=np.float64)
    info = _Info()
    rc = lib().orc_cg_shift_pc(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(x), _c2(m), _c2(g),
                               ctypes.c_double(rho), ctypes.c_double(sigma), ctypes.c_double(tol), int(max_iter),
                               ctypes.byref(info), _dp(hist))
    if rc:
        raise ValueError("oracle cg_shift_pc failed")
    return x, CGInfo(info.iterations, info.reliable_updates, bool(info.converged),
                     info.rel_residual_recursive, info.rel_residual_true, hist[: info.iterations + 1].copy())


def rational_apply(phi, eta, m, g, alpha0, alphas, betas, rho=1.0, tol=1e-10, max_iter=100000,
                   pc_cutoff=100.0, method="auto"):
    """PAPER.md:877-892 Eq. (7.6)-(7.7) with the rule of PAPER.md:948: out = alpha_0 eta +
    sum_i alpha_i X_i, (M^dag M + beta_i) X_i = eta solved one shift at a time by CG --
    preconditioned (Eq. 7.14) for beta_i <= pc_cutoff, plain (Eq. 7.13) above it.
    Returns (out, [CGInfo per shift])."""
    eta = np.ascontiguousarray(eta, dtype=np.complex128)
    out = alpha0 * eta
    infos = []
    for a_i, b_i in zip(alphas, betas):
        if b_i <= pc_cutoff:
            X, info = cg_shift_pc(phi, eta, m, g, float(b_i), rho, tol, max_iter, method)
        else:
            X, info = cg_shift(phi, eta, m, g, float(b_i), rho, tol, max_iter, method)
        out = out + a_i * X
        infos.append(info)
    return out, infos


def cg_multishift(phi, b, m, g, sigmas, rho=1.0, tol=1e-10, max_iter=100000, method="auto"):
    """Multi-shift CG (oracle O8): all (M^dag M + sigma_i) X_i = b from one Krylov space, complex128.
    Returns (X[nshift, 4, T, L1, L2, L3], [CGInfo per shift], matvecs)."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    sig = np.ascontiguousarray(sigmas, dtype=np.float64)
    d = int(sig.size)
    dims = phi.shape
    X = np.zeros((d,) + b.shape, dtype=np.complex128)
    infos = (_Info * max(d, 1))()
    mv = ctypes.c_int(0)
    rc = lib().orc_cg_multishift(_method(dims, method), _dims(dims), _dp(phi), _dp(b), d, _dp(sig), _dp(X),
                                 _c2(m), _c2(g), ctypes.c_double(rho), ctypes.c_double(tol), int(max_iter),
                                 infos, ctypes.byref(mv))
    if rc:
        raise ValueError("oracle cg_multishift failed")
    out = [CGInfo(i.iterations, i.reliable_updates, bool(i.converged), i.rel_residual_recursive,
                  i.rel_residual_true, np.zeros(0)) for i in infos[:d]]
    return X, out, int(mv.value)


def cg_dc(phi, b, m, g, rho=1.0, tol=1e-10, inner_tol=1e-3, max_iter=100000, method="auto"):
    """Defect correction (oracle O9): complex128 outer loop, complex64-rounded inner CG restarted at every
    outer step.  Returns (X, CGInfo) with iterations = inner iterations in total and reliable_updates =
    the number of outer corrections."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    X = np.zeros_like(b)
    info = _Info()
    rc = lib().orc_cg_dc(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(X), _c2(m), _c2(g),
                         ctypes.c_double(rho), ctypes.c_double(tol), ctypes.c_double(inner_tol), int(max_iter),
                         ctypes.byref(info))
    if rc:
        raise ValueError("oracle cg_dc failed")
    return X, CGInfo(info.iterations, info.reliable_updates, bool(info.converged), info.rel_residual_recursive,
                     info.rel_residual_true, np.zeros(0))


def round_f16(x):
    """The oracle's IEEE binary16 rounding model (round to nearest even, saturating), element-wise on float64."""
    L = lib()
    L.orc_round_f16.restype = ctypes.c_double
    L.orc_round_f16.argtypes = [ctypes.c_double]
    a = np.asarray(x, dtype=np.float64)
    return np.array([L.orc_round_f16(float(v)) for v in a.ravel()]).reshape(a.shape)


def cg_dc_f16(phi, b, m, g, rho=1.0, tol=1e-6, inner_tol=1e-1, max_iter=100000, method="auto"):
    """Defect correction with binary16 STORAGE of the inner solver's r, p, chi (oracle O10).  Returns (X, CGInfo)
    with iterations = inner iterations in total and reliable_updates = outer corrections."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    X = np.zeros_like(b)
    info = _Info()
    rc = lib().orc_cg_dc_f16(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(X), _c2(m), _c2(g),
                             ctypes.c_double(rho), ctypes.c_double(tol), ctypes.c_double(inner_tol), int(max_iter),
                             ctypes.byref(info))
    if rc:
        raise ValueError("oracle cg_dc_f16 failed")
    return X, CGInfo(info.iterations, info.reliable_updates, bool(info.converged), info.rel_residual_recursive,
                     info.rel_residual_true, np.zeros(0))


def cg_f16ru(phi, b, m, g, rho=1.0, tol=1e-6, max_iter=100000, delta=0.1, method="auto"):
    """binary16 storage of r, p, chi with complex128 reliable updates and rescaling (oracle O11).
    Returns (X, CGInfo)."""
    phi = np.ascontiguousarray(phi, dtype=np.complex128)
    b = np.ascontiguousarray(b, dtype=np.complex128)
    dims = phi.shape
    X = np.zeros_like(b)
    info = _Info()
    rc = lib().orc_cg_f16ru(_method(dims, method), _dims(dims), _dp(phi), _dp(b), _dp(X), _c2(m), _c2(g),
                            ctypes.c_double(rho), ctypes.c_double(tol), int(max_iter), ctypes.c_double(delta),
                            ctypes.byref(info))
    if rc:
        raise ValueError("oracle cg_f16ru failed")
    return X, CGInfo(info.iterations, info.reliable_updates, bool(info.converged), info.rel_residual_recursive,
                     info.rel_residual_true, np.zeros(0))
