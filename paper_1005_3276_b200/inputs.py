"""Seeded synthetic inputs shared by the tests, the oracle harness and bench.py.

This module holds NONE of the method's arithmetic: it only turns a seed into the
bytes of phi(x) and of the sources b_j.  Both the CUDA path and the CPU oracle are
fed the same arrays from here.

Recipe ("random Gaussian b"; BASELINE.json configs for the widths):
  * SplitMix64 seeded with  seed * 2**32 + stream_id   (stream 0 = phi, 1+j = source j);
  * consecutive pairs of 64-bit outputs (a, b) give 53-bit uniforms
        u1 = ((a >> 11) + 1) / 2**53  in (0, 1],   u2 = (b >> 11) / 2**53  in [0, 1);
  * Box-Muller: z0 = sqrt(-2 ln u1) cos(2 pi u2), z1 = sqrt(-2 ln u1) sin(2 pi u2);
  * (Re, Im) of consecutive elements in layout order = (z0, z1) * sigma.
Layout: phi = [x0][x1][x2][x3]; spinor = [spin][x0][x1][x2][x3], x3 fastest.
complex64 inputs are generated in double and rounded to float once.
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, n: int) -> np.ndarray:
    """First n outputs of SplitMix64 started at state `seed` (uint64 wraparound)."""
    with np.errstate(over="ignore"):
        idx = np.arange(1, n + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + idx * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def gaussian_complex(seed: int, stream_id: int, n: int, sigma: float = 1.0) -> np.ndarray:
    """n complex128 numbers with Re, Im ~ N(0, sigma^2), i.i.d."""
    raw = splitmix64((int(seed) << 32) + int(stream_id), 2 * n)
    a = raw[0::2] >> np.uint64(11)
    b = raw[1::2] >> np.uint64(11)
    u1 = (a.astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)
    u2 = b.astype(np.float64) * (1.0 / 9007199254740992.0)
    rad = np.sqrt(-2.0 * np.log(u1))
    ang = 2.0 * np.pi * u2
    out = np.empty(n, dtype=np.complex128)
    out.real = rad * np.cos(ang) * sigma
    out.imag = rad * np.sin(ang) * sigma
    return out


def make_phi(seed: int, dims, sigma: float, dtype=np.complex128) -> np.ndarray:
    """phi(x), shape (T, L1, L2, L3)."""
    T, L1, L2, L3 = dims
    v = gaussian_complex(seed, 0, T * L1 * L2 * L3, sigma).reshape(T, L1, L2, L3)
    return np.ascontiguousarray(v.astype(dtype))


def make_source(seed: int, j: int, dims, dtype=np.complex128) -> np.ndarray:
    """Gaussian source b_j, shape (4, T, L1, L2, L3), unit variance per real component."""
    T, L1, L2, L3 = dims
    v = gaussian_complex(seed, 1 + j, 4 * T * L1 * L2 * L3, 1.0).reshape(4, T, L1, L2, L3)
    return np.ascontiguousarray(v.astype(dtype))


def make_sources(seed: int, nsrc: int, dims, dtype=np.complex128) -> np.ndarray:
    """Batch of sources, shape (nsrc, 4, T, L1, L2, L3)."""
    return np.stack([make_source(seed, j, dims, dtype) for j in range(nsrc)])


# BASELINE.json configs.  dims = (T, L1, L2, L3).
CONFIGS = {
    1: dict(dims=(4, 4, 4, 4), dtype="c128", sigma=0.3, m=0.1, g=0.5, rho=1.0, nsrc=1, tol=1e-10, seed=1),
    2: dict(dims=(8, 8, 8, 8), dtype="c128", sigma=0.3, m=0.05, g=1.0, rho=1.0, nsrc=1, tol=1e-10, seed=2),
    3: dict(dims=(16, 16, 16, 16), dtype="c64", sigma=0.5, m=0.02, g=1.0, rho=1.0, nsrc=4, tol=1e-6, seed=3),
    4: dict(dims=(32, 32, 32, 32), dtype="c64", sigma=0.5, m=0.01, g=1.5, rho=1.0, nsrc=12, tol=1e-6, seed=4),
    "5a": dict(dims=(48, 24, 24, 24), dtype="c64", sigma=0.5, m=0.005, g=1.5, rho=1.0, nsrc=1, tol=1e-6, seed=5),
    "5b": dict(dims=(64, 64, 64, 64), dtype="c64", sigma=0.5, m=0.005, g=1.5, rho=1.0, nsrc=1, tol=1e-6, seed=5),
}


def rational_ladder(d: int = 20, lo: float = 1e-2, hi: float = 1e3, gamma: float = 0.25, pad: float = 4.0):
    """Synthetic stand-in for the coefficients of Eq. (7.6), which the paper does not print
    ("chosen to minimize errors over the range of eigenvalues"; d = 20 at
    PAPER.md:931).  Returns (alpha_0, alpha[d], beta[d]) with
        x^-gamma ~ alpha_0 + sum_i alpha_i / (x + beta_i)   for lo <= x <= hi,
    from the trapezoid rule in u = ln t on  x^-gamma = sin(pi gamma)/pi * int_0^inf t^-gamma/(x+t) dt:
    a geometric ladder of positive shifts beta_i from lo e^-pad to hi e^+pad (all alpha_i > 0),
    alpha_0 = the tail beyond the last node.  Not Remez-optimal (about 1 % at d = 20, pad = 4 over
    five decades); what matters here is the form of the input: d shifts spread over the spectrum.
    These are INPUTS of the method, like phi and b; both sides consume the same arrays."""
    u = np.linspace(np.log(lo) - pad, np.log(hi) + pad, d)
    h = u[1] - u[0]
    c = np.sin(np.pi * gamma) / np.pi
    beta = np.exp(u)
    alpha = c * h * np.exp((1.0 - gamma) * u)
    alpha0 = c * np.exp(-gamma * (u[-1] + 0.5 * h)) / gamma
    return float(alpha0), alpha, beta
