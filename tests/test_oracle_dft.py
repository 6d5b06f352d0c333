"""Pins for the oracle's DFTs.  CPU only."""
import numpy as np
import pytest


def _rand(shape, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 2, 6), (6, 12, 4, 8)])
def test_naive_matches_numpy_fftn(orc, dims):
    a = _rand((2,) + dims, 1)
    f = orc.dft4d(a, +1, False, "naive")
    ref = np.fft.fftn(a, axes=(1, 2, 3, 4))           # library routine: exp(-2 pi i n x/L), unnormalised
    assert np.abs(f - ref).max() <= 1e-12 * np.abs(ref).max()
    b = orc.dft4d(a, -1, False, "naive")
    refi = np.fft.ifftn(a, axes=(1, 2, 3, 4))         # exp(+...), times 1/V
    assert np.abs(b - refi).max() <= 1e-12 * np.abs(refi).max()


@pytest.mark.parametrize("dims", [(16, 4, 8, 2), (32, 16, 2, 4)])
def test_radix2_matches_numpy_and_naive(orc, dims):
    a = _rand((1,) + dims, 2)
    f2 = orc.dft4d(a, +1, False, "radix2")
    f0 = orc.dft4d(a, +1, False, "naive")
    ref = np.fft.fftn(a, axes=(1, 2, 3, 4))
    scale = np.abs(ref).max()
    assert np.abs(f2 - ref).max() <= 1e-13 * scale
    assert np.abs(f2 - f0).max() <= 1e-12 * scale
    for apbc in (False, True):
        g2 = orc.dft4d(a, -1, apbc, "radix2")
        g0 = orc.dft4d(a, -1, apbc, "naive")
        assert np.abs(g2 - g0).max() <= 1e-13 * np.abs(g0).max()


def test_radix2_rejects_non_power_of_two(orc):
    with pytest.raises(ValueError):
        orc.dft4d(np.zeros((6, 4, 4, 4), complex), +1, False, "radix2")


@pytest.mark.parametrize("method", ["naive", "radix2"])
@pytest.mark.parametrize("apbc", [False, True])
def test_round_trip_and_parseval(orc, method, apbc):
    dims = (8, 4, 16, 2)
    a = _rand((4,) + dims, 3)
    f = orc.dft4d(a, +1, apbc, method)
    back = orc.dft4d(f, -1, apbc, method)
    assert np.abs(back - a).max() <= 1e-13
    V = np.prod(dims)
    assert abs((np.abs(f) ** 2).sum() - V * (np.abs(a) ** 2).sum()) <= 1e-12 * V * (np.abs(a) ** 2).sum()


def test_delta_gives_plane_wave(orc):
    dims = (4, 6, 8, 2)
    x = (1, 5, 3, 1)
    a = np.zeros(dims, complex)
    a[x] = 1.0
    f = orc.dft4d(a, +1, False, "naive")
    n = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    phase = sum(n[mu] * x[mu] / dims[mu] for mu in range(4))
    assert np.abs(f - np.exp(-2j * np.pi * phase)).max() <= 1e-13
    # antiperiodic in time: p0 = 2 pi (n0 + 1/2)/T
    f = orc.dft4d(a, +1, True, "naive")
    phase = (n[0] + 0.5) * x[0] / dims[0] + sum(n[mu] * x[mu] / dims[mu] for mu in (1, 2, 3))
    assert np.abs(f - np.exp(-2j * np.pi * phase)).max() <= 1e-13


def test_antiperiodic_plane_wave_is_single_bin(orc):
    # psi(x) = exp(i p x) with p0 = pi (2 n0 + 1)/T is antiperiodic in time
    # and must land in exactly one bin of the twisted transform.
    dims = (8, 4, 4, 16)
    nvec = (5, 3, 0, 9)
    x = np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")
    phase = (nvec[0] + 0.5) * x[0] / dims[0] + sum(nvec[mu] * x[mu] / dims[mu] for mu in (1, 2, 3))
    psi = np.exp(2j * np.pi * phase)
    for method in ("naive", "radix2"):
        f = orc.dft4d(psi, +1, True, method)
        want = np.zeros(dims, complex)
        want[nvec] = np.prod(dims)
        assert np.abs(f - want).max() <= 1e-10
