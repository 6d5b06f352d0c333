"""Pins of the oracle's locality probe (pin P9; Fig. 1)."""
import numpy as np

from paper_1005_3276_b200 import inputs  # noqa: F401  (path set-up by conftest)


def test_locality_profile_fig1_properties(orc):
    """Fig. 1 caption: 'The value of f at r=0 is zero ... Even r are consistently lower than odd r';
    text: 'a long tail', no exponential localisation.  16^4 as in the figure."""
    dims = (16, 16, 16, 16)
    f, psi = orc.locality_profile(dims, spin=0)
    assert len(f) == 33
    assert f[0] < 1e-13                      # sum_p Dslash(p) = 0: odd symbol on a p -> -p symmetric set
    assert np.all(f[1:] > 0)
    for r in range(4, 32, 2):                # two branches: even r below both odd neighbours
        assert f[r] < f[r - 1] and f[r] < f[r + 1], r
    assert np.all(np.diff(f[1:33:2]) < 0) and np.all(np.diff(f[2:33:2]) < 0)  # each branch decays ...
    assert f[31] / f[1] > 1e-3               # ... but slowly: a long tail, no exponential localisation
    assert f[31] / f[15] > 0.3
    # taxi distance bookkeeping: the furthest site is at r = 4 * 8
    assert f[32] > 0


def test_dslash_point_source_is_spin_off_diagonal(orc):
    """gamma5 Dslash gamma5 = -Dslash (Eq. 3.4): a source in a P- component only reaches P+ components."""
    dims = (8, 4, 4, 4)
    f, psi = orc.locality_profile(dims, spin=1)
    assert np.abs(psi[:2]).max() < 1e-13 and np.abs(psi[2:]).max() > 1e-3
