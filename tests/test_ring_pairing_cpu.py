"""Host logic of the ring-grid front end (no GPU): which rings share a Legendre recurrence (nusht_ring_pairing,
include/nusht.h).  Mirror rings theta_a + theta_b = pi pair up; the equator and rings of an asymmetric grid stay
single; pairs are ordered from the poles towards the equator."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def nusht():
    from paper_2406_14542_b200 import nusht as n
    return n


def test_symmetric_grid_pairs_every_ring(nusht):
    xg, _ = np.polynomial.legendre.leggauss(64)
    theta = np.arccos(xg[::-1])
    theta[32:] = np.pi - theta[:32][::-1]
    pairs = nusht.ring_pairing(theta)
    assert len(pairs) == 32
    for j, (a, b) in enumerate(pairs):
        assert (a, b) == (j, 63 - j)


def test_equator_and_poles(nusht):
    theta = np.pi * np.arange(9) / 8          # Clenshaw-Curtis: both poles, the equator ring alone
    pairs = nusht.ring_pairing(theta)
    assert pairs == [(0, 8), (1, 7), (2, 6), (3, 5), (4, -1)]


def test_unsorted_and_asymmetric_rings(nusht):
    theta = np.array([2.0, 0.3, np.pi - 0.3, 1.0, 2.5, 0.1])
    pairs = nusht.ring_pairing(theta)
    assert sorted(pairs) == sorted([(5, -1), (1, 2), (4, -1), (3, -1), (0, -1)])
    # every ring appears exactly once
    seen = sorted([a for a, _ in pairs] + [b for _, b in pairs if b >= 0])
    assert seen == list(range(6))
    # ordered by the distance from the nearer pole
    d = [min(theta[a], np.pi - theta[a]) for a, _ in pairs]
    assert d == sorted(d)


def test_two_ulp_tolerance_and_bad_input(nusht):
    t = 0.7
    assert nusht.ring_pairing([t, np.pi - t]) == [(0, 1)]
    assert nusht.ring_pairing([t, np.nextafter(np.pi - t, 4.0)]) == [(0, 1)]
    assert nusht.ring_pairing([t, np.pi - t + 1e-14]) != [(0, 1)]
    with pytest.raises(nusht.NushtError):
        nusht.ring_pairing([0.5, 3.5])
    assert nusht.ring_pairing([]) == []
