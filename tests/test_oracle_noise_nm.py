"""Pins for the oracle's Philox / Box-Muller / normal-mode matrix."""
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answers():
    n = 0
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == v[6:10]
        n += 1
    assert n == 3


def test_box_muller_matches_definition_and_moments():
    # definition (N4) re-evaluated from the raw Philox words with numpy
    x = oracle.philox4x32_10([7, 3 * 8 + 5, 11, 1], [42, 0])
    u = [(w + 0.5) / 2.0 ** 32 for w in x]
    want = [np.sqrt(-2 * np.log(u[0])) * np.cos(2 * np.pi * u[1]), np.sqrt(-2 * np.log(u[0])) * np.sin(2 * np.pi * u[1]),
            np.sqrt(-2 * np.log(u[2])) * np.cos(2 * np.pi * u[3])]
    got = oracle.normal3(42, 7, 3 * 8 + 5, 11, 1)
    assert np.allclose(got, want, rtol=0, atol=1e-14)
    # sample moments of a standard normal; independence between components
    xs = np.array([oracle.normal3(1234, a, m, 5, 0) for a in range(200) for m in range(100)])
    assert abs(xs.mean()) < 0.02 and abs(xs.var() - 1.0) < 0.02
    assert abs(np.mean(xs ** 4) - 3.0) < 0.1
    c = np.corrcoef(xs.T)
    assert np.abs(c - np.eye(3)).max() < 0.03
    # different tag / step / seed -> different stream
    assert not np.allclose(oracle.normal3(1, 0, 0, 0, 0), oracle.normal3(1, 0, 0, 0, 1))
    assert not np.allclose(oracle.normal3(1, 0, 0, 0, 0), oracle.normal3(1, 0, 0, 1, 0))
    assert not np.allclose(oracle.normal3(1, 0, 0, 0, 0), oracle.normal3(1 << 32, 0, 0, 0, 0))


@pytest.mark.parametrize("P", [1, 2, 3, 4, 5, 8, 32, 128])
def test_nm_matrix_orthogonal_and_diagonalises_ring(P):
    C = oracle.nm_matrix(P)
    assert np.abs(C @ C.T - np.eye(P)).max() < 1e-13
    assert np.abs(C.T @ C - np.eye(P)).max() < 1e-13
    # ring spring matrix K: sum_k (q_k - q_{k+1})^2 = q^T K q
    K = np.zeros((P, P))
    for k in range(P):
        kn = (k + 1) % P
        K[k, k] += 1; K[kn, kn] += 1; K[k, kn] -= 1; K[kn, k] -= 1
    D = C.T @ K @ C
    lam = 4 * np.sin(np.arange(P) * np.pi / P) ** 2
    assert np.abs(D - np.diag(lam)).max() < 1e-12
    assert np.allclose(C[:, 0], 1 / np.sqrt(P))  # centroid mode
