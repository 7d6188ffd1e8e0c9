"""Seeded synthetic inputs (pimd_inputs): shapes, bond lengths, density."""
import numpy as np
import pytest

import pimd_inputs as pi


def test_weight_counts():
    # 52 033 for (3,32,64,2); 288 769 for (3,64,128,3)
    assert pi.n_weights(3, 32, 64, 2) == 52033
    assert pi.n_weights(3, 64, 128, 3) == 288769
    w = pi.pack_weights(0, 3, 32, 64, 2)
    assert w.dtype == np.float32 and w.size == 52033
    assert np.array_equal(w, pi.pack_weights(0, 3, 32, 64, 2))  # seeded
    assert not np.array_equal(w, pi.pack_weights(1, 3, 32, 64, 2))


def test_xavier_scale():
    H, K = 128, 64
    w = pi.pack_weights(1, 3, K, H, 3)
    off = 3 * H
    We1 = w[off:off + H * K]
    assert abs(We1.std() - np.sqrt(2.0 / (H + K))) < 0.01
    be1 = w[off + H * K: off + H * K + H]
    assert np.all(be1 == 0.0)
    wb = pi.pack_weights(1, 3, K, H, 3, bias_scale=0.1)
    assert np.any(wb[off + H * K: off + H * K + H] != 0.0)


def test_fad_geometry():
    g = pi.fad_geometry(0, jitter=0.0)
    d = lambda a, b: np.linalg.norm(g[a] - g[b])
    assert abs(d(0, 2) - 1.22) < 1e-12 and abs(d(0, 3) - 1.32) < 1e-12 and abs(d(0, 1) - 1.10) < 1e-12
    assert abs(d(3, 4) - 0.98) < 1e-12
    assert abs(d(3, 7) - 2.70) < 1e-9 and abs(d(8, 2) - 2.70) < 1e-9  # O(h)...O(c) both H bonds
    assert 1.6 < d(4, 7) < 1.85  # H...O
    assert np.allclose(g[:, 2], 0.0)  # planar
    gj = pi.fad_geometry(3)
    assert 0.01 < np.abs(gj - g).std() < 0.1


@pytest.mark.parametrize("name,natoms,R,P", [("fad_p8", 10, 1, 8), ("fad_x64_p32", 10, 64, 32),
                                              ("water64", 192, 1, 32), ("ice512", 1536, 1, 32)])
def test_workload_shapes(name, natoms, R, P):
    w = pi.make_workload(name)
    assert w.n_atoms == natoms and w.n_replicas == R and w.P == P
    assert w.positions.shape == (R, natoms, 3) and w.species.dtype == np.int32
    assert w.net.weights.size == pi.n_weights(3, w.net.n_rbf, w.net.hidden, w.net.n_layers)
    assert w.dt == 0.25 and w.gamma == 1.0


def test_water64_molecules():
    w = pi.make_workload("water64")
    x = w.positions[0].reshape(64, 3, 3)
    oh1 = np.linalg.norm(x[:, 1] - x[:, 0], axis=1)
    oh2 = np.linalg.norm(x[:, 2] - x[:, 0], axis=1)
    assert np.allclose(oh1, 0.96) and np.allclose(oh2, 0.96)
    cosang = np.einsum("ij,ij->i", x[:, 1] - x[:, 0], x[:, 2] - x[:, 0]) / 0.96 ** 2
    assert np.allclose(np.degrees(np.arccos(cosang)), 104.5)
    O = x[:, 0]
    d = O[None] - O[:, None]
    d -= w.box * np.round(d / w.box)
    r = np.sqrt((d * d).sum(-1)) + 10 * np.eye(64)
    assert r.min() >= 2.5
    # density 1.0 g/cm^3: 64 * 18.015 amu / 12.42^3 A^3
    rho = 64 * 18.015 * 1.66053906660 / 12.42 ** 3
    assert abs(rho - 1.0) < 0.01


def test_ice_geometry():
    w = pi.make_workload("ice512")
    x = w.positions[0].reshape(512, 3, 3)
    assert np.allclose(np.linalg.norm(x[:, 1] - x[:, 0], axis=1), 0.96)
    cosang = np.einsum("ij,ij->i", x[:, 1] - x[:, 0], x[:, 2] - x[:, 0]) / 0.96 ** 2
    assert np.allclose(cosang, -1.0 / 3.0)  # tetrahedral
    assert np.allclose(w.box, 25.4) and w.T == 250.0 and w.net.gemm_dtype == 1
