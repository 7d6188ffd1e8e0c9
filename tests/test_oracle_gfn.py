"""Pins for the oracle's GFN-style direct-force network.

The paper prints no network output, so numerical parity is pinned by what the construction
fixes: momentum / angular-momentum conservation of central pair forces, E(3) equivariance,
permutation equivariance, periodic-image invariance, continuity at the cutoff, an L=0 two-atom
hand evaluation, and an independently written dense numpy evaluation in another algebraic form.
"""
import numpy as np
import pytest

import pimd_inputs as pi
from oracle import RefNet, RefPIMD

from dense_gfn import dense_forces, unpack, silu

MASSES = np.array([1.008, 12.011, 15.999])


def ref_forces(species, x, box, net):
    sim = RefPIMD(species, MASSES, x[None], box, 1, 300.0, 0.25, -1.0, 0, net)
    return sim.forces()[0, 0]


def make_net(K=8, H=16, L=2, rc=3.0, seed=0, bias=0.2):
    return RefNet(0, 3, K, H, L, rc, 1.0 / 7.0, 0.3, 0.0, pi.pack_weights(seed, 3, K, H, L, bias_scale=bias))


def rand_rot(rng):
    q = rng.standard_normal(4); q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


@pytest.fixture(scope="module")
def cluster():
    rng = np.random.default_rng(1)
    x = rng.uniform(0, 4.0, (14, 3))
    sp = rng.integers(0, 3, 14).astype(np.int32)
    return sp, x


def test_conservation_and_equivariance_open(cluster):
    sp, x = cluster
    net = make_net()
    box = np.zeros(3)
    F = ref_forces(sp, x, box, net)
    scale = np.abs(F).max()
    assert scale > 1e-3
    assert np.abs(F.sum(0)).max() < 1e-13 * max(1, scale) * len(x)  # sum F = 0
    assert np.abs(np.cross(x, F).sum(0)).max() < 1e-12  # sum r x F = 0 (central pair forces)
    rng = np.random.default_rng(2)
    Rm = rand_rot(rng); t = rng.standard_normal(3) * 5
    F2 = ref_forces(sp, x @ Rm.T + t, box, net)
    assert np.abs(F2 - F @ Rm.T).max() < 1e-12  # F(Rx + t) = R F(x)
    perm = rng.permutation(len(x))
    F3 = ref_forces(sp[perm], x[perm], box, net)
    assert np.abs(F3 - F[perm]).max() < 1e-13
    # species matter
    sp2 = sp.copy(); sp2[0] = (sp2[0] + 1) % 3
    assert np.abs(ref_forces(sp2, x, box, net) - F).max() > 1e-4


def test_periodic_invariants():
    rng = np.random.default_rng(3)
    box = np.array([6.5, 7.0, 9.2]); rc = 3.0
    x = rng.uniform(0, 1, (50, 3)) * box
    sp = rng.integers(0, 3, 50).astype(np.int32)
    net = make_net(rc=rc)
    F = ref_forces(sp, x, box, net)
    assert np.abs(F.sum(0)).max() < 1e-12
    y = x.copy(); y[3] += [box[0], 0, -box[2]]; y[20] -= 2 * box
    assert np.abs(ref_forces(sp, y, box, net) - F).max() < 1e-11  # image shift
    assert np.abs(ref_forces(sp, x + [0.37, -1.2, 5.5], box, net) - F).max() < 1e-11  # translation


def test_matches_independent_dense_numpy(cluster):
    sp, x = cluster
    for (K, H, L, rc, box) in [(8, 16, 2, 3.0, np.zeros(3)), (6, 8, 3, 2.5, np.array([5.5, 6.0, 5.1])), (5, 8, 0, 3.0, np.zeros(3))]:
        net = make_net(K, H, L, rc, seed=4)
        xx = x if box[0] == 0 else x * 1.2
        F = ref_forces(sp, xx, box, net)
        Fd = dense_forces(sp, xx, box, net.weights, 3, K, H, L, net.r_cut, net.agg_norm, net.force_scale)
        assert np.abs(F - Fd).max() < 1e-12 * max(1.0, np.abs(F).max()), (K, H, L)


def test_gross_pair_term_scale_matches_dense_numpy(cluster):
    """The diagnostic the bf16 parity bound is stated against: the sum of the magnitudes of all terms of F_i (>= |F_i|)."""
    sp, x = cluster
    for (K, H, L, rc, box) in [(8, 16, 2, 3.0, np.zeros(3)), (6, 8, 3, 2.5, np.array([5.5, 6.0, 5.1]))]:
        net = make_net(K, H, L, rc, seed=4)
        xx = x if box[0] == 0 else x * 1.2
        sim = RefPIMD(sp, MASSES, xx[None], box, 1, 300.0, 0.25, -1.0, 0, net)
        F, g = sim.forces()[0, 0], sim.force_gross()[0, 0]
        Fd, gd = dense_forces(sp, xx, box, net.weights, 3, K, H, L, net.r_cut, net.agg_norm, net.force_scale, gross=True)
        assert np.abs(g - gd).max() < 1e-12 * max(1.0, gd.max())
        assert np.all(np.linalg.norm(F, axis=1) <= g + 1e-12) and g.max() > 0


def test_two_atoms_L0_by_hand():
    K, H, rc = 6, 8, 4.0
    net = make_net(K, H, 0, rc, seed=5)
    p = unpack(net.weights, 3, K, H, 0)
    d = 1.7
    x = np.array([[0.1, 0.2, 0.3], [0.1 + d, 0.2, 0.3]])
    F = ref_forces(np.array([0, 2], np.int32), x, np.zeros(3), net)
    dl = rc / (K - 1)
    g = np.exp(-((d - dl * np.arange(K)) ** 2) / (2 * dl * dl))
    e0 = p["W_e2"] @ silu(p["W_e1"] @ g + p["b_e1"]) + p["b_e2"]
    s = p["w_f2"] @ silu(p["W_f1"] @ e0 + p["b_f1"]) + p["b_f2"]
    c = 0.5 * (np.cos(np.pi * d / rc) + 1)
    f = net.force_scale * c * s
    # u_01 = (r_0 - r_1)/d = -x_hat: atom 0 feels f * (-x_hat), atom 1 the opposite
    assert np.allclose(F[0], [-f, 0, 0], atol=1e-14) and np.allclose(F[1], [f, 0, 0], atol=1e-14)
    assert abs(f) > 1e-4


def test_continuity_at_cutoff_and_isolated_atom():
    net = make_net(rc=3.0)
    sp = np.array([0, 1, 2], np.int32)
    base = np.array([[0, 0, 0], [1.0, 0.2, 0], [0, 0, 0]], float)
    Fs = []
    for d in (3.0 - 1e-7, 3.0 + 1e-7):
        x = base.copy(); x[2] = [0, d, 0]
        Fs.append(ref_forces(sp, x, np.zeros(3), net))
    assert np.abs(Fs[0] - Fs[1]).max() < 1e-9  # c(d) -> 0 smoothly
    x = base.copy(); x[2] = [50, 50, 50]
    F = ref_forces(sp, x, np.zeros(3), net)
    assert np.all(F[2] == 0.0)  # no neighbours -> zero force


def test_workload_force_magnitudes():
    # G6 constants give O(1) eV/A forces (SURVEY: rms 0.58 FAD / 0.68 water-64 at step 0)
    for name, lo, hi in [("fad_p8", 0.2, 1.5), ("water64", 0.2, 1.5)]:
        w = pi.make_workload(name)
        F = ref_forces(w.species, w.positions[0], w.box, RefNet.from_spec(w.net))
        rms = np.sqrt((F ** 2).sum(-1).mean())
        assert lo < rms < hi, (name, rms)
        assert np.abs(F.sum(0)).max() < 1e-10
