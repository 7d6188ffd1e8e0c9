"""Pins for the oracle's well-tempered metadynamics and the paper's two collective variables (PAPER.md L136-152,
L164, L215, L411, L452): closed forms (two-atom Debye sum, hand geometry for s_dimer), finite-difference gradients, the
well-tempered height recursion and its continuous-time solution, bias force = -dV_G/ds grad s by finite differences."""
import numpy as np
import pytest

import oracle
from oracle import RefNet, RefPIMD, KB_EV

MASSES = np.array([1.008, 12.011, 15.999])
Q_PAPER = 4 * np.pi * np.sin(np.deg2rad(11.95)) / 1.54          # theta = 11.95 deg, lambda = 1.54 A


def _sim(pos, species, box=np.zeros(3), P=1, kind=2, T=300.0, dt=0.5, gamma=-1.0):
    return RefPIMD(np.asarray(species, np.int32), MASSES, np.asarray(pos, float)[None], box, P, T, dt, gamma, 3, RefNet(kind=kind))


def test_debye_two_atoms_closed_form():
    R = 2.3
    s = _sim([[0, 0, 0], [R, 0, 0]], [2, 0])
    f = np.array([1.0, 6.0, 8.0])
    s.metad_enable("debye", 0.1, 0.01, 10.0, 100, f_species=f, Q=Q_PAPER)
    cv, g = s.metad_cv()
    x = Q_PAPER * R
    want = 0.5 * (f[2] ** 2 + f[0] ** 2 + 2 * f[2] * f[0] * np.sin(x) / x)      # (1/N) sum over all ordered pairs, i = j included
    assert abs(cv[0, 0] - want) < 1e-13
    dg = 0.5 * 2 * f[2] * f[0] * (np.cos(x) - np.sin(x) / x) / R                  # ds/dR
    assert np.allclose(g[0, 0, 1], [dg, 0, 0], atol=1e-13) and np.allclose(g[0, 0, 0], [-dg, 0, 0], atol=1e-13)
    assert abs(Q_PAPER - 1.6896) < 1e-3


def test_dimer_cv_hand_geometry():
    # O1-H1...O2 on the x axis, O4-H2...O3 on the y axis (indices O1,H1,O2,O4,H2,O3 = 0..5)
    pos = [[0, 0, 0], [1.0, 0, 0], [2.7, 0, 0], [0, 5, 0], [0, 6.1, 0], [0, 7.5, 0]]
    s = _sim(pos, [2, 0, 2, 2, 0, 2])
    s.metad_enable("dimer", 0.1, 0.01, 10.0, 100, atoms=[0, 1, 2, 3, 4, 5])
    cv, g = s.metad_cv()
    assert abs(cv[0, 0] - ((1.0 - 1.7) + (1.1 - 1.4))) < 1e-13
    assert np.allclose(g[0, 0, 1], [2, 0, 0]) and np.allclose(g[0, 0, 4], [0, 2, 0])  # a proton between its two oxygens: both terms push it
    assert np.allclose(g[0, 0].sum(axis=0), 0)                                        # translation invariance


@pytest.mark.parametrize("cv", ["dimer", "debye"])
def test_cv_gradient_by_finite_differences(cv):
    rng = np.random.default_rng(2)
    N = 12
    box = np.array([9.0, 9.5, 10.0]) if cv == "debye" else np.zeros(3)
    pos = rng.uniform(0, 1, (N, 3)) * (box if box[0] > 0 else 4.0) + (0 if box[0] > 0 else 0)
    sp = rng.integers(0, 3, N)
    kw = dict(atoms=[0, 1, 2, 3, 4, 5]) if cv == "dimer" else dict(f_species=[1.0, 6.0, 8.0], Q=Q_PAPER)
    def value(p):
        s = _sim(p, sp, box)
        s.metad_enable(cv, 0.1, 0.01, 10.0, 100, **kw)
        return s.metad_cv()
    s0, g0 = value(pos)
    h = 1e-6
    for i, a in [(0, 0), (1, 2), (4, 1), (7, 0), (11, 2)]:
        pp = pos.copy(); pp[i, a] += h
        pm = pos.copy(); pm[i, a] -= h
        fd = (value(pp)[0][0, 0] - value(pm)[0][0, 0]) / (2 * h)
        assert abs(fd - g0[0, 0, i, a]) < 1e-6 * max(1.0, abs(fd)), (cv, i, a, fd, g0[0, 0, i, a])


def test_well_tempered_heights_follow_the_recursion_and_its_continuous_limit():
    """Depositing again and again at the same CV value: h_n = w0 exp(-V_n / (k_B T (gamma - 1))), V_n = sum of the earlier heights
    (PAPER.md L140); for small w0 the sum follows dV/dn = w0 exp(-V / (kT (gamma - 1))): V(n) = kT (gamma-1) ln(1 + n w0 / (kT (gamma-1)))."""
    T, biasf, w0 = 300.0, 10.0, 1.0 * 0.0103642697                                   # 1 kJ/mol, bias factor 10
    s = _sim([[0, 0, 0], [1.0, 0, 0], [2.7, 0, 0], [0, 5, 0], [0, 6.1, 0], [0, 7.5, 0]], [2, 0, 2, 2, 0, 2], T=T)
    s.metad_enable("dimer", 0.05, w0, biasf, 100, atoms=[0, 1, 2, 3, 4, 5])
    cv0 = s.metad_cv()[0][0, 0]
    n = 400
    for _ in range(n):
        s.metad_deposit_now()
    c, h = s.metad_gaussians()
    assert len(c) == n and np.all(c == cv0)
    kTg = KB_EV * T * (biasf - 1)
    V = 0.0
    for k in range(n):
        assert abs(h[k] - w0 * np.exp(-V / kTg)) < 1e-12 * w0
        V += h[k]
    assert abs(s.metad_bias(cv0) - V) < 1e-12 * V
    assert abs(V / (kTg * np.log(1 + n * w0 / kTg)) - 1) < 0.03
    assert abs(h[-1] / h[0] * (1 + n * w0 / kTg) - 1) < 0.03                          # h(n) = w0 / (1 + n w0 / (kT (gamma - 1))): they decay


def test_bias_force_is_minus_the_gradient_of_the_bias_energy():
    rng = np.random.default_rng(4)
    N, P = 8, 3
    box = np.array([8.0, 8.5, 9.0])
    pos = rng.uniform(0, 1, (N, 3)) * box
    sp = rng.integers(0, 3, N)
    s = RefPIMD(sp.astype(np.int32), MASSES, pos[None], box, P, 300.0, 0.5, -1.0, 3, RefNet(kind=2))
    s.metad_enable("debye", 0.3, 0.02, 10.0, 100, f_species=[1.0, 6.0, 8.0], Q=Q_PAPER)
    q, p, _ = s.get_state()
    q = q + 0.1 * rng.standard_normal(q.shape)
    s.set_state(q, p, 0)
    s.metad_deposit_now()                                        # P Gaussians, one per bead, height w0 / P each
    c, h = s.metad_gaussians()
    assert len(c) == P and np.allclose(h, 0.02 / P) and np.allclose(np.sort(c), np.sort(s.metad_cv()[0][0]))
    q[0, 1] += 0.05 * rng.standard_normal((N, 3))                # move bead 1 off its Gaussian
    s.set_state(q, p, 0)
    F = s.forces()                                               # free ring polymer: the only force is the bias force
    def energy(qq):
        s.set_state(qq, p, 0)
        cv = s.metad_cv()[0][0]
        return sum(s.metad_bias(cv[k]) for k in range(P))
    hh = 1e-5
    for k, i, a in [(1, 0, 0), (1, 3, 2), (0, 5, 1), (2, 7, 0)]:
        qp = q.copy(); qp[0, k, i, a] += hh
        qm = q.copy(); qm[0, k, i, a] -= hh
        fd = -(energy(qp) - energy(qm)) / (2 * hh)
        assert abs(fd - F[0, k, i, a]) < 1e-6 * max(1e-3, np.abs(F).max()), (k, i, a, fd, F[0, k, i, a])
    assert np.abs(F).max() > 1e-5


def test_deposition_stride_inside_step():
    s = _sim([[0, 0, 0], [1.0, 0, 0], [2.7, 0, 0], [0, 5, 0], [0, 6.1, 0], [0, 7.5, 0]], [2, 0, 2, 2, 0, 2], P=2, kind=1)
    s.metad_enable("dimer", 0.05, 0.01, 10.0, 7, atoms=[0, 1, 2, 3, 4, 5])
    s.step(20)
    c, h = s.metad_gaussians()
    assert len(c) == 2 * (20 // 7)                                # every 7 steps, one Gaussian per bead (every 100 steps)
