"""Pins for the oracle's ring-polymer integrator and estimators.

Closed forms used: exact conservation of the free ring-polymer Hamiltonian, time reversibility,
velocity Verlet at P=1, exact thermostat variance, and the finite-P harmonic oscillator energy
(PAPER.md L358 with the missing square restored, converging to PAPER.md L350).
"""
import numpy as np
import pytest

import oracle
from oracle import RefNet, RefPIMD, KB_EV, HBAR_EVFS, AMU_INTERNAL


def ring_energy(q, p, mass, P, T, omega=0.0):
    """H_P = sum p^2/2m + 1/2 m w_P^2 sum (q_k - q_{k+1})^2 + sum_k V(q_k); q,p [R][P][N][3]."""
    wP = P * KB_EV * T / HBAR_EVFS
    m = mass[None, None, :, None]
    kin = (p * p / (2 * m)).sum()
    dq = q - np.roll(q, -1, axis=1)
    spr = (0.5 * m * wP ** 2 * dq * dq).sum()
    pot = (0.5 * m * omega ** 2 * q * q).sum()
    return kin + spr + pot


def qho_energy_P(P, T, omega):
    """E5: <k+v> per atom (3-D) at finite P."""
    kT = KB_EV * T
    l = np.arange(1, P + 1)
    return 3 * kT * np.sum(1.0 / (1.0 + ((2 * P * kT / (HBAR_EVFS * omega)) * np.sin(l * np.pi / P)) ** 2))


def qho_energy_exact(T, omega):
    """PAPER.md L350 (x3 dimensions)."""
    hw = HBAR_EVFS * omega
    return 1.5 * hw / np.tanh(hw / (2 * KB_EV * T))


def test_qho_formula_limits():
    # E5 -> P:L350 as P grows, and = classical 3 k_B T at P = 1
    T, w = 10.0, 12.44e-3  # P:L362-364, omega read as ps^-1
    assert abs(qho_energy_P(1, T, w) - 3 * KB_EV * T) < 1e-15
    ex = qho_energy_exact(T, w)
    errs = [abs(qho_energy_P(P, T, w) - ex) / ex for P in (8, 32, 128, 4096)]
    assert errs[0] > errs[1] > errs[2] > errs[3] and errs[2] < 1e-3 and errs[3] < 2e-6
    assert abs(HBAR_EVFS * w / KB_EV - 95.0) < 0.1  # hbar*omega/k_B = 95 K: deep-quantum at 10 K


def _sys(N, R, P, kind, T=300.0, dt=0.25, gamma=-1.0, omega=0.0, seed=7, spread=0.3):
    rng = np.random.default_rng(5)
    species = rng.integers(0, 3, N).astype(np.int32)
    masses = np.array([1.008, 12.011, 15.999])
    pos = spread * rng.standard_normal((R, N, 3))
    net = RefNet(kind=kind, harmonic_omega=omega)
    sim = RefPIMD(species, masses, pos, np.zeros(3), P, T, dt, gamma, seed, net)
    return sim, masses[species] * AMU_INTERNAL


def _spread_beads(sim, scale=0.05, seed=3):
    q, p, st = sim.get_state()
    q = q + scale * np.random.default_rng(seed).standard_normal(q.shape)
    sim.set_state(q, p, st)


@pytest.mark.parametrize("P,dt", [(2, 0.25), (5, 3.0), (8, 0.25), (32, 10.0)])
def test_free_ring_polymer_exact_conservation(P, dt):
    sim, m = _sys(4, 2, P, kind=2, dt=dt)
    _spread_beads(sim)
    q0, p0, _ = sim.get_state()
    e0 = ring_energy(q0, p0, m, P, 300.0)
    sim.step(50)
    q1, p1, st = sim.get_state()
    assert st == 50
    e1 = ring_energy(q1, p1, m, P, 300.0)
    assert abs(e1 - e0) / abs(e0) < 1e-11  # exact for ANY dt
    # centroid moves uniformly: q_c(t) = q_c(0) + t p_c / m
    qc0, qc1, pc = q0.mean(1), q1.mean(1), p0.mean(1)
    assert np.allclose(qc1, qc0 + 50 * dt * pc / m[None, :, None], atol=1e-10)
    # time reversal: flip momenta, same number of steps, recover the start
    sim.set_state(q1, -p1, 0)
    sim.step(50)
    q2, p2, _ = sim.get_state()
    assert np.abs(q2 - q0).max() < 1e-9 and np.abs(p2 + p0).max() < 1e-9


def test_free_ring_mode_frequency():
    # a single excited mode k oscillates at omega_k = 2 w_P sin(k pi / P): after one period it returns
    P, T, k = 8, 300.0, 3
    sim, m = _sys(1, 1, P, kind=2, T=T)
    C = oracle.nm_matrix(P)
    wk = 2 * (P * KB_EV * T / HBAR_EVFS) * np.sin(k * np.pi / P)
    q = np.zeros((1, P, 1, 3)); p = np.zeros((1, P, 1, 3))
    q[0, :, 0, 0] = 0.1 * C[:, k]
    nsteps = 40
    sim2 = RefPIMD(np.zeros(1, np.int32), np.array([1.008, 12.011, 15.999]), np.zeros((1, 1, 3)), np.zeros(3), P, T,
                   2 * np.pi / wk / nsteps, -1.0, 0, RefNet(kind=2))
    sim2.set_state(q, p, 0)
    sim2.step(nsteps // 2)
    qh, _, _ = sim2.get_state()
    assert np.allclose(qh, -q, atol=1e-12)
    sim2.step(nsteps // 2)
    qf, pf, _ = sim2.get_state()
    assert np.allclose(qf, q, atol=1e-12) and np.abs(pf).max() < 1e-10


def test_harmonic_nve_bounded_no_drift():
    P, T, w = 8, 300.0, 0.2
    sim, m = _sys(6, 1, P, kind=1, omega=w)
    _spread_beads(sim)
    q, p, _ = sim.get_state()
    e0 = ring_energy(q, p, m, P, T, w)
    dev = []
    for _ in range(40):
        sim.step(100)
        q, p, _ = sim.get_state()
        dev.append((ring_energy(q, p, m, P, T, w) - e0) / e0)
    dev = np.array(dev)
    assert np.abs(dev).max() < 5e-3  # O(dt^2) fluctuation
    assert abs(dev[:20].mean() - dev[20:].mean()) < 2e-3  # no secular drift


def test_P1_is_velocity_verlet():
    # P = 1, thermostat off: textbook velocity Verlet on V = 1/2 m w^2 r^2
    w, dt, n = 0.2, 0.25, 37
    sim, m = _sys(3, 2, 1, kind=1, omega=w, dt=dt)
    q, p, _ = sim.get_state()
    sim.step(n)
    q1, p1, _ = sim.get_state()
    mm = m[None, None, :, None]
    f = -mm * w * w * q
    for _ in range(n):
        p = p + 0.5 * dt * f
        q = q + dt * p / mm
        f = -mm * w * w * q
        p = p + 0.5 * dt * f
    assert np.abs(q - q1).max() < 1e-12 and np.abs(p - p1).max() < 1e-12


def test_initial_momenta_and_thermostat_variance():
    # N5: p~_k ~ N(0, m/beta_P) for every mode; O step keeps that variance exactly (c1^2 + c2^2 = 1)
    P, T, N = 4, 300.0, 3000
    species = np.zeros(N, np.int32)
    masses = np.array([1.008, 12.011, 15.999])
    sim = RefPIMD(species, masses, np.zeros((1, N, 3)), np.zeros(3), P, T, 0.25, 20.0, 11, RefNet(kind=2))
    C = oracle.nm_matrix(P)
    var_want = masses[0] * AMU_INTERNAL * KB_EV * T * P
    for nstep in (0, 3):
        sim.step(nstep)
        _, p, _ = sim.get_state()
        pt = np.einsum("jk,rjia->rkia", C, p)
        for k in range(P):
            v = pt[0, k].var()
            assert abs(v / var_want - 1.0) < 0.05, (nstep, k, v / var_want)
    # P=1 initial momentum equals sqrt(m k T) * xi(tag 2) exactly
    sim1 = RefPIMD(species[:5], masses, np.zeros((1, 5, 3)), np.zeros(3), 1, T, 0.25, 1.0, 11, RefNet(kind=2))
    _, p1, _ = sim1.get_state()
    for i in range(5):
        xi = oracle.normal3(11, i, 0, 0, 2)
        assert np.allclose(p1[0, 0, i], np.sqrt(masses[0] * AMU_INTERNAL * KB_EV * T) * xi, rtol=1e-14)


def test_thermostat_noise_is_keyed_by_step_and_seed():
    a, _ = _sys(3, 1, 4, kind=2, gamma=5.0, seed=1)
    b, _ = _sys(3, 1, 4, kind=2, gamma=5.0, seed=1)
    c, _ = _sys(3, 1, 4, kind=2, gamma=5.0, seed=2)
    a.step(10); b.step(4); b.step(6); c.step(10)
    qa, pa, _ = a.get_state(); qb, pb, _ = b.get_state(); qc, pc, _ = c.get_state()
    assert np.array_equal(qa, qb) and np.array_equal(pa, pb)  # split runs are identical
    assert not np.allclose(pa, pc)
    # checkpoint / resume through get_state / set_state is bit exact
    d, _ = _sys(3, 1, 4, kind=2, gamma=5.0, seed=1)
    d.step(4)
    q, p, st = d.get_state()
    e, _ = _sys(3, 1, 4, kind=2, gamma=5.0, seed=1)
    e.set_state(q, p, st)
    e.step(6)
    qe, pe, _ = e.get_state()
    assert np.array_equal(qe, qa) and np.array_equal(pe, pa)


def test_qho_estimators_reach_finite_P_energy():
    """Harmonic well + PILE-L: E1+E4, E2+E4, E3+E4 all -> E5 (finite-P target), not the P->inf value."""
    P, T, w, N = 8, 300.0, 0.2, 1024
    species = np.zeros(N, np.int32)
    masses = np.array([1.008, 12.011, 15.999])
    sim = RefPIMD(species, masses, np.zeros((1, N, 3)), np.zeros(3), P, T, 0.25, 50.0, 3,
                  RefNet(kind=1, harmonic_omega=w))
    sim.step(1500)
    acc = np.zeros(5); n = 0
    for _ in range(300):
        sim.step(10)
        acc += sim.estimators()[0]; n += 1
    acc /= n
    target = qho_energy_P(P, T, w)  # per atom
    exact = qho_energy_exact(T, w)
    assert abs(target - 0.19069) < 2e-5  # SURVEY 8(c) pins: 0.19069 eV for these parameters
    for kin in acc[:3]:
        e = (kin + acc[3]) / N
        assert abs(e - target) / target < 0.005, (e, target)
        assert abs(e - exact) / exact > 0.02  # distinguishes finite-P from P->inf (4.6 % apart)
    assert abs(acc[4] - T) / T < 0.03  # centroid temperature
