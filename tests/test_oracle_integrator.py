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


# ---- PILE-L friction (PAPER.md L426 names the thermostat): c1_k = exp(-gamma_k dt/2), gamma_k = 2 omega_k for
# k >= 1, gamma_0 = the input in ps^-1.  The variance pins above hold for ANY c1 in (0, 1); these three do not.
def pile_mode_ratio_setup(P, T, N, amp=100.0):
    """q = 0 and a large deterministic mode momentum p~_k = amp * sqrt(m/beta_P) on every (atom, dim, mode): (q, p, sigma)."""
    masses = np.array([1.008, 12.011, 15.999])
    sig = np.sqrt(masses[0] * AMU_INTERNAL * KB_EV * T * P)
    C = oracle.nm_matrix(P)
    pt = np.full((1, P, N, 3), amp * sig)
    p = np.einsum("jk,rkia->rjia", C, pt)
    return np.zeros((1, P, N, 3)), p, pt, C


def pile_expected_ratio(P, T, dt, gamma_ps):
    """E[p~_k(after one O A O step with F = 0, q~ = 0)] / p~_k = c1_k^2 cos(omega_k dt)."""
    wP = P * KB_EV * T / HBAR_EVFS
    wk = 2 * wP * np.sin(np.arange(P) * np.pi / P)
    gam = 2.0 * wk
    gam[0] = gamma_ps * 1e-3            # ps^-1 -> fs^-1
    return np.exp(-gam * dt) * np.cos(wk * dt)


def test_pile_friction_one_step_mean_ratio():
    P, T, dt, gamma_ps, N = 6, 300.0, 0.7, 80.0, 4096
    q, p, pt, C = pile_mode_ratio_setup(P, T, N)
    sim = RefPIMD(np.zeros(N, np.int32), np.array([1.008, 12.011, 15.999]), np.zeros((1, N, 3)), np.zeros(3), P, T, dt,
                  gamma_ps, 5, RefNet(kind=2))
    sim.set_state(q, p, 0)
    sim.step(1)
    _, p1, _ = sim.get_state()
    ratio = (np.einsum("jk,rjia->rkia", C, p1) / pt)[0].reshape(P, -1)
    want = pile_expected_ratio(P, T, dt, gamma_ps)
    # noise per sample <= sqrt(2)/amp; 3 sigma of the mean over 3N samples
    tol = 3 * np.sqrt(2.0) / 100.0 / np.sqrt(3 * N)
    got = ratio.mean(axis=1)
    assert np.all(np.abs(got - want) < tol), (got, want, tol)
    # the alternatives a plausible mistake would give are far outside: gamma_k = omega_k, gamma_0 off by 1000x
    wP = P * KB_EV * T / HBAR_EVFS
    w1 = 2 * wP * np.sin(np.pi / P)
    assert abs(np.exp(-w1 * dt) * np.cos(w1 * dt) - want[1]) > 100 * tol
    assert abs(np.exp(-gamma_ps * dt) - want[0]) > 100 * tol and abs(np.exp(-gamma_ps * 1e-6 * dt) - want[0]) > 100 * tol


def test_pile_internal_modes_are_critically_damped():
    """gamma_k = 2 omega_k is critical damping of the free ring-polymer mode: <q~_k(t)> = q0 (1 + w t) exp(-w t), no overshoot
    (closed form of the damped oscillator, independent of the integrator's own constants; small dt)."""
    P, T, dt, N, k = 8, 300.0, 0.05, 3000, 1
    masses = np.array([1.008, 12.011, 15.999])
    C = oracle.nm_matrix(P)
    wk = 2 * (P * KB_EV * T / HBAR_EVFS) * np.sin(k * np.pi / P)
    sig_q = np.sqrt(KB_EV * T * P / (masses[0] * AMU_INTERNAL)) / wk        # thermal width of the mode
    q0 = 200.0 * sig_q
    q = np.zeros((1, P, N, 3)); q[0, :, :, :] = (q0 * C[:, k])[:, None, None]
    sim = RefPIMD(np.zeros(N, np.int32), masses, np.zeros((1, N, 3)), np.zeros(3), P, T, dt, 1.0, 9, RefNet(kind=2))
    sim.set_state(q, np.zeros_like(q), 0)
    t = 0.0
    for _ in range(4):
        sim.step(60)
        t += 60 * dt
        qn, _, _ = sim.get_state()
        got = np.einsum("j,jia->ia", C[:, k], qn[0]).mean() / q0
        want = (1.0 + wk * t) * np.exp(-wk * t)
        under = np.exp(-0.5 * wk * t) * (np.cos(np.sqrt(0.75) * wk * t) + np.sin(np.sqrt(0.75) * wk * t) / np.sqrt(3.0))  # gamma = omega
        assert abs(got - want) < 2e-3, (t, got, want)
        assert abs(under - want) > 0.02


def test_centroid_friction_is_in_inverse_picoseconds():
    """P = 1, free particle: Ornstein-Uhlenbeck mean decay <p(t)> = p0 exp(-gamma t) with gamma given in ps^-1 (OBABO with
    F = 0 reproduces it exactly at the step boundaries)."""
    T, dt, gamma_ps, N = 300.0, 2.0, 25.0, 4096
    masses = np.array([1.008, 12.011, 15.999])
    sig = np.sqrt(masses[0] * AMU_INTERNAL * KB_EV * T)
    p = np.full((1, 1, N, 3), 100.0 * sig)
    sim = RefPIMD(np.zeros(N, np.int32), masses, np.zeros((1, N, 3)), np.zeros(3), 1, T, dt, gamma_ps, 2, RefNet(kind=2))
    sim.set_state(np.zeros_like(p), p, 0)
    sim.step(20)                                   # t = 40 fs = 0.04 ps: exp(-1)
    _, p1, _ = sim.get_state()
    got = (p1 / p).mean()
    assert abs(got - np.exp(-gamma_ps * 1e-3 * 20 * dt)) < 3 * 1.0 / 100.0 / np.sqrt(3 * N) + 1e-12, got
