"""Pins for the oracle's integrator variants: staging transformation, primitive PIMD with
explicit bead springs, PILE-G global thermostat.

What fixes them, other than the oracle itself: the definition of the staging variables (inverse pair, the spring-energy
identity that makes staging modes independent oscillators, the chain rule for momenta); exact conservation and exact
periodicity of the free ring polymer in staging variables for any dt; a second-order integrator converges as dt^2
(primitive); the strong-friction and zero-friction limits of the stochastic velocity rescaling, its invariance of the
direction of the centroid momentum, and the equilibrium kinetic energy it samples.
"""
import numpy as np
import pytest

import oracle
from oracle import RefNet, RefPIMD, KB_EV, HBAR_EVFS, AMU_INTERNAL
from oracle.ref import stage_map
from test_oracle_integrator import ring_energy, qho_energy_P, _sys, _spread_beads


def _matrix(name, P):
    """columns = the map applied to the unit vectors"""
    return np.stack([stage_map(name, np.eye(P)[k]) for k in range(P)], axis=1)


@pytest.mark.parametrize("P", [1, 2, 3, 4, 8, 32])
def test_staging_maps_against_their_definition(P):
    rng = np.random.default_rng(P)
    q = rng.standard_normal(P)
    u = stage_map("fwd", q)
    # definition (PAPER.md L52 names the transformation; variables as in the oracle header): u_0 = q_0, u_j = q_j - (j q_{j+1} + q_0)/(j+1)
    qn = np.roll(q, -1)
    want = np.array([q[0]] + [q[j] - (j * qn[j] + q[0]) / (j + 1) for j in range(1, P)])
    assert np.abs(u - want).max() < 1e-14
    assert np.abs(stage_map("inv", u) - q).max() < 1e-13                       # inverse pair
    # the ring springs are diagonal in the staging variables with lam_j = (j+1)/j: independent oscillators at w_P
    lam = np.array([0.0] + [(j + 1) / j for j in range(1, P)])
    assert abs(((q - qn) ** 2).sum() - (lam * u * u).sum()) < 1e-12 * max(1.0, (q * q).sum())
    # canonical momenta: p_u = (dq/du)^T p_q and p_q = (du/dq)^T p_u
    F, J = _matrix("fwd", P), _matrix("inv", P)                                 # du/dq, dq/du
    assert np.abs(F @ J - np.eye(P)).max() < 1e-13
    f = rng.standard_normal(P)
    assert np.abs(stage_map("force", f) - J.T @ f).max() < 1e-13
    assert np.abs(stage_map("mom_to_bead", f) - F.T @ f).max() < 1e-13


def _staging_energy(q, p, m, P, T, omega=0.0):
    """Conserved quantity of the staging integrator: the staging modes carry the kinetic masses m lam_k (the fictitious masses m'
    of PAPER.md L50-52), H = sum p_u^2 / (2 m lam) + sum 1/2 m lam w_P^2 u^2 + V; u, p_u recovered from the bead arrays with F and J^T."""
    F, J = _matrix("fwd", P), _matrix("inv", P)
    u = np.einsum("kj,rjia->rkia", F, q)
    pu = np.einsum("jk,rjia->rkia", J, p)
    lam_k = np.array([1.0] + [(j + 1) / j for j in range(1, P)])[None, :, None, None]
    lam_s = np.array([0.0] + [(j + 1) / j for j in range(1, P)])[None, :, None, None]
    wP = P * KB_EV * T / HBAR_EVFS
    mm = m[None, None, :, None]
    return ((pu ** 2 / (2 * mm * lam_k)).sum() + (0.5 * mm * lam_s * wP ** 2 * u ** 2).sum() + (0.5 * mm * omega ** 2 * q * q).sum()), u, pu


@pytest.mark.parametrize("P,dt", [(2, 0.25), (4, 0.5), (8, 3.0), (32, 10.0)])
def test_staging_free_ring_is_propagated_exactly(P, dt):
    """Staging PIMD gives the modes the masses m (j+1)/j, so every mode j >= 1 is an oscillator at w_P and u_0 a free particle:
    the staging Hamiltonian is conserved to round-off for ANY dt, and after one period 2 pi / w_P all u_j (j >= 1) are back."""
    T = 300.0
    s, m = _sys(4, 2, P, kind=2, T=T, dt=dt)
    s.set_integrator("staging")
    _spread_beads(s)
    q0, p0, _ = s.get_state()
    e0, u0, pu0 = _staging_energy(q0, p0, m, P, T)
    s.step(50)
    q1, p1, _ = s.get_state()
    e1, _, _ = _staging_energy(q1, p1, m, P, T)
    assert abs(e1 - e0) < 1e-10 * abs(e0)
    # one period in n steps
    wP = P * KB_EV * T / HBAR_EVFS
    n = 16
    s2, _ = _sys(4, 2, P, kind=2, T=T, dt=2 * np.pi / wP / n)
    s2.set_integrator("staging")
    s2.set_state(q0, p0, 0)
    s2.step(n)
    q2, p2, _ = s2.get_state()
    _, u2, pu2 = _staging_energy(q2, p2, m, P, T)
    assert np.abs(u2[:, 1:] - u0[:, 1:]).max() < 1e-9 * max(1.0, np.abs(u0).max())
    assert np.abs(pu2 - pu0).max() < 1e-9 * np.abs(pu0).max()
    tau = 2 * np.pi / wP
    assert np.abs(u2[:, 0] - (u0[:, 0] + tau * pu0[:, 0] / m[None, :, None])).max() < 1e-9 * max(1.0, np.abs(u2).max())


def test_staging_harmonic_well_energy_is_bounded():
    P, T, omega = 8, 300.0, 0.2
    s, m = _sys(3, 2, P, kind=1, T=T, dt=0.25, omega=omega)
    s.set_integrator("staging")
    _spread_beads(s)
    q0, p0, _ = s.get_state()
    e0, _, _ = _staging_energy(q0, p0, m, P, T, omega)
    es = []
    for _ in range(10):
        s.step(200)
        q, p, _ = s.get_state()
        es.append(_staging_energy(q, p, m, P, T, omega)[0])
    es = np.array(es)                      # bounded O((omega dt)^2) oscillation, no drift
    assert np.abs(es - e0).max() < 1e-2 * abs(e0) and abs(es[5:].mean() - es[:5].mean()) < 2e-3 * abs(e0)


def test_primitive_converges_to_the_exact_propagation_as_dt_squared():
    """Primitive PIMD integrates the springs with velocity Verlet: second order in dt against the exact normal-mode propagation."""
    P, T, omega = 8, 300.0, 0.1
    ref, m = _sys(3, 1, P, kind=1, dt=0.0125, omega=omega)
    _spread_beads(ref)
    q0, p0, _ = ref.get_state()
    ref.step(320)                                       # 4 fs, the fine normal-mode run is the reference
    qx, _, _ = ref.get_state()
    errs = []
    for dt, n in [(0.1, 40), (0.05, 80), (0.025, 160)]:
        s, _ = _sys(3, 1, P, kind=1, dt=dt, omega=omega)
        s.set_integrator("primitive")
        s.set_state(q0, p0, 0)
        s.step(n)
        errs.append(np.abs(s.get_state()[0] - qx).max())
    assert errs[0] > errs[1] > errs[2] and errs[2] < 1e-3
    assert 3.0 < errs[0] / errs[1] < 5.0 and 3.0 < errs[1] / errs[2] < 5.0, errs
    # and the ring Hamiltonian has no drift over a long run (bounded O(dt^2) fluctuation)
    s, m = _sys(3, 1, P, kind=2, dt=0.05)
    s.set_integrator("primitive")
    s.set_state(q0, p0, 0)
    e0 = ring_energy(q0, p0, m, P, T)
    es = []
    for _ in range(10):
        s.step(200)
        q, p, _ = s.get_state()
        es.append(ring_energy(q, p, m, P, T))
    assert np.abs(np.array(es) - e0).max() < 2e-3 * abs(e0) and abs(es[-1] - es[0]) < 1e-3 * abs(e0)


def test_initial_momenta_have_the_mode_variances():
    """N5 in staging variables: p_u,k ~ N(0, m lam_k / beta_P); checked on the staging momenta recovered with J^T."""
    P, T, N, R = 8, 300.0, 6, 400
    s, m = _sys(N, R, P, kind=2, T=T, gamma=1.0)
    s.set_integrator("staging")
    _, p, _ = s.get_state()
    J = _matrix("inv", P)
    pu = np.einsum("jk,rjia->rkia", J, p)                                       # p_u = J^T p_q
    lam = np.array([1.0] + [(j + 1) / j for j in range(1, P)])
    var = (pu ** 2 / m[None, None, :, None]).mean(axis=(0, 2, 3))               # <p_u^2 / m> per mode
    want = lam * KB_EV * T * P
    assert np.all(np.abs(var / want - 1.0) < 5 * np.sqrt(2.0 / (R * N * 3)))


def test_staging_pile_reaches_the_finite_P_energy():
    """Same target as the normal-mode run (PAPER.md L358 with the square restored): the thermostatted staging integrator samples it."""
    P, T, omega, N, R = 4, 300.0, 0.2, 1, 256
    rng = np.random.default_rng(0)
    net = RefNet(kind=1, harmonic_omega=omega)
    s = RefPIMD(np.zeros(N, np.int32), np.array([1.008, 12.011, 15.999]), 0.05 * rng.standard_normal((R, N, 3)), np.zeros(3),
                P, T, 0.5, 50.0, 11, net)
    s.set_integrator("staging")
    s.step(400)
    acc = []
    for _ in range(60):
        s.step(20)
        e = s.estimators()
        acc.append((e[:, 2] + e[:, 3]).mean())                                  # centroid-virial kinetic + potential
    target = qho_energy_P(P, T, omega)
    assert abs(np.mean(acc) / target - 1.0) < 0.02, (np.mean(acc), target)


def _centroid(p, P):
    return p.sum(axis=1) / np.sqrt(P)                                           # mode 0 of the normal-mode matrix: [R][N][3]


def test_pile_g_limits_and_direction():
    P, T, N, R, seed = 4, 300.0, 5, 2, 21
    kTP = KB_EV * T * P
    # strong friction (c = exp(-gamma dt/2) -> 0): after a step the kinetic energy of the replica's centroid modes is the chi-square
    # draw (R1^2 + S) k_B T P / 2 of the second O of that step (tag 1), whatever it was before; the DIRECTION of the 3N-vector
    # of centroid momenta (in units of sqrt(m)) is kept up to the sign of alpha; free ring polymer, so B and A do not touch it
    s, m = _sys(N, R, P, kind=2, T=T, dt=1.0, gamma=2.0e5, seed=seed)
    s.set_integrator("normal_modes", "pile_g")
    _, p0, _ = s.get_state()
    s.step(1)
    _, p1, _ = s.get_state()
    c0, c1 = _centroid(p0, P), _centroid(p1, P)
    for r in range(R):
        xi = np.array([oracle.normal3(seed, i, r * P + 0, 0, 1) for i in range(N)])   # [N][3] normals of (atom, mode 0, step 0, tag 1)
        chi2 = (xi ** 2).sum()
        K1 = (c1[r] ** 2 / (2 * m[:, None])).sum()
        assert abs(K1 / (0.5 * kTP * chi2) - 1.0) < 1e-9
        ratio = (c1[r] / c0[r]).ravel()
        assert np.abs(ratio / ratio[0] - 1.0).max() < 1e-9                      # one factor for all atoms and dimensions
    # no friction (c = 1): alpha = 1, the centroid momenta are untouched; the internal modes are thermostatted as in PILE-L
    s, m = _sys(N, R, P, kind=2, T=T, dt=1.0, gamma=0.0, seed=seed)
    s.set_integrator("normal_modes", "pile_g")
    _, p0, _ = s.get_state()
    s.step(3)
    _, p1, _ = s.get_state()
    assert np.abs(_centroid(p1, P) - _centroid(p0, P)).max() < 1e-12 * np.abs(p0).max()
    assert np.abs(p1 - p0).max() > 1e-3 * np.abs(p0).max()


def test_pile_g_without_friction_is_the_default_integrator():
    """PILE-G only replaces the thermostat of the free mode: with the thermostat off (NVE) the normal-mode PILE-G path must follow
    the default normal-mode integrator (harmonic well, so that B, A and the bead <-> mode maps of q AND p all matter)."""
    a, _ = _sys(5, 2, 8, kind=1, dt=0.5, omega=0.2)
    b, _ = _sys(5, 2, 8, kind=1, dt=0.5, omega=0.2)
    b.set_integrator("normal_modes", "pile_g")
    _spread_beads(a)
    q0, p0, _ = a.get_state()
    b.set_state(q0, p0, 0)
    a.step(40); b.step(40)
    qa, pa, _ = a.get_state(); qb, pb, _ = b.get_state()
    assert np.abs(qa - qb).max() < 1e-12 * max(1.0, np.abs(qa).max()) and np.abs(pa - pb).max() < 1e-12 * max(1.0, np.abs(pa).max())


def test_pile_g_samples_the_canonical_centroid_kinetic_energy():
    P, T, N, R = 4, 300.0, 4, 8
    s, m = _sys(N, R, P, kind=2, T=T, dt=1.0, gamma=500.0, seed=5)             # gamma dt = 0.5: quick decorrelation
    s.set_integrator("staging", "pile_g")
    Ks = []
    for _ in range(1500):
        s.step(1)
        _, p, _ = s.get_state()
        pu0 = p.sum(axis=1)                                                     # staging free mode: p_u0 = sum_j p_qj
        Ks.append((pu0 ** 2 / (2 * m[None, :, None])).sum(axis=(1, 2)))
    Ks = np.array(Ks)
    want = 1.5 * N * KB_EV * T * P                                              # 3N/2 k_B T P
    assert abs(Ks.mean() / want - 1.0) < 0.03, Ks.mean() / want
    assert abs(Ks.var() / (want ** 2 / (1.5 * N)) - 1.0) < 0.2                  # chi-square with 3N degrees of freedom
