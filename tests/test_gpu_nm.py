"""GPU parity: normal-mode integrator, PILE-L noise and estimators vs the fp64 oracle (through the C-ABI)."""
import numpy as np
import pytest

import pimd_inputs as pi
from gpu_util import make_pair, gpu_state, spread_beads

pytestmark = pytest.mark.gpu


def _spec(kind, omega=0.0):
    return pi.NetSpec(kind=kind, harmonic_omega=omega)


def _system(N=7, R=2, seed=5):
    rng = np.random.default_rng(seed)
    return rng.integers(0, 3, N).astype(np.int32), 0.3 * rng.standard_normal((R, N, 3))


@pytest.mark.parametrize("P", [1, 2, 3, 5, 8, 32, 128, 256])
@pytest.mark.parametrize("gamma", [-1.0, 20.0])
def test_harmonic_trajectory_matches_oracle(cuda_device, P, gamma):
    sp, pos = _system()
    gpu, ref = make_pair(sp, pos, np.zeros(3), P, 300.0, 0.25, gamma, 17, _spec(1, 0.2))
    qg, pg, _ = gpu_state(gpu)
    qr, pr, _ = ref.get_state()
    assert np.abs(pg - pr).max() < 1e-12 * max(1.0, np.abs(pr).max())  # initial momenta (Philox + Box-Muller)
    assert np.array_equal(qg, qr)
    spread_beads(gpu, ref)
    n = 60 if P <= 32 else 12
    gpu.step(n); ref.step(n)
    qg, pg, sg = gpu_state(gpu)
    qr, pr, sr = ref.get_state()
    assert sg == sr == n
    assert np.abs(qg - qr).max() < 1e-10, np.abs(qg - qr).max()
    assert np.abs(pg - pr).max() < 1e-9 * max(1.0, np.abs(pr).max())


def test_columns_span_several_tiles_and_ragged_tail(cuda_device):
    # 3N = 210 columns: 6 full 32-column tiles + a ragged one of 18; 3 replicas
    sp, pos = _system(N=70, R=3)
    gpu, ref = make_pair(sp, pos, np.zeros(3), 8, 250.0, 0.5, 5.0, 99, _spec(2))
    spread_beads(gpu, ref)
    gpu.step(25); ref.step(25)
    qg, pg, _ = gpu_state(gpu); qr, pr, _ = ref.get_state()
    assert np.abs(qg - qr).max() < 1e-10 and np.abs(pg - pr).max() < 1e-9 * np.abs(pr).max()


def test_estimators_match_oracle(cuda_device):
    sp, pos = _system(N=33, R=3)
    gpu, ref = make_pair(sp, pos, np.zeros(3), 8, 300.0, 0.25, 10.0, 3, _spec(1, 0.15))
    spread_beads(gpu, ref)
    gpu.step(20); ref.step(20)
    eg, er = gpu.estimators(), ref.estimators()
    assert np.allclose(eg, er, rtol=1e-9, atol=1e-11), (eg, er)
    # free ring polymer: v_pot = 0, virial terms are 0 (F = 0)
    gpu2, ref2 = make_pair(sp, pos, np.zeros(3), 4, 300.0, 0.25, 10.0, 3, _spec(2))
    gpu2.step(5); ref2.step(5)
    eg, er = gpu2.estimators(), ref2.estimators()
    assert np.allclose(eg, er, rtol=1e-9, atol=1e-11)
    assert np.all(eg[:, 3] == 0.0) and np.all(eg[:, 1] == 0.0)


def test_checkpoint_resume_bit_exact_and_deterministic(cuda_device):
    import torch
    sp, pos = _system(N=20, R=2)
    a, _ = make_pair(sp, pos, np.zeros(3), 8, 300.0, 0.25, 5.0, 1, _spec(1, 0.2))
    b, _ = make_pair(sp, pos, np.zeros(3), 8, 300.0, 0.25, 5.0, 1, _spec(1, 0.2))
    a.step(10)
    b.step(4)
    q, p, st = b.get_state()
    c, _ = make_pair(sp, pos, np.zeros(3), 8, 300.0, 0.25, 5.0, 1, _spec(1, 0.2))
    c.set_state(q, p, st)
    c.step(6)
    qa, pa, _ = a.get_state(); qc, pc, sc = c.get_state()
    assert sc == 10 and torch.equal(qa, qc) and torch.equal(pa, pc)


def test_invalid_arguments(cuda_device):
    import paper_2503_23728_b200 as pb
    sp, pos = _system()
    with pytest.raises(pb.PimdError) as e:
        pb.PIMD(sp, pi.MASSES_AMU, pos, np.zeros(3), 0, 300.0, 0.25, 1.0, 0, _spec(2))
    assert e.value.code == -1
    with pytest.raises(pb.PimdError):
        pb.PIMD(sp, pi.MASSES_AMU, pos, np.zeros(3), 4, -5.0, 0.25, 1.0, 0, _spec(2))
    w = pi.make_workload("water64")
    w.box[:] = 11.0  # < 2 r_cut
    with pytest.raises(pb.PimdError):
        pb.PIMD.from_workload(w)
    w = pi.make_workload("fad_p8")
    w.net.weights = w.net.weights[:-1]
    with pytest.raises(pb.PimdError):
        pb.PIMD.from_workload(w)


def test_pile_friction_constants_on_gpu(cuda_device):
    """PILE-L friction pinned against closed forms, not against the oracle (which could share a mistake): one O A O step with
    F = 0 from q = 0 and a large deterministic mode momentum gives E[p~_k'] / p~_k = exp(-gamma_k dt) cos(omega_k dt) with
    gamma_k = 2 omega_k (k >= 1) and gamma_0 given in ps^-1."""
    import oracle
    from oracle import KB_EV, HBAR_EVFS, AMU_INTERNAL
    import paper_2503_23728_b200 as pb
    P, T, dt, gamma_ps, N, amp = 6, 300.0, 0.7, 80.0, 4096, 100.0
    sig = np.sqrt(pi.MASSES_AMU[0] * AMU_INTERNAL * KB_EV * T * P)
    C = oracle.nm_matrix(P)      # the matrix convention N2 (pinned by C C^T = I and the ring diagonalisation)
    pt = np.full((1, P, N, 3), amp * sig)
    p = np.einsum("jk,rkia->rjia", C, pt)
    gpu = pb.PIMD(np.zeros(N, np.int32), pi.MASSES_AMU, np.zeros((1, N, 3)), np.zeros(3), P, T, dt, gamma_ps, 5, _spec(2))
    gpu.set_state(np.zeros_like(p), p, 0)
    gpu.step(1)
    _, p1, _ = gpu_state(gpu)
    got = (np.einsum("jk,rjia->rkia", C, p1) / pt)[0].reshape(P, -1).mean(axis=1)
    wk = 2 * (P * KB_EV * T / HBAR_EVFS) * np.sin(np.arange(P) * np.pi / P)
    gam = 2.0 * wk
    gam[0] = gamma_ps * 1e-3
    want = np.exp(-gam * dt) * np.cos(wk * dt)
    tol = 3 * np.sqrt(2.0) / amp / np.sqrt(3 * N)
    assert np.all(np.abs(got - want) < tol), (got, want, tol)


@pytest.mark.parametrize("transform,thermostat", [("staging", "pile_l"), ("staging", "pile_g"), ("normal_modes", "pile_g"),
                                                  ("primitive", "pile_l")])
@pytest.mark.parametrize("P", [1, 4, 32])
def test_integrator_variants_match_oracle(cuda_device, transform, thermostat, P):
    """staging transformation, primitive PIMD with explicit springs, PILE-G; the
    device builds the staging maps as matrices from the definition (F, F^-1 by elimination, inverse transposes for the momenta),
    the oracle applies the recurrences: two derivations of the same maps."""
    sp, pos = _system(N=11, R=3)
    for gamma in (-1.0, 20.0):
        if thermostat == "pile_g" and gamma < 0:
            continue
        gpu, ref = make_pair(sp, pos, np.zeros(3), P, 300.0, 0.25, gamma, 23, _spec(1, 0.2))
        gpu.set_integrator(transform, thermostat); ref.set_integrator(transform, thermostat)
        qg, pg, _ = gpu_state(gpu)
        qr, pr, _ = ref.get_state()
        assert np.abs(pg - pr).max() < 1e-12 * max(1.0, np.abs(pr).max())      # initial momenta in the chosen representation
        spread_beads(gpu, ref)
        gpu.step(40); ref.step(40)
        qg, pg, sg = gpu_state(gpu)
        qr, pr, sr = ref.get_state()
        assert sg == sr == 40
        assert np.abs(qg - qr).max() < 1e-10, (transform, thermostat, P, gamma, np.abs(qg - qr).max())
        assert np.abs(pg - pr).max() < 1e-9 * max(1.0, np.abs(pr).max())


def test_integrator_variant_is_chosen_before_the_first_step(cuda_device):
    import paper_2503_23728_b200 as pb
    sp, pos = _system()
    gpu, ref = make_pair(sp, pos, np.zeros(3), 4, 300.0, 0.25, 1.0, 1, _spec(2))
    with pytest.raises(pb.PimdError):
        gpu.set_integrator("primitive", "pile_g")       # no free mode to rescale
    gpu.step(1)
    with pytest.raises(pb.PimdError):
        gpu.set_integrator("staging", "pile_l")


def test_non_finite_positions_latch_the_nan_error(cuda_device):
    """PIMD_ERR_NAN (-4): a non-finite position or force met by a kernel is latched in the device error word and returned by the
    next synchronising call."""
    import torch
    import paper_2503_23728_b200 as pb
    sp, pos = _system()
    gpu, ref = make_pair(sp, pos, np.zeros(3), 4, 300.0, 0.25, 1.0, 1, _spec(1, 0.2))
    q, p, st = gpu.get_state()
    p[0, 1, 2, 0] = float("nan")                    # one poisoned momentum: the A step turns it into a non-finite position
    gpu.set_state(q, p, st)
    gpu.step(2)
    with pytest.raises(pb.PimdError) as e:
        gpu.sync()
    assert e.value.code == -4


def test_state_accessors_take_page_locked_host_pointers(cuda_device):
    """include/pimd.h: q, p and the cached forces may live in device memory or in page-locked host memory.  A trajectory
    driven from pinned host buffers (set -> step -> get, every step) equals the one kept on the device, bit for bit."""
    import ctypes as C
    import torch
    import paper_2503_23728_b200 as pb

    w = pi.make_workload("fad_p8")
    a = pb.PIMD.from_workload(w, device="cuda:0")
    b = pb.PIMD.from_workload(w, device="cuda:0")
    lib = pb.load_library()
    a.step(3); b.step(3)
    q, p, st = b.get_state()
    F = b.get_forces_cached()
    hq, hp, hF = q.cpu().pin_memory(), p.cpu().pin_memory(), F.cpu().pin_memory()
    for i in range(4):
        assert lib.pimd_set_state(b._h, C.c_void_p(hq.data_ptr()), C.c_void_p(hp.data_ptr()), C.c_int64(st + i)) == 0
        assert lib.pimd_set_forces_cached(b._h, C.c_void_p(hF.data_ptr())) == 0
        assert lib.pimd_step(b._h, 1) == 0
        assert lib.pimd_get_forces_cached(b._h, C.c_void_p(hF.data_ptr())) == 0
        stc = C.c_int64()
        assert lib.pimd_get_state(b._h, C.c_void_p(hq.data_ptr()), C.c_void_p(hp.data_ptr()), C.byref(stc)) == 0
        assert stc.value == st + i + 1
    a.step(4)
    qa, pa, sta = a.get_state()
    assert sta == st + 4
    assert torch.equal(qa.cpu(), hq) and torch.equal(pa.cpu(), hp)
    assert torch.equal(a.get_forces_cached().cpu(), hF)
