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
