"""GPU parity: well-tempered metadynamics with the paper's two collective variables vs the fp64 oracle."""
import numpy as np
import pytest

import pimd_inputs as pi
from gpu_util import make_pair, gpu_state, spread_beads

pytestmark = pytest.mark.gpu

Q_PAPER = 4 * np.pi * np.sin(np.deg2rad(11.95)) / 1.54
KJ_MOL = 0.0103642697                                        # eV
F_SPECIES = [1.0, 6.0, 8.0]


def _spec(kind, omega=0.0):
    return pi.NetSpec(kind=kind, harmonic_omega=omega)


def _enable(gpu, ref, cv, every, sigma=0.2, height=1.0 * KJ_MOL, biasf=10.0):
    kw = dict(atoms=[3, 4, 7, 8, 9, 2]) if cv == "dimer" else dict(f_species=F_SPECIES, Q=Q_PAPER)
    gpu.metad_enable(cv, sigma, height, biasf, every, **kw)
    ref.metad_enable(cv, sigma, height, biasf, every, **kw)


@pytest.mark.parametrize("cv,box", [("dimer", 0.0), ("debye", 0.0), ("debye", 9.0)])
def test_cv_and_gradient_match_oracle(cuda_device, cv, box):
    rng = np.random.default_rng(1)
    N = 150 if cv == "debye" else 12          # Debye: two blocks of atoms with a ragged tail
    b = np.array([box, box + 0.5, box + 1.0]) if box > 0 else np.zeros(3)
    pos = rng.uniform(0, 1, (2, N, 3)) * (b if box > 0 else 5.0)
    sp = rng.integers(0, 3, N).astype(np.int32)
    gpu, ref = make_pair(sp, pos, b, 3, 300.0, 0.5, 1.0, 5, _spec(2))
    _enable(gpu, ref, cv, 100)
    spread_beads(gpu, ref, scale=0.1)
    sg, gg = gpu.metad_cv()
    sr, gr = ref.metad_cv()
    assert np.abs(sg.cpu().numpy() - sr).max() < 1e-12 * max(1.0, np.abs(sr).max())
    assert np.abs(gg.cpu().numpy() - gr).max() < 1e-12 * max(1.0, np.abs(gr).max())
    assert np.abs(gr).max() > 1e-3


@pytest.mark.parametrize("cv,kind", [("dimer", 2), ("debye", 1)])
def test_biased_trajectory_matches_oracle(cuda_device, cv, kind):
    """Deposition every 5 steps (PAPER.md L411 uses 100), thermostat on: positions, momenta and the list of Gaussians must agree."""
    rng = np.random.default_rng(3)
    N = 10 if cv == "dimer" else 40
    pos = rng.uniform(0, 1, (2, N, 3)) * 4.0
    sp = rng.integers(0, 3, N).astype(np.int32)
    gpu, ref = make_pair(sp, pos, np.zeros(3), 4, 300.0, 0.5, 20.0, 9, _spec(kind, 0.05))
    _enable(gpu, ref, cv, 5, sigma=0.05 if cv == "dimer" else 0.5, height=20.0 * KJ_MOL)
    spread_beads(gpu, ref, scale=0.05)
    gpu.step(42); ref.step(42)
    qg, pg, sg = gpu_state(gpu)
    qr, pr, sr = ref.get_state()
    assert sg == sr == 42
    assert np.abs(qg - qr).max() < 1e-9, np.abs(qg - qr).max()
    assert np.abs(pg - pr).max() < 1e-8 * max(1.0, np.abs(pr).max())
    for r in range(2):
        cg, hg = gpu.metad_gaussians(r)
        cr, hr = ref.metad_gaussians(r)
        assert len(cg) == len(cr) == 8 * 4                       # 8 events, one Gaussian per bead
        assert np.abs(cg - cr).max() < 1e-9 and np.abs(hg - hr).max() < 1e-12
        assert np.all(hr <= hr[0] * (1 + 1e-12))                # well-tempered: no Gaussian is higher than the first (w0 / P)
        if cv == "dimer":
            assert hr[-1] < hr[0]                                # ... and on visited ground the later ones are lower


def test_bias_force_on_top_of_the_force_net(cuda_device):
    """fad_p8 with the s_dimer bias: GFN forces (fp32) plus the fp64 bias force against the oracle's sum."""
    w = pi.make_workload("fad_p8")
    from gpu_util import pair_from_workload
    gpu, ref = pair_from_workload(w)
    _enable(gpu, ref, "dimer", 100, sigma=0.05, height=50.0 * KJ_MOL)
    spread_beads(gpu, ref, scale=0.03)
    F0 = gpu.forces().cpu().numpy().astype(np.float64)
    gpu.metad_deposit_now(); ref.metad_deposit_now()
    q, p, st = ref.get_state()
    q = q + 0.02 * np.random.default_rng(0).standard_normal(q.shape)   # move off the Gaussians: a bias force appears
    ref.set_state(q, p, st)
    import torch
    gpu.set_state(torch.tensor(q, device="cuda:0"), torch.tensor(p, device="cuda:0"), st)
    Fg = gpu.forces().cpu().numpy().astype(np.float64)
    Fr = ref.forces()
    assert np.all(np.abs(Fg - Fr) <= 1e-4 * np.abs(Fr) + 1e-4), np.abs(Fg - Fr).max()
    assert np.abs(Fg - F0).max() > 1e-2                          # (the bias force is there)
