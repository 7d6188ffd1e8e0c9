"""pimd_debye_cv_static: the Debye collective variable through the entry point that allocates nothing (include/pimd.h).

Its scratch is a fixed device array inside the library that every call shares and that keeps the last call's contents, so
the test calls it twice in a row on DIFFERENT inputs (the second with fewer systems and fewer atom blocks than the first:
stale partial sums of the first call sit right behind the entries the second one uses) and compares each result with the
existing path, pimd_metad_cv on a context, on the same positions.  Both paths use the same block partition and summation
order, so the comparison is exact; the stated tolerance is the one of tests/test_gpu_metad.py (1e-12 relative).

This file is meant to be collected last (pytest -x stops at the first failure).
"""
import numpy as np
import pytest

import pimd_inputs as pi
from gpu_util import make_pair

pytestmark = pytest.mark.gpu

Q_PAPER = 4 * np.pi * np.sin(np.deg2rad(11.95)) / 1.54
F_SPECIES = [1.0, 6.0, 8.0]
RTOL = 1e-12


def _existing_path(sp, pos, box, P, seed):
    """CV and gradient of every bead-system from a context (pimd_metad_cv), and the positions they were evaluated at."""
    gpu, ref = make_pair(sp, pos, box, P, 300.0, 0.5, 1.0, 5, pi.NetSpec(kind=2, harmonic_omega=0.0))
    gpu.metad_enable("debye", 0.2, 0.01, 10.0, 100, f_species=F_SPECIES, Q=Q_PAPER)
    q, p, st = gpu.get_state()
    rng = np.random.default_rng(seed)
    import torch
    q = q + torch.as_tensor(0.1 * rng.standard_normal(tuple(q.shape)), device=q.device)
    gpu.set_state(q, p, st)
    s, g = gpu.metad_cv()
    gpu.sync()
    return q.contiguous(), s, g


def _check_case(N, R, P, box, seed):
    import torch
    import paper_2503_23728_b200 as pb

    rng = np.random.default_rng(seed)
    b = np.asarray(box, dtype=np.float64)
    pos = rng.uniform(0, 1, (R, N, 3)) * (b if b[0] > 0 else 5.0)
    sp = rng.integers(0, 3, N).astype(np.int32)
    q, s_ref, g_ref = _existing_path(sp, pos, b, P, seed + 1)
    dev = q.device
    q3 = q.reshape(R * P, N, 3)
    s_out = torch.full((R * P,), float("nan"), dtype=torch.float64, device=dev)
    g_out = torch.full((R * P, N, 3), float("nan"), dtype=torch.float64, device=dev)
    pb.debye_cv_static(q3, torch.as_tensor(sp, device=dev), b, F_SPECIES, Q_PAPER, s_out, g_out)
    torch.cuda.synchronize(dev)
    s_ref = s_ref.reshape(-1).cpu().numpy(); g_ref = g_ref.reshape(R * P, N, 3).cpu().numpy()
    s_new = s_out.cpu().numpy(); g_new = g_out.cpu().numpy()
    assert np.isfinite(s_new).all() and np.isfinite(g_new).all()
    assert np.abs(g_ref).max() > 1e-3
    assert np.abs(s_new - s_ref).max() <= RTOL * max(1.0, np.abs(s_ref).max()), np.abs(s_new - s_ref).max()
    assert np.abs(g_new - g_ref).max() <= RTOL * max(1.0, np.abs(g_ref).max()), np.abs(g_new - g_ref).max()
    # value only (no gradient buffer)
    s_only = torch.empty_like(s_out)
    pb.debye_cv_static(q3, torch.as_tensor(sp, device=dev), b, F_SPECIES, Q_PAPER, s_only, None)
    torch.cuda.synchronize(dev)
    assert torch.equal(s_only, s_out)


def test_two_calls_in_a_row_match_the_context_path(cuda_device):
    # first call: 3 atom blocks with a ragged tail, 6 bead-systems, periodic; second: 1 block, 2 bead-systems, open boundary
    _check_case(N=300, R=2, P=3, box=[9.0, 9.5, 10.0], seed=11)
    _check_case(N=70, R=1, P=2, box=[0.0, 0.0, 0.0], seed=12)


def test_sizes_beyond_the_fixed_scratch_are_rejected(cuda_device):
    import torch
    import paper_2503_23728_b200 as pb

    dev = torch.device("cuda:0")
    sp = torch.zeros(8, dtype=torch.int32, device=dev)
    q = torch.zeros((257, 8, 3), dtype=torch.float64, device=dev)      # 257 systems > 256
    with pytest.raises(pb.PimdError) as e:
        pb.debye_cv_static(q, sp, np.zeros(3), F_SPECIES, Q_PAPER, torch.empty(257, dtype=torch.float64, device=dev))
    assert e.value.code == -1 and "max 256" in str(e.value)
    sp = torch.zeros(8193, dtype=torch.int32, device=dev)               # 65 blocks of 128 atoms > 64
    q = torch.zeros((1, 8193, 3), dtype=torch.float64, device=dev)
    with pytest.raises(pb.PimdError) as e:
        pb.debye_cv_static(q, sp, np.zeros(3), F_SPECIES, Q_PAPER, torch.empty(1, dtype=torch.float64, device=dev))
    assert e.value.code == -1 and "max 8192" in str(e.value)
