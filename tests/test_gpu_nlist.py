"""GPU parity: neighbour lists must be BIT-EXACT against the oracle (CSR row_ptr and col)."""
import numpy as np
import pytest

import torch

import oracle
import paper_2503_23728_b200 as pb
import pimd_inputs as pi
from gpu_util import make_pair, pair_from_workload, spread_beads

pytestmark = pytest.mark.gpu


def _compare(gpu, ref):
    rp, col = gpu.nlist()
    rp, col = rp.cpu().numpy(), col.cpu().numpy()
    rr, cr = ref.nlist()
    assert rp.shape == rr.shape and np.array_equal(rp, rr)
    assert col.shape == cr.shape and np.array_equal(col, cr)
    return rp, col


def _net(rc, K=32, H=64):
    return pi.NetSpec(0, 3, K, H, 1, 0, rc, 0.1, 0.1, 0.0, pi.pack_weights(0, 3, K, H, 1))


@pytest.mark.parametrize("ncell", [0, 2, 3, 4, 5])
def test_random_boxes_bit_exact(cuda_device, ncell):
    rng = np.random.default_rng(ncell)
    rc = 2.0
    if ncell == 0:
        box = np.zeros(3); x = rng.uniform(0, 5, (2, 40, 3))
    else:
        box = np.array([ncell * rc + 0.3, ncell * rc + 0.9, ncell * rc + 0.01])
        x = rng.uniform(0, 1, (2, 60 * ncell, 3)) * box
        x[:, ::7] += box * rng.integers(-3, 4, (2, len(x[0, ::7]), 3))
        x[:, 1] = [0.0, 0.0, 0.0]
        x[:, 2] = [rc, 2 * rc, box[2]]
        x[:, 3] = x[:, 1] + [rc, 0, 0]   # exactly at the cutoff: excluded
        x[:, 4] = [-1e-300, box[1] * (1 - 1e-17), 0.5]
    sp = rng.integers(0, 3, x.shape[1]).astype(np.int32)
    gpu, ref = make_pair(sp, x, box, 3, 300.0, 0.25, 1.0, 0, _net(rc))
    _compare(gpu, ref)
    spread_beads(gpu, ref, scale=0.2)
    rp, col = _compare(gpu, ref)
    assert rp[-1] > 0


@pytest.mark.parametrize("name", ["fad_p8", "water64", "ice512"])
def test_workloads_bit_exact(cuda_device, name):
    w = pi.make_workload(name)
    gpu, ref = pair_from_workload(w)
    _compare(gpu, ref)
    spread_beads(gpu, ref, scale=0.05)
    rp, _ = _compare(gpu, ref)
    assert abs(rp[-1] / w.rows - {"fad_p8": 8.8, "water64": 89.6, "ice512": 85.0}[name]) < 2.5


def test_replicas_bit_exact(cuda_device):
    w = pi.make_workload("fad_x64_p32")
    gpu, ref = pair_from_workload(w)
    spread_beads(gpu, ref, scale=0.1)
    _compare(gpu, ref)


def test_water4096_bit_exact(cuda_device):
    w = pi.make_workload("water4096")
    gpu, ref = pair_from_workload(w)
    spread_beads(gpu, ref, scale=0.05)
    rp, _ = _compare(gpu, ref)
    assert rp[-1] > 30_000_000


def test_empty_rows_and_single_atom(cuda_device):
    x = np.array([[[0, 0, 0], [100.0, 0, 0], [0.5, 0, 0]]])
    gpu, ref = make_pair(np.array([0, 1, 2], np.int32), x, np.zeros(3), 2, 300.0, 0.25, 1.0, 0, _net(2.0))
    rp, col = _compare(gpu, ref)
    assert list(np.diff(rp)) == [1, 0, 1, 1, 0, 1]
    gpu, ref = make_pair(np.array([1], np.int32), x[:, :1], np.zeros(3), 2, 300.0, 0.25, 1.0, 0, _net(2.0))
    rp, col = _compare(gpu, ref)
    assert rp[-1] == 0


def test_pair_capacity_overflow_is_reported(cuda_device):
    import paper_2503_23728_b200 as pb
    # dense blob: every atom sees > 2*expected+32 neighbours in a periodic box with a void
    rng = np.random.default_rng(0)
    N = 600
    x = rng.uniform(0, 3.0, (1, N, 3))
    box = np.full(3, 40.0)
    gpu = pb.PIMD(rng.integers(0, 3, N).astype(np.int32), pi.MASSES_AMU, x, box, 1, 300.0, 0.25, 1.0, 0, _net(5.0))
    with pytest.raises(pb.PimdError) as e:
        gpu.nlist()
    assert e.value.code == -3


def test_crowded_cells_bit_exact(cuda_device):
    """More atoms in a cell than the count kernel stages in shared memory (128): the rest of the home atoms is read from
    global memory and counted through global counters.  Two cells per axis, each 1.49 r_c wide, about 135 atoms per cell."""
    rng = np.random.default_rng(77)
    rc = 2.0
    box = np.array([5.97, 5.9, 5.99])
    x = rng.uniform(0, 1, (1, 1080, 3)) * box
    sp = rng.integers(0, 3, x.shape[1]).astype(np.int32)
    gpu, ref = make_pair(sp, x, box, 2, 300.0, 0.25, 1.0, 0, _net(rc))
    spread_beads(gpu, ref, scale=0.05)
    rp, _ = _compare(gpu, ref)
    assert np.diff(rp).max() < 512 and np.diff(rp).mean() > 100


def test_list_reuse_gives_the_same_lists_and_forces(cuda_device):
    """candidate lists within r_cut + skin are kept until an atom has moved by skin/2; the exact list is filtered
    from them every step.  Over 60 steps (with several rebuilds) the exported CSR equals the oracle's list at the same positions,
    and a run with skin = 0 (cell-list pass every step) gives bitwise the same trajectory."""
    w = pi.make_workload("water64")
    w.P = 4
    a = pb.PIMD.from_workload(w, device="cuda:0")
    b = pb.PIMD.from_workload(w, device="cuda:0")
    a.set_nlist_skin(0.2)          # water64: box 12.42 A allows r_cut + skin <= 6.21
    b.set_nlist_skin(0.0)
    ref = oracle.RefPIMD.from_workload(w)
    for it in range(6):
        a.step(10); b.step(10)
        qa, pa, _ = a.get_state(); qb, pb_, _ = b.get_state()
        assert torch.equal(qa, qb) and torch.equal(pa, pb_)                    # same forces, bit for bit
        ref.set_state(qa.cpu().numpy(), pa.cpu().numpy(), 10 * (it + 1))
        rp, col = a.nlist()
        rr, cr = ref.nlist()
        assert np.array_equal(rp.cpu().numpy(), rr) and np.array_equal(col.cpu().numpy(), cr)
    na, nb = a.nlist_rebuilds(), b.nlist_rebuilds()
    assert nb >= 60 and 2 <= na < nb // 2, (na, nb)                            # reuse happened, and so did rebuilds


def test_skin_is_limited_by_the_box(cuda_device):
    w = pi.make_workload("water64")
    g = pb.PIMD.from_workload(w, device="cuda:0")
    with pytest.raises(pb.PimdError):
        g.set_nlist_skin(0.5)      # 2 (6 + 0.5) > 12.42
    g.set_nlist_skin(0.1)


def test_list_reuse_on_the_tensor_core_path_is_bitwise_the_direct_path(cuda_device):
    """On the tcgen05 configs both fill kernels (direct and filtered) also write the per-pair displacement and segment kind that
    the first pair pass streams (nlist_kernels.cu: store_pair_geometry): with and without list reuse the trajectory must be the
    same bit for bit, across rebuilds."""
    w = pi.make_workload("ice512")
    w.P = 2
    a = pb.PIMD.from_workload(w, device="cuda:0")
    b = pb.PIMD.from_workload(w, device="cuda:0")
    a.set_nlist_skin(0.5)
    b.set_nlist_skin(0.0)
    for it in range(3):
        a.step(8); b.step(8)
        qa, pa, _ = a.get_state(); qb, pb_, _ = b.get_state()
        assert torch.equal(qa, qb) and torch.equal(pa, pb_)
    na, nb = a.nlist_rebuilds(), b.nlist_rebuilds()
    assert nb >= 24 and 2 <= na < nb, (na, nb)
