"""Pins for the oracle's neighbour list: cell list == brute-force definition,
symmetry, closed-form ice-Ic shell counts, boundary cases."""
import os

import numpy as np
import pytest

import oracle
import pimd_inputs as pi

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def numpy_pairs(x, box, rc):
    """L1 definition written with dense numpy (round half away from zero like C round())."""
    d = x[None, :, :] - x[:, None, :]
    if box[0] > 0:
        t = d / box
        d = d - box * (np.sign(t) * np.floor(np.abs(t) + 0.5))
    r2 = (d[..., 0] * d[..., 0] + d[..., 1] * d[..., 1]) + d[..., 2] * d[..., 2]
    m = (r2 < rc * rc) & ~np.eye(len(x), dtype=bool)
    return [np.nonzero(m[i])[0] for i in range(len(x))]


def rows(row_ptr, col):
    return [col[row_ptr[i]:row_ptr[i + 1]] for i in range(len(row_ptr) - 1)]


@pytest.mark.parametrize("ncell", [0, 2, 3, 4, 5])
def test_cell_equals_brute_and_definition(ncell):
    rng = np.random.default_rng(ncell)
    rc = 2.0
    if ncell == 0:
        box = np.zeros(3); x = rng.uniform(0, 5, (40, 3))
    else:
        box = np.array([ncell * rc + 0.3, ncell * rc + 0.9, ncell * rc + 0.01])
        x = rng.uniform(0, 1, (60 * ncell, 3)) * box
        x[::7] += box * rng.integers(-3, 4, (len(x[::7]), 3))  # unwrapped atoms, whole box vectors away
        x[1] = [0.0, 0.0, 0.0]  # on the box corner
        x[2] = [rc, 2 * rc, box[2]]  # on cell faces / the far boundary
        x[3] = x[1] + [rc, 0, 0]  # exactly at the cutoff from atom 1: strict '<' excludes it
        x[4] = [-1e-300, box[1] * (1 - 1e-17), 0.5]  # wrapped fraction rounds to 1.0 -> clamped to last cell
    rb, cb = oracle.nlist_brute(x, box, rc)
    rcell, ccell = oracle.nlist_cell(x, box, rc)
    assert np.array_equal(rb, rcell) and np.array_equal(cb, ccell)
    want = numpy_pairs(x, box, rc)
    got = rows(rb, cb)
    for i in range(len(x)):
        assert np.array_equal(got[i], want[i])
    if ncell:
        assert 3 not in got[1] and 1 not in got[3]
    # symmetry
    s = {(i, int(j)) for i in range(len(x)) for j in got[i]}
    assert all((j, i) in s for (i, j) in s)


def test_image_shift_invariance_of_list():
    rng = np.random.default_rng(9)
    box = np.array([8.0, 9.0, 10.0]); rc = 3.0
    x = rng.uniform(0, 1, (80, 3)) * box
    r0, c0 = oracle.nlist_cell(x, box, rc)
    y = x.copy(); y[5] += [box[0], -2 * box[1], 0]; y[17] -= [0, 0, 3 * box[2]]
    r1, c1 = oracle.nlist_cell(y, box, rc)
    # images shifted by exact box multiples: rounding of x/L may differ in the last bit only for pairs
    # at the cutoff, none here
    assert np.array_equal(r0, r1) and np.array_equal(c0, c1)


def test_ice_ic_shell_counts():
    a = 6.35
    O = pi.ice_ic_geometry(4, a, 2)[::3]
    box = np.full(3, 4 * a)
    shells = [tuple(map(float, l.split())) for l in open(os.path.join(GOLD, "ice_ic_shells.txt"))
              if l.strip() and not l.startswith("#")]
    cum = 0
    for dist, cnt in shells:
        cum += int(cnt)
        rc = dist * a + 0.01
        if 2 * rc > box[0]:
            break
        rp, col = oracle.nlist_cell(O, box, rc)
        assert np.all(np.diff(rp) == cum), (dist, cum)
    rp, col = oracle.nlist_cell(O, box, 6.0)
    assert np.all(np.diff(rp) == 28)  # 4 + 12 + 12 oxygens within 6 A


@pytest.mark.parametrize("name,mean,lo,hi", [("fad_p8", 8.8, 7, 9), ("water64", 89.6, 70, 105), ("ice512", 85.0, 77, 92)])
def test_workload_pair_counts(name, mean, lo, hi):
    w = pi.make_workload(name)
    rp, col = oracle.nlist_cell(w.positions[0], w.box, w.net.r_cut)
    cnt = np.diff(rp)
    assert abs(cnt.mean() - mean) < 0.2 and cnt.min() >= lo and cnt.max() <= hi
    if w.box[0] > 0:  # ideal-gas estimate rho * 4/3 pi rc^3 within 10 %
        est = w.n_atoms / np.prod(w.box) * 4 / 3 * np.pi * w.net.r_cut ** 3
        assert abs(cnt.mean() - est) / est < 0.1


def test_context_nlist_matches_per_system_lists():
    w = pi.make_workload("fad_p8")
    sim = oracle.RefPIMD.from_workload(w)
    sim.step(3)  # beads spread a little
    q, _, _ = sim.get_state()
    rp, col = sim.nlist()
    rpb, colb = sim.nlist(brute=True)
    assert np.array_equal(rp, rpb) and np.array_equal(col, colb)
    N = w.n_atoms
    for s in range(w.P):
        r1, c1 = oracle.nlist_brute(q[0, s], w.box, w.net.r_cut)
        assert np.array_equal(rp[s * N:(s + 1) * N + 1] - rp[s * N], r1)
        assert np.array_equal(col[rp[s * N]:rp[(s + 1) * N]], c1)


def test_capacity_overflow_reported():
    x = np.random.default_rng(0).uniform(0, 3, (20, 3))
    with pytest.raises(RuntimeError):
        oracle.nlist_cell(x, np.zeros(3), 5.0, cap=10)


def test_skin_list_filtered_to_the_cutoff_equals_the_exact_list():
    """Neighbour-list reuse: candidates within r_c + skin at reference positions, filtered with the exact predicate at
    the current positions, give the exact list as long as no atom has moved by skin/2 or more (triangle inequality on the
    minimum-image distance); the oracle's brute-force list is the definition on both sides."""
    rng = np.random.default_rng(8)
    box = np.array([13.0, 12.5, 14.0])
    N, rc, skin = 150, 3.0, 0.6
    q_ref = rng.uniform(0, 1, (N, 3)) * box
    step = rng.standard_normal((N, 3))
    step *= (0.999 * skin / 2) / np.linalg.norm(step, axis=1).max()            # largest displacement just below skin/2
    q = q_ref + step
    rp_c, col_c = oracle.nlist_brute(q_ref, box, rc + skin)
    rp_x, col_x = oracle.nlist_brute(q, box, rc)
    rows, cols = [], []
    for i in range(N):
        cand = col_c[rp_c[i]:rp_c[i + 1]]
        d = q[cand] - q[i]
        d = d - box * np.round(d / box)
        keep = cand[(d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1]) + d[:, 2] * d[:, 2] < np.float64(np.float32(rc)) ** 2]
        rows.append(len(keep)); cols.append(keep)
    assert np.array_equal(np.concatenate([[0], np.cumsum(rows)]), rp_x)
    assert np.array_equal(np.concatenate(cols), col_x)
    # and a displacement beyond skin/2 can lose a pair: the rebuild criterion is needed
    q_far = q_ref + step * 4.0
    rp_f, col_f = oracle.nlist_brute(q_far, box, rc)
    lost = 0
    for i in range(N):
        lost += len(set(col_f[rp_f[i]:rp_f[i + 1]]) - set(col_c[rp_c[i]:rp_c[i + 1]]))
    assert lost > 0
