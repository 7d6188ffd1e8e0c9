"""Geometry, weight-blob and run-parameter generators for BASELINE.json `configs[0..4]`.

Recipes follow SURVEY.md §8(d) D1-D3 and §8(c) G0/G6.  Everything is seeded
(`numpy.random.default_rng`) and synthetic.  No arithmetic of the PIMD method
lives here (see package docstring).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# type indices ascending in Z
SPECIES_H, SPECIES_C, SPECIES_O = 0, 1, 2
# BASELINE.json configs[0]: masses C 12.011, H 1.008, O 15.999
MASSES_AMU = np.array([1.008, 12.011, 15.999], dtype=np.float64)


# --------------------------------------------------------------------------
# weight blob
# --------------------------------------------------------------------------
def weight_layout(S: int, K: int, H: int, L: int):
    """[(name, shape)] in packing order; matrices are row-major [out][in]."""
    lay = [("Emb", (S, H)), ("W_e1", (H, K)), ("b_e1", (H,)), ("W_e2", (H, H)), ("b_e2", (H,))]
    for l in range(L):
        lay += [
            (f"W_s.{l}", (H, H)),
            (f"W_vn.{l}", (H, H)),
            (f"W_vm.{l}", (H, H)),
            (f"b_v1.{l}", (H,)),
            (f"W_v2.{l}", (H, H)),
            (f"b_v2.{l}", (H,)),
            (f"W_a.{l}", (H, H)),
            (f"b_a.{l}", (H,)),
        ]
    lay += [("W_f1", (H, H)), ("b_f1", (H,)), ("w_f2", (H,)), ("b_f2", (1,))]
    return lay


def n_weights(S: int, K: int, H: int, L: int) -> int:
    return int(sum(int(np.prod(s)) for _, s in weight_layout(S, K, H, L)))


def pack_weights(seed: int, S: int, K: int, H: int, L: int, bias_scale: float = 0.0) -> np.ndarray:
    """Xavier-normal random-init weights (BASELINE configs[0]), fp32 blob.

    Draws are taken in packing order in fp64 and cast to fp32.  Embeddings are
    unit normal; biases are `bias_scale` x unit normal (0 for the named
    workloads; tests pass a non-zero value so that bias terms are exercised).
    """
    rng = np.random.default_rng(seed)
    parts = []
    for name, shape in weight_layout(S, K, H, L):
        if name == "Emb":
            w = rng.standard_normal(shape)
        elif name.startswith("b_"):
            w = bias_scale * rng.standard_normal(shape) if bias_scale != 0.0 else np.zeros(shape)
        elif name == "w_f2":
            w = rng.standard_normal(shape) * np.sqrt(2.0 / (shape[0] + 1))
        else:
            fan_out, fan_in = shape
            w = rng.standard_normal(shape) * np.sqrt(2.0 / (fan_in + fan_out))
        parts.append(np.asarray(w, dtype=np.float64).ravel())
    return np.concatenate(parts).astype(np.float32)


# --------------------------------------------------------------------------
# geometries
# --------------------------------------------------------------------------
def _fad_monomer():
    """Planar HCOOH from internal coordinates; C at origin, O-C-O bisector along +x.

    Order: C, H(formyl), O(carbonyl), O(hydroxyl), H(hydroxyl).
    """
    half = np.deg2rad(125.0 / 2.0)
    c = np.zeros(3)
    o_c = 1.22 * np.array([np.cos(half), np.sin(half), 0.0])
    o_h = 1.32 * np.array([np.cos(half), -np.sin(half), 0.0])
    h_f = 1.10 * np.array([-1.0, 0.0, 0.0])
    # hydroxyl H: |O-H| = 0.98, angle C-O-H = 108 deg, in plane, the rotamer with the larger x
    to_c = (c - o_h) / np.linalg.norm(c - o_h)
    ang = np.deg2rad(108.0)
    cands = []
    for sgn in (+1.0, -1.0):
        ca, sa = np.cos(sgn * ang), np.sin(sgn * ang)
        d = np.array([ca * to_c[0] - sa * to_c[1], sa * to_c[0] + ca * to_c[1], 0.0])
        cands.append(o_h + 0.98 * d)
    h_o = max(cands, key=lambda v: v[0])
    return np.stack([c, h_f, o_c, o_h, h_o])


def fad_geometry(seed: int, jitter: float = 0.05) -> np.ndarray:
    """Cyclic doubly H-bonded formic-acid dimer, O...O = 2.70 A, + Gaussian jitter (D1)."""
    mono = _fad_monomer()

    def oo_dist(x0):
        second = 2.0 * np.array([x0, 0.0, 0.0]) - mono
        return np.linalg.norm(mono[3] - second[2])

    lo, hi = 1.0, 4.0  # oo_dist is increasing on this bracket
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if oo_dist(mid) < 2.70:
            lo = mid
        else:
            hi = mid
    x0 = 0.5 * (lo + hi)
    pos = np.concatenate([mono, 2.0 * np.array([x0, 0.0, 0.0]) - mono])
    rng = np.random.default_rng(seed)
    return pos + jitter * rng.standard_normal((10, 3))


FAD_SPECIES = np.array([SPECIES_C, SPECIES_H, SPECIES_O, SPECIES_O, SPECIES_H] * 2, dtype=np.int32)


def _min_image(d, box):
    return d - box * np.round(d / box)


def water_geometry(n_mol: int, box: float, seed: int, oo_min: float = 2.5) -> np.ndarray:
    """Liquid-like water: random sequential insertion of O, random rigid orientation (D2).

    Atom order O, H, H per molecule.  Only the O-O distance criterion is applied.
    """
    rng = np.random.default_rng(seed)
    placed = np.empty((n_mol, 3))
    n = 0
    while n < n_mol:
        cand = rng.uniform(0.0, box, size=(1024, 3))
        for c in cand:
            if n:
                d = _min_image(placed[:n] - c, box)
                if np.min(np.einsum("ij,ij->i", d, d)) < oo_min * oo_min:
                    continue
            placed[n] = c
            n += 1
            if n == n_mol:
                break
    quat = rng.standard_normal((n_mol, 4))
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    w, x, y, z = quat.T
    rot = np.empty((n_mol, 3, 3))
    rot[:, 0, 0] = 1 - 2 * (y * y + z * z)
    rot[:, 0, 1] = 2 * (x * y - z * w)
    rot[:, 0, 2] = 2 * (x * z + y * w)
    rot[:, 1, 0] = 2 * (x * y + z * w)
    rot[:, 1, 1] = 1 - 2 * (x * x + z * z)
    rot[:, 1, 2] = 2 * (y * z - x * w)
    rot[:, 2, 0] = 2 * (x * z - y * w)
    rot[:, 2, 1] = 2 * (y * z + x * w)
    rot[:, 2, 2] = 1 - 2 * (x * x + y * y)
    half = np.deg2rad(104.5 / 2.0)
    h1 = 0.96 * np.array([np.sin(half), np.cos(half), 0.0])
    h2 = 0.96 * np.array([-np.sin(half), np.cos(half), 0.0])
    pos = np.empty((n_mol, 3, 3))
    pos[:, 0] = placed
    pos[:, 1] = placed + rot @ h1
    pos[:, 2] = placed + rot @ h2
    return pos.reshape(3 * n_mol, 3)


def ice_ic_geometry(n_cells: int = 4, a: float = 6.35, seed: int = 2, oh: float = 0.96) -> np.ndarray:
    """Cubic ice Ic: O on a diamond lattice, two H per O along seeded-random bonds (D3)."""
    fcc = np.array([[0, 0, 0], [0, 0.5, 0.5], [0.5, 0, 0.5], [0.5, 0.5, 0]], dtype=np.float64)
    basis = np.concatenate([fcc, fcc + 0.25])  # sub-lattice A then B
    sub = np.array([0, 0, 0, 0, 1, 1, 1, 1])
    dirs = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=np.float64) / np.sqrt(3.0)
    rng = np.random.default_rng(seed)
    out = []
    for ix in range(n_cells):
        for iy in range(n_cells):
            for iz in range(n_cells):
                for b in range(8):
                    o = (basis[b] + np.array([ix, iy, iz])) * a
                    sign = 1.0 if sub[b] == 0 else -1.0
                    pick = rng.choice(4, size=2, replace=False)
                    out.append(o)
                    out.append(o + oh * sign * dirs[pick[0]])
                    out.append(o + oh * sign * dirs[pick[1]])
    return np.array(out)


def water_species(n_mol: int) -> np.ndarray:
    return np.array([SPECIES_O, SPECIES_H, SPECIES_H] * n_mol, dtype=np.int32)


# --------------------------------------------------------------------------
# workloads
# --------------------------------------------------------------------------
@dataclass
class NetSpec:
    kind: int = 0  # 0 GFN, 1 harmonic well, 2 free ring polymer
    n_species: int = 3
    n_rbf: int = 32
    hidden: int = 64
    n_layers: int = 2
    gemm_dtype: int = 0  # 0 fp32, 1 bf16 inputs + fp32 accumulate
    r_cut: float = 5.0
    agg_norm: float = 1.0 / 9.0
    force_scale: float = 0.25
    harmonic_omega: float = 0.0  # rad/fs, kind 1
    weights: np.ndarray = field(default_factory=lambda: np.zeros(0, np.float32))


@dataclass
class Workload:
    name: str
    species: np.ndarray  # int32 [N]
    masses_amu: np.ndarray  # f64 [S]
    positions: np.ndarray  # f64 [R][N][3]
    box: np.ndarray  # f64 [3]; zeros = non-periodic
    P: int
    T: float
    dt: float
    gamma: float  # ps^-1, centroid friction; <0 = NVE
    seed: int  # Philox key
    net: NetSpec
    n_steps: int

    @property
    def n_atoms(self) -> int:
        return int(self.species.shape[0])

    @property
    def n_replicas(self) -> int:
        return int(self.positions.shape[0])

    @property
    def rows(self) -> int:
        return self.n_replicas * self.P * self.n_atoms


def workload_names():
    return ["fad_p8", "fad_x64_p32", "water64", "ice512", "water4096"]


def _gfn(K, H, L, r_cut, agg, fscale, wseed, gemm_dtype=0):
    return NetSpec(0, 3, K, H, L, gemm_dtype, r_cut, agg, fscale, 0.0, pack_weights(wseed, 3, K, H, L))


def make_workload(name: str) -> Workload:
    """BASELINE.json configs[0..4] by name (see `workload_names`)."""
    if name == "fad_p8":  # configs[0]
        pos = fad_geometry(0)[None]
        return Workload(name, FAD_SPECIES.copy(), MASSES_AMU.copy(), pos, np.zeros(3), 8, 300.0, 0.25, 1.0, 0,
                        _gfn(32, 64, 2, 5.0, 1.0 / 9.0, 0.25, 0), 200)
    if name == "fad_x64_p32":  # configs[1]
        pos = np.stack([fad_geometry(r) for r in range(64)])
        return Workload(name, FAD_SPECIES.copy(), MASSES_AMU.copy(), pos, np.zeros(3), 32, 300.0, 0.25, 1.0, 0,
                        _gfn(32, 64, 2, 5.0, 1.0 / 9.0, 0.25, 0), 1000)
    if name == "water64":  # configs[2]
        pos = water_geometry(64, 12.42, 1)[None]
        return Workload(name, water_species(64), MASSES_AMU.copy(), pos, np.full(3, 12.42), 32, 300.0, 0.25, 1.0, 0,
                        _gfn(64, 128, 3, 6.0, 1.0 / 90.0, 0.1, 1), 200)
    if name == "ice512":  # configs[3], headline
        pos = ice_ic_geometry(4, 6.35, 2)[None]
        return Workload(name, water_species(512), MASSES_AMU.copy(), pos, np.full(3, 25.4), 32, 250.0, 0.25, 1.0, 0,
                        _gfn(64, 128, 3, 6.0, 1.0 / 90.0, 0.1, 1, gemm_dtype=1), 200)
    if name == "water4096":  # configs[4]
        pos = water_geometry(4096, 49.66, 3)[None]
        return Workload(name, water_species(4096), MASSES_AMU.copy(), pos, np.full(3, 49.66), 32, 300.0, 0.25, 1.0, 0,
                        _gfn(64, 128, 3, 6.0, 1.0 / 90.0, 0.1, 1, gemm_dtype=1), 200)
    raise KeyError(name)
