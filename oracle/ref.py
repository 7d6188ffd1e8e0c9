"""ctypes front-end of oracle/pimd_oracle.c (TEST INFRASTRUCTURE).

Argument marshalling only; every number is produced by the C file.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

# libgomp's default active spin-wait is very slow on shared/cgroup-limited hosts (many short parallel regions)
os.environ.setdefault("OMP_WAIT_POLICY", "passive")

import numpy as np

from . import build as _build

KB_EV = 8.617333262145e-5
HBAR_EVFS = 0.658211956548
AMU_INTERNAL = 103.6426965268

_lib = None


class _NetParams(C.Structure):
    _fields_ = [
        ("kind", C.c_int32), ("n_species", C.c_int32), ("n_rbf", C.c_int32), ("hidden", C.c_int32),
        ("n_layers", C.c_int32),
        ("r_cut", C.c_double), ("agg_norm", C.c_double), ("force_scale", C.c_double), ("harmonic_omega", C.c_double),
        ("weights", C.POINTER(C.c_float)), ("n_weights", C.c_int64),
    ]


class _Estimators(C.Structure):
    _fields_ = [("k_prim", C.c_double), ("k_vir", C.c_double), ("k_cvir", C.c_double), ("v_pot", C.c_double),
                ("t_centroid", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, ip, u32p = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_uint32)
        L.ref_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.ref_normal3.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, dp]
        L.ref_nm_matrix.argtypes = [C.c_int, dp]
        for f in (L.ref_nlist_brute, L.ref_nlist_cell):
            f.argtypes = [C.c_int, dp, dp, C.c_double, ip, ip, C.c_int64]
            f.restype = C.c_int64
        L.ref_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, ip, dp, dp, dp, C.c_int, C.c_double,
                                 C.c_double, C.c_double, C.c_uint64, C.POINTER(_NetParams)]
        L.ref_destroy.argtypes = [C.c_void_p]
        L.ref_destroy.restype = None
        L.ref_step.argtypes = [C.c_void_p, C.c_int]
        L.ref_set_integrator.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.ref_metad_enable.argtypes = [C.c_void_p, C.c_int, ip, dp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int]
        L.ref_metad_cv.argtypes = [C.c_void_p, dp, dp]
        L.ref_metad_gaussians.argtypes = [C.c_void_p, C.c_int, dp, dp, C.c_int]
        L.ref_metad_bias.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.ref_metad_bias.restype = C.c_double
        L.ref_metad_deposit_now.argtypes = [C.c_void_p]
        for f in (L.ref_stage_fwd, L.ref_stage_inv, L.ref_stage_force, L.ref_stage_mom_to_bead):
            f.argtypes = [dp, dp, C.c_int]
            f.restype = None
        L.ref_forces.argtypes = [C.c_void_p, dp]
        L.ref_force_gross.argtypes = [C.c_void_p, dp]
        L.ref_get_state.argtypes = [C.c_void_p, dp, dp, C.POINTER(C.c_int64)]
        L.ref_set_state.argtypes = [C.c_void_p, dp, dp, C.c_int64]
        L.ref_nlist.argtypes = [C.c_void_p, ip, ip, C.c_int64, C.POINTER(C.c_int64), C.c_int]
        L.ref_estimators.argtypes = [C.c_void_p, C.POINTER(_Estimators)]
        L.ref_n_weights.argtypes = [C.c_int] * 4
        L.ref_n_weights.restype = C.c_int64
        L.ref_num_threads.restype = C.c_int
        L.ref_set_num_threads.argtypes = [C.c_int]
        L.ref_set_num_threads.restype = None
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def stage_map(name, v):
    """One of the oracle's four staging maps ('fwd' q->u, 'inv' u->q, 'force' f_q->f_u (also p_q->p_u), 'mom_to_bead' p_u->p_q)
    applied to a vector of P bead values."""
    v = np.ascontiguousarray(v, dtype=np.float64)
    out = np.zeros_like(v)
    getattr(lib(), "ref_stage_" + name)(_dp(v), _dp(out), int(v.size))
    return out


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def set_num_threads(n: int) -> None:
    """OpenMP threads of the oracle (bench.py's single-thread leg)."""
    lib().ref_set_num_threads(int(n))


def num_threads() -> int:
    return int(lib().ref_num_threads())


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().ref_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def normal3(seed, atom, sysmode, step, tag):
    o = np.zeros(3)
    lib().ref_normal3(int(seed), int(atom), int(sysmode), int(step), int(tag), _dp(o))
    return o


def nm_matrix(P: int) -> np.ndarray:
    """C[j, k]: bead j, mode k."""
    Cm = np.zeros((P, P))
    lib().ref_nm_matrix(P, _dp(Cm))
    return Cm


def _nlist(fn, q, box, r_cut, cap=None):
    q = np.ascontiguousarray(q, dtype=np.float64)
    N = q.shape[0]
    box = np.ascontiguousarray(box, dtype=np.float64)
    cap = int(cap if cap is not None else N * max(N - 1, 1) + 1)
    row_ptr = np.zeros(N + 1, np.int32)
    col = np.zeros(cap, np.int32)
    n = fn(N, _dp(q), _dp(box), float(np.float32(r_cut)), _ip(row_ptr), _ip(col), cap)
    if n < 0:
        raise RuntimeError("pair capacity exceeded")
    return row_ptr, col[:n].copy()


def nlist_brute(q, box, r_cut, cap=None):
    """Definition L1: O(N^2) minimum-image pairs with d^2 < r_c^2, rows ascending j."""
    return _nlist(lib().ref_nlist_brute, q, box, r_cut, cap)


def nlist_cell(q, box, r_cut, cap=None):
    """Cell list (L2, L4); must equal `nlist_brute`."""
    return _nlist(lib().ref_nlist_cell, q, box, r_cut, cap)


@dataclass
class RefNet:
    kind: int = 0
    n_species: int = 3
    n_rbf: int = 32
    hidden: int = 64
    n_layers: int = 2
    r_cut: float = 5.0
    agg_norm: float = 1.0
    force_scale: float = 1.0
    harmonic_omega: float = 0.0
    weights: np.ndarray | None = None

    @classmethod
    def from_spec(cls, spec):
        """Accepts a pimd_inputs.NetSpec (duck-typed; floats pass through fp32 like the C-ABI struct)."""
        return cls(spec.kind, spec.n_species, spec.n_rbf, spec.hidden, spec.n_layers, float(np.float32(spec.r_cut)),
                   float(np.float32(spec.agg_norm)), float(np.float32(spec.force_scale)), float(spec.harmonic_omega),
                   np.ascontiguousarray(spec.weights, dtype=np.float32))


class RefPIMD:
    """Oracle twin of the C-ABI context: create / step / forces / estimators / state / nlist."""

    def __init__(self, species, masses_amu, positions, box, P, T, dt, gamma, seed, net: RefNet):
        L = lib()
        self.species = np.ascontiguousarray(species, dtype=np.int32)
        self.masses = np.ascontiguousarray(masses_amu, dtype=np.float64)
        pos = np.ascontiguousarray(positions, dtype=np.float64)
        if pos.ndim == 2:
            pos = pos[None]
        self.R, self.N = int(pos.shape[0]), int(pos.shape[1])
        self.P = int(P)
        self.box = np.ascontiguousarray(box, dtype=np.float64)
        self.net = net
        w = net.weights if net.weights is not None else np.zeros(1, np.float32)
        self._w = np.ascontiguousarray(w, dtype=np.float32)
        np_ = _NetParams(net.kind, net.n_species, net.n_rbf, net.hidden, net.n_layers, net.r_cut, net.agg_norm,
                         net.force_scale, net.harmonic_omega, self._w.ctypes.data_as(C.POINTER(C.c_float)),
                         int(self._w.size if net.kind == 0 else 0))
        h = C.c_void_p()
        rc = L.ref_create(C.byref(h), self.N, self.R, _ip(self.species), _dp(self.masses), _dp(pos), _dp(self.box),
                          self.P, float(T), float(dt), float(gamma), int(seed), C.byref(np_))
        if rc != 0:
            raise ValueError(f"ref_create failed: {rc}")
        self._h = h
        self.shape = (self.R, self.P, self.N, 3)

    @classmethod
    def from_workload(cls, w):
        return cls(w.species, w.masses_amu, w.positions, w.box, w.P, w.T, w.dt, w.gamma, w.seed,
                   RefNet.from_spec(w.net))

    def close(self):
        if getattr(self, "_h", None):
            lib().ref_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    TRANSFORMS = {"normal_modes": 0, "staging": 1, "primitive": 2}
    THERMOSTATS = {"pile_l": 0, "pile_g": 1}

    def set_integrator(self, transform="normal_modes", thermostat="pile_l"):
        """SURVEY 8(f)4 variants; before the first step (redraws the initial momenta in the chosen representation)."""
        rc = lib().ref_set_integrator(self._h, self.TRANSFORMS[transform], self.THERMOSTATS[thermostat])
        if rc != 0:
            raise RuntimeError(f"ref_set_integrator failed: {rc}")

    # ---- well-tempered metadynamics ----
    def metad_enable(self, cv, sigma, height, bias_factor, deposit_every, max_gaussians=4096, atoms=None, f_species=None, Q=0.0):
        """cv 'dimer' (atoms = O1, H1, O2, O4, H2, O3) or 'debye' (f_species, Q); height in eV."""
        a = np.ascontiguousarray(atoms if atoms is not None else np.zeros(6), dtype=np.int32)
        f = np.ascontiguousarray(f_species if f_species is not None else np.zeros(16), dtype=np.float64)
        rc = lib().ref_metad_enable(self._h, {"dimer": 1, "debye": 2}[cv], _ip(a), _dp(f), float(Q), float(sigma), float(height),
                                    float(bias_factor), int(deposit_every), int(max_gaussians))
        if rc != 0:
            raise RuntimeError(f"ref_metad_enable failed: {rc}")

    def metad_cv(self):
        s = np.zeros(self.shape[:2]); g = np.zeros(self.shape)
        rc = lib().ref_metad_cv(self._h, _dp(s), _dp(g))
        if rc != 0:
            raise RuntimeError(f"ref_metad_cv failed: {rc}")
        return s, g

    def metad_gaussians(self, r=0, cap=65536):
        c = np.zeros(cap); h = np.zeros(cap)
        n = lib().ref_metad_gaussians(self._h, int(r), _dp(c), _dp(h), cap)
        return c[:n].copy(), h[:n].copy()

    def metad_bias(self, s, r=0):
        return lib().ref_metad_bias(self._h, int(r), float(s))

    def metad_deposit_now(self):
        rc = lib().ref_metad_deposit_now(self._h)
        if rc != 0:
            raise RuntimeError(f"ref_metad_deposit_now failed: {rc}")

    def step(self, n=1):
        rc = lib().ref_step(self._h, int(n))
        if rc != 0:
            raise RuntimeError(f"ref_step failed: {rc}")

    def forces(self):
        out = np.zeros(self.shape)
        rc = lib().ref_forces(self._h, _dp(out))
        if rc != 0:
            raise RuntimeError(f"ref_forces failed: {rc}")
        return out

    def force_gross(self):
        """[R][P][N]: force_scale * sum_j c_ij (sum_o |w_f2[o] SiLU(t_o)| + |b_f2|), the sum of the magnitudes of all
        terms added up into F_i -- the scale forward error bounds of F_i are stated against."""
        out = np.zeros(self.shape[:3])
        rc = lib().ref_force_gross(self._h, _dp(out))
        if rc != 0:
            raise RuntimeError(f"ref_force_gross failed: {rc}")
        return out

    def get_state(self):
        q, p = np.zeros(self.shape), np.zeros(self.shape)
        st = C.c_int64()
        lib().ref_get_state(self._h, _dp(q), _dp(p), C.byref(st))
        return q, p, int(st.value)

    def set_state(self, q, p, step):
        q = np.ascontiguousarray(q, dtype=np.float64).reshape(self.shape)
        p = np.ascontiguousarray(p, dtype=np.float64).reshape(self.shape)
        lib().ref_set_state(self._h, _dp(q), _dp(p), int(step))

    def nlist(self, brute=False, cap_per_row=None):
        rows = self.R * self.P * self.N
        cap = int(rows * (cap_per_row if cap_per_row else max(self.N - 1, 1)))
        row_ptr = np.zeros(rows + 1, np.int32)
        col = np.zeros(cap, np.int32)
        n = C.c_int64()
        rc = lib().ref_nlist(self._h, _ip(row_ptr), _ip(col), cap, C.byref(n), int(bool(brute)))
        if rc != 0:
            raise RuntimeError(f"ref_nlist failed: {rc}")
        return row_ptr, col[: n.value].copy()

    def estimators(self):
        out = (_Estimators * self.R)()
        rc = lib().ref_estimators(self._h, out)
        if rc != 0:
            raise RuntimeError(f"ref_estimators failed: {rc}")
        return np.array([[e.k_prim, e.k_vir, e.k_cvir, e.v_pot, e.t_centroid] for e in out])
