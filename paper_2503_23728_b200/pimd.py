"""ctypes binding of include/pimd.h (argument marshalling only; same names as the C-ABI)."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libpimd_b200.so")
_lib = None


class PimdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pimd error {code}: {msg}")
        self.code = code


class NetParams(C.Structure):
    """Mirror of `pimd_net_params`."""
    _fields_ = [
        ("kind", C.c_int32), ("n_species", C.c_int32), ("n_rbf", C.c_int32), ("hidden", C.c_int32),
        ("n_layers", C.c_int32), ("gemm_dtype", C.c_int32),
        ("r_cut", C.c_float), ("agg_norm", C.c_float), ("force_scale", C.c_float),
        ("harmonic_omega", C.c_double),
        ("weights", C.POINTER(C.c_float)), ("n_weights", C.c_int64),
    ]


class Estimators(C.Structure):
    """Mirror of `pimd_estimators_t`."""
    _fields_ = [("k_prim", C.c_double), ("k_vir", C.c_double), ("k_cvir", C.c_double), ("v_pot", C.c_double),
                ("t_centroid", C.c_double)]


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """Loads libpimd_b200.so (built in-tree by paper_2503_23728_b200/build.py).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2503_23728_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32)
    L.pimd_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, dp, C.POINTER(NetParams), C.POINTER(C.c_size_t)]
    L.pimd_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, ip, dp, dp, dp, C.c_int, C.c_double, C.c_double,
                              C.c_double, C.c_uint64, C.POINTER(NetParams), vp, C.c_size_t, vp]
    L.pimd_step.argtypes = [vp, C.c_int]
    L.pimd_set_integrator.argtypes = [vp, C.c_int, C.c_int]
    L.pimd_metad_enable.argtypes = [vp, C.c_int, ip, dp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int]
    L.pimd_metad_cv.argtypes = [vp, vp, vp]
    L.pimd_metad_gaussians.argtypes = [vp, C.c_int, dp, dp, C.c_int, C.POINTER(C.c_int)]
    L.pimd_metad_deposit_now.argtypes = [vp]
    L.pimd_debye_cv_static.argtypes = [vp, vp, C.c_int, C.c_int, dp, dp, C.c_int, C.c_double, vp, vp, vp]
    L.pimd_set_nlist_skin.argtypes = [vp, C.c_double]
    L.pimd_nlist_rebuilds.argtypes = [vp, C.POINTER(C.c_int64)]
    L.pimd_forces.argtypes = [vp, vp]
    L.pimd_estimators.argtypes = [vp, C.POINTER(Estimators)]
    L.pimd_get_state.argtypes = [vp, vp, vp, C.POINTER(C.c_int64)]
    L.pimd_set_state.argtypes = [vp, vp, vp, C.c_int64]
    L.pimd_get_forces_cached.argtypes = [vp, vp]
    L.pimd_set_forces_cached.argtypes = [vp, vp]
    L.pimd_nlist.argtypes = [vp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
    L.pimd_sync.argtypes = [vp]
    L.pimd_profile.argtypes = [vp, C.c_int]
    L.pimd_profile_read.argtypes = [vp, dp, C.POINTER(C.c_int64)]
    L.pimd_measure_fp32_fma_tflops.argtypes = [vp, dp]
    L.pimd_launch_count.argtypes = [vp]
    L.pimd_launch_count.restype = C.c_int64
    L.pimd_last_error.restype = C.c_char_p
    L.pimd_destroy.argtypes = [vp]
    L.pimd_destroy.restype = None
    _lib = L
    return L


def measure_fp32_fma_tflops(stream=None) -> float:
    """Measured FP32 FMA rate of the current CUDA device (TFLOP/s); see include/pimd.h."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    v = C.c_double()
    _check(load_library().pimd_measure_fp32_fma_tflops(C.c_void_p(st.cuda_stream), C.byref(v)))
    return float(v.value)


def debye_cv_static(q, species, box, f_species, Q, s_out, grad_out=None, stream=None):
    """pimd_debye_cv_static (include/pimd.h): the Debye CV of every bead-system in q [n_systems][N][3] (float64 device tensor) into
    s_out [n_systems] (and grad_out, same shape as q), with no device allocation inside the library.  species: int32 device tensor."""
    import torch
    assert q.dtype == torch.float64 and q.is_contiguous() and q.dim() == 3 and q.shape[2] == 3
    assert species.dtype == torch.int32 and species.is_contiguous() and species.numel() == q.shape[1]
    assert s_out.dtype == torch.float64 and s_out.is_contiguous() and s_out.numel() == q.shape[0]
    if grad_out is not None:
        assert grad_out.dtype == torch.float64 and grad_out.is_contiguous() and grad_out.shape == q.shape
    b = np.ascontiguousarray(box, dtype=np.float64)
    f = np.ascontiguousarray(f_species, dtype=np.float64)
    st = stream if stream is not None else torch.cuda.current_stream(q.device)
    with torch.cuda.device(q.device):
        _check(load_library().pimd_debye_cv_static(
            C.c_void_p(q.data_ptr()), C.c_void_p(species.data_ptr()), int(q.shape[1]), int(q.shape[0]),
            b.ctypes.data_as(C.POINTER(C.c_double)), f.ctypes.data_as(C.POINTER(C.c_double)), int(f.size), float(Q),
            C.c_void_p(s_out.data_ptr()), C.c_void_p(grad_out.data_ptr() if grad_out is not None else None), C.c_void_p(st.cuda_stream)))


def _check(rc):
    if rc != 0:
        raise PimdError(rc, load_library().pimd_last_error().decode())


def _net_struct(net, keep):
    """net: any object with the NetSpec fields (duck-typed)."""
    w = np.ascontiguousarray(net.weights if net.weights is not None else np.zeros(0), dtype=np.float32)
    keep.append(w)
    return NetParams(int(net.kind), int(net.n_species), int(net.n_rbf), int(net.hidden), int(net.n_layers),
                     int(getattr(net, "gemm_dtype", 0)), float(net.r_cut), float(net.agg_norm),
                     float(net.force_scale), float(net.harmonic_omega),
                     w.ctypes.data_as(C.POINTER(C.c_float)), int(w.size if int(net.kind) == 0 else 0))


class PIMD:
    """Owns the torch workspace tensor and the `pimd_ctx*`; methods are the C-ABI calls."""

    def __init__(self, species, masses_amu, positions, box, P, T, dt, gamma, seed, net, device="cuda:0",
                 stream=None):
        import torch

        L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_23728_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        species = np.ascontiguousarray(species, dtype=np.int32)
        masses = np.ascontiguousarray(masses_amu, dtype=np.float64)
        pos = np.ascontiguousarray(positions, dtype=np.float64)
        if pos.ndim == 2:
            pos = pos[None]
        box = np.ascontiguousarray(box, dtype=np.float64)
        self.R, self.N, self.P = int(pos.shape[0]), int(pos.shape[1]), int(P)
        self.rows = self.R * self.P * self.N
        self.shape = (self.R, self.P, self.N, 3)
        self._keep = []
        npar = _net_struct(net, self._keep)
        self.kind = int(net.kind)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        nbytes = C.c_size_t()
        _check(L.pimd_workspace_bytes(self.N, self.R, self.P, box.ctypes.data_as(dp), C.byref(npar), C.byref(nbytes)))
        self.workspace_bytes = int(nbytes.value)
        self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        _check(L.pimd_create(C.byref(h), self.N, self.R, species.ctypes.data_as(ip), masses.ctypes.data_as(dp),
                             pos.ctypes.data_as(dp), box.ctypes.data_as(dp), self.P, float(T), float(dt), float(gamma),
                             int(seed), C.byref(npar), C.c_void_p(self._ws_ptr), self.workspace_bytes,
                             C.c_void_p(self.stream.cuda_stream)))
        self._h = h

    @classmethod
    def from_workload(cls, w, **kw):
        return cls(w.species, w.masses_amu, w.positions, w.box, w.P, w.T, w.dt, w.gamma, w.seed, w.net, **kw)

    def close(self):
        if getattr(self, "_h", None):
            load_library().pimd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- C-ABI calls -------------------------------------------------------------------------
    TRANSFORMS = {"normal_modes": 0, "staging": 1, "primitive": 2}
    THERMOSTATS = {"pile_l": 0, "pile_g": 1}

    def set_integrator(self, transform="normal_modes", thermostat="pile_l"):
        """Integrator variant (before the first step): normal-mode / staging / primitive, PILE-L / PILE-G."""
        _check(load_library().pimd_set_integrator(self._h, self.TRANSFORMS[transform], self.THERMOSTATS[thermostat]))

    def set_nlist_skin(self, skin):
        """Verlet skin (A) of the reusable candidate lists; 0 = cell-list pass every step.  Results do not depend on it."""
        _check(load_library().pimd_set_nlist_skin(self._h, float(skin)))

    def metad_enable(self, cv, sigma, height, bias_factor, deposit_every, atoms=None, f_species=None, Q=0.0):
        """Well-tempered metadynamics: cv 'dimer' (atoms = O1, H1, O2, O4, H2, O3) or 'debye' (f_species, Q); height in eV."""
        a = np.ascontiguousarray(atoms if atoms is not None else np.zeros(6), dtype=np.int32)
        f = np.ascontiguousarray(f_species if f_species is not None else np.zeros(16), dtype=np.float64)
        self._keep += [a, f]
        _check(load_library().pimd_metad_enable(self._h, {"dimer": 1, "debye": 2}[cv], a.ctypes.data_as(C.POINTER(C.c_int32)),
                                                f.ctypes.data_as(C.POINTER(C.c_double)), float(Q), float(sigma), float(height),
                                                float(bias_factor), int(deposit_every)))

    def metad_cv(self):
        t = self._torch
        s = t.empty(self.shape[:2], dtype=t.float64, device=self.device)
        g = t.empty(self.shape, dtype=t.float64, device=self.device)
        _check(load_library().pimd_metad_cv(self._h, C.c_void_p(s.data_ptr()), C.c_void_p(g.data_ptr())))
        return s, g

    def metad_gaussians(self, r=0, cap=16384):
        c = np.zeros(cap); h = np.zeros(cap); n = C.c_int()
        _check(load_library().pimd_metad_gaussians(self._h, int(r), c.ctypes.data_as(C.POINTER(C.c_double)),
                                                   h.ctypes.data_as(C.POINTER(C.c_double)), cap, C.byref(n)))
        return c[: n.value].copy(), h[: n.value].copy()

    def metad_deposit_now(self):
        _check(load_library().pimd_metad_deposit_now(self._h))

    def nlist_rebuilds(self):
        n = C.c_int64()
        _check(load_library().pimd_nlist_rebuilds(self._h, C.byref(n)))
        return int(n.value)

    def step(self, n=1):
        _check(load_library().pimd_step(self._h, int(n)))

    def forces(self, out=None):
        t = self._torch
        if out is None:
            out = t.empty(self.shape, dtype=t.float32, device=self.device)
        _check(load_library().pimd_forces(self._h, C.c_void_p(out.data_ptr())))
        return out

    def estimators(self):
        out = (Estimators * self.R)()
        _check(load_library().pimd_estimators(self._h, out))
        return np.array([[e.k_prim, e.k_vir, e.k_cvir, e.v_pot, e.t_centroid] for e in out])

    def get_state(self):
        t = self._torch
        q = t.empty(self.shape, dtype=t.float64, device=self.device)
        p = t.empty(self.shape, dtype=t.float64, device=self.device)
        st = C.c_int64()
        _check(load_library().pimd_get_state(self._h, C.c_void_p(q.data_ptr()), C.c_void_p(p.data_ptr()), C.byref(st)))
        return q, p, int(st.value)

    def set_state(self, q, p, step):
        t = self._torch
        q = t.as_tensor(q, dtype=t.float64, device=self.device).contiguous()
        p = t.as_tensor(p, dtype=t.float64, device=self.device).contiguous()
        assert q.numel() == self.rows * 3 and p.numel() == self.rows * 3
        _check(load_library().pimd_set_state(self._h, C.c_void_p(q.data_ptr()), C.c_void_p(p.data_ptr()), int(step)))
        self.sync()  # q, p temporaries may be freed by the caller right after

    def get_forces_cached(self, out=None):
        t = self._torch
        if out is None:
            out = t.empty(self.shape, dtype=t.float64, device=self.device)
        _check(load_library().pimd_get_forces_cached(self._h, C.c_void_p(out.data_ptr())))
        return out

    def set_forces_cached(self, F):
        assert F.dtype == self._torch.float64 and F.is_contiguous() and F.numel() == self.rows * 3
        _check(load_library().pimd_set_forces_cached(self._h, C.c_void_p(F.data_ptr())))

    def set_state_async(self, q, p, step):
        """pimd_set_state without the synchronisation: q, p must be contiguous float64 device tensors that outlive the call."""
        _check(load_library().pimd_set_state(self._h, C.c_void_p(q.data_ptr()), C.c_void_p(p.data_ptr()), int(step)))

    def nlist(self, cap_per_row=None):
        t = self._torch
        cap = int(self.rows * (cap_per_row if cap_per_row else min(max(self.N - 1, 1), 512)))
        row_ptr = t.empty(self.rows + 1, dtype=t.int32, device=self.device)
        col = t.empty(max(cap, 1), dtype=t.int32, device=self.device)
        n = C.c_int64()
        _check(load_library().pimd_nlist(self._h, C.c_void_p(row_ptr.data_ptr()), C.c_void_p(col.data_ptr()), cap,
                                         C.byref(n)))
        return row_ptr, col[: n.value]

    def sync(self):
        _check(load_library().pimd_sync(self._h))

    PROF_CLASSES = ("pimd_nm", "nlist", "gfn.pair", "gfn.node", "gfn.head", "other")

    def profile(self, enable: bool):
        _check(load_library().pimd_profile(self._h, int(bool(enable))))

    def profile_read(self):
        """{class: (total_ms, timed_launch_groups)} measured with CUDA events on the context's stream."""
        ms = (C.c_double * 6)()
        n = (C.c_int64 * 6)()
        _check(load_library().pimd_profile_read(self._h, ms, n))
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(self.PROF_CLASSES)}

    def launch_count(self) -> int:
        return int(load_library().pimd_launch_count(self._h))
