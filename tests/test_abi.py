"""CPU checks of the boundary: the C-ABI library loads and exports every symbol include/pimd.h declares."""
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import paper_2503_23728_b200.build as b
    b.build()
    import paper_2503_23728_b200 as pb
    return pb.load_library()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "pimd.h")).read()
    names = set(re.findall(r"\b(pimd_[a-z_]+)\s*\(", hdr))
    assert {"pimd_create", "pimd_step", "pimd_forces", "pimd_estimators", "pimd_nlist", "pimd_get_state",
            "pimd_set_state", "pimd_workspace_bytes", "pimd_destroy", "pimd_last_error"} <= names
    for n in names:
        assert hasattr(lib, n), n


def test_no_torch_or_oracle_in_the_library():
    import paper_2503_23728_b200 as pb
    out = subprocess.run(["ldd", pb.library_path()], capture_output=True, text=True).stdout
    assert "torch" not in out and "oracle" not in out and "c10" not in out


def test_sm100a_code_and_no_oracle_import():
    import paper_2503_23728_b200 as pb
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", pb.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    pkg = os.path.join(ROOT, "paper_2503_23728_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "pimd_oracle" not in src, f


def test_workspace_bytes_host_only(lib):
    """pimd_workspace_bytes is pure host logic: callable without a GPU."""
    import ctypes as C
    import numpy as np
    import paper_2503_23728_b200 as pb
    import pimd_inputs as pi
    w = pi.make_workload("ice512")
    keep = []
    from paper_2503_23728_b200.pimd import _net_struct
    npar = _net_struct(w.net, keep)
    n = C.c_size_t()
    box = np.ascontiguousarray(w.box)
    rc = lib.pimd_workspace_bytes(w.n_atoms, 1, w.P, box.ctypes.data_as(C.POINTER(C.c_double)), C.byref(npar), C.byref(n))
    assert rc == 0 and 100e6 < n.value < 8e9   # incl. the tile images the tcgen05 pair passes keep (pair capacity x 280 B)
    bad = np.array([5.0, 5.0, 5.0])
    rc = lib.pimd_workspace_bytes(w.n_atoms, 1, w.P, bad.ctypes.data_as(C.POINTER(C.c_double)), C.byref(npar), C.byref(n))
    assert rc == -1 and b"r_cut" in lib.pimd_last_error()
    rc = lib.pimd_workspace_bytes(w.n_atoms, 1, 1000, box.ctypes.data_as(C.POINTER(C.c_double)), C.byref(npar), C.byref(n))
    assert rc == -1
