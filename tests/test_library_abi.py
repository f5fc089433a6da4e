"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, and exports every symbol include/loc.h declares.
No compute call is made here (no GPU in the build container)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "loc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(loc_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for n in ("loc_create_model", "loc_set_species", "loc_simulate", "loc_solve", "loc_iterate", "loc_spectra"):
        assert n in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2009_12609_b200 import binding as B
    lib = B.lib()
    for n in _declared_symbols():
        assert hasattr(lib, n), n
    assert sorted(B.SYMBOLS) == _declared_symbols()


def test_sass_is_sm100a():
    from paper_2009_12609_b200 import build
    import subprocess
    so = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", so], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_workspace_bytes_host_only():
    """loc_workspace_bytes is pure host arithmetic: callable without a GPU; rejects bad arguments."""
    import numpy as np
    from paper_2009_12609_b200 import binding as B
    g, keep = B.make_shell_grid(np.array([1.0, 2.0, 3.0]), np.array([0.5, 1.5, 2.5]), np.array([1.0, 1.0, 1.0]))
    n = B.loc_workspace_bytes(g, 64, 5, 4, 1)
    assert n > 0 and n % 256 == 0
    with pytest.raises(B.LocError):
        B.loc_workspace_bytes(g, 0, 5, 4, 1)
    g3 = B.loc_grid(kind=B.LOC_GRID_OCTREE, nx=4, ny=4, nz=4, root_cell_cm=1.0, nlevel=1,
                    level_offset=np.array([0, 64], np.int64).ctypes.data_as(ctypes.c_void_p))
    assert B.loc_workspace_bytes(g3, 32, 3, 2, 12) > 0


def test_no_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import loc_workloads as W
    from paper_2009_12609_b200 import LocModel, binding as B
    with pytest.raises(B.LocError):
        LocModel(W.shell_config(1))
