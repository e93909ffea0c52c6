"""The C-ABI library loads without a GPU and exports every entry point include/pfc.h declares; the
Python binding lists exactly the same names (no compute calls here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "pfc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return set(re.findall(r"\b(pfc_[a-z0-9_]+)\s*\(", text))


def test_library_exports_every_declared_symbol():
    from paper_2412_18271_b200 import build, pfc
    build.build_libpfc()
    lib = ctypes.CDLL(pfc.LIB_PATH)
    names = _declared()
    assert {"pfc_create", "pfc_energy_forces", "pfc_step", "pfc_destroy"} <= names      # the north_star four
    missing = [n for n in sorted(names) if not hasattr(lib, n)]
    assert not missing, missing
    assert set(pfc.EXPORTS) == names


def test_host_only_entry_points_work_without_a_device():
    from paper_2412_18271_b200 import pfc
    lib = pfc.load_library()
    assert lib.pfc_workspace_bytes(22, 1) > 0
    assert lib.pfc_workspace_bytes(0, 1) == 0 and lib.pfc_workspace_bytes(5, 9) == 0
    assert lib.pfc_error_string(0) is not None and lib.pfc_error_string(-1) != lib.pfc_error_string(-2)
    assert lib.pfc_step(None, 1, ctypes.c_float(0.5)) != 0                              # NULL handle: error code, no crash
    assert lib.pfc_step_langevin(None, 1, ctypes.c_float(0.5), ctypes.c_float(0.0), ctypes.c_float(300.0), 1) != 0
    assert lib.pfc_set_frames(None, None, 0, 0) != 0
