"""The C-ABI library loads without a GPU and exports every entry point include/*.h declares; the
Python binding lists exactly the same names (no compute calls here); the library reads no
environment variable."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(header="pfc.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return set(re.findall(r"\b(pfc_[a-z0-9_]+)\s*\(", text))


def test_library_exports_every_declared_symbol():
    from paper_2412_18271_b200 import build, pfc
    build.build_libpfc()
    lib = ctypes.CDLL(pfc.LIB_PATH)
    names, debug, noalloc = _declared("pfc.h"), _declared("pfc_debug.h"), _declared("pfc_noalloc.h")
    assert {"pfc_create", "pfc_energy_forces", "pfc_step", "pfc_destroy"} <= names      # the north_star four
    missing = [n for n in sorted(names | debug | noalloc) if not hasattr(lib, n)]
    assert not missing, missing
    assert set(pfc.EXPORTS) == names
    assert set(pfc.DEBUG_EXPORTS) == debug
    assert set(pfc.NOALLOC_EXPORTS) == noalloc
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["pfc.h", "pfc_debug.h", "pfc_noalloc.h"]
    assert len(names) <= 16                                    # "keep them few"


def test_library_reads_no_environment_variable():
    """SURVEY.md section 5 / north_star: no env-var dispatch.  Tuning goes through pfc_tuning_t."""
    csrc = os.path.join(ROOT, "paper_2412_18271_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f
    from paper_2412_18271_b200 import pfc
    import ctypes as C
    assert C.sizeof(pfc.Tuning) == 32                          # mirrors pfc_tuning_t


def test_host_only_entry_points_work_without_a_device():
    from paper_2412_18271_b200 import pfc
    lib = pfc.load_library()
    assert lib.pfc_workspace_bytes(22, 1) > 0
    assert lib.pfc_workspace_bytes(0, 1) == 0 and lib.pfc_workspace_bytes(5, 9) == 0
    assert lib.pfc_error_string(0) is not None and lib.pfc_error_string(-1) != lib.pfc_error_string(-2)
    assert lib.pfc_step(None, 1, ctypes.c_float(0.5)) != 0                              # NULL handle: error code, no crash
    assert lib.pfc_step_langevin(None, 1, ctypes.c_float(0.5), ctypes.c_float(0.0), ctypes.c_float(300.0), 1) != 0
    assert lib.pfc_set_frames(None, None, 0, 0) != 0
