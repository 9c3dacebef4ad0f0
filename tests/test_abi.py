"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol that
include/sg.h declares; the binding lists the same names; argument validation that needs no GPU."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "sg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sg_[a-z_0-9]+)\s*\(", src)))


def _lib():
    from paper_1403_4560_b200 import build
    return ctypes.CDLL(build.build())


def test_library_exports_every_declared_symbol():
    names = _declared()
    assert "sg_create" in names and "sg_sweep" in names and "sg_pt_exchange" in names and "sg_measure" in names \
        and "sg_destroy" in names and "sg_run" in names
    lib = _lib()
    for n in names:
        assert hasattr(lib, n), n


def test_binding_covers_the_header():
    import importlib.util
    spec = importlib.util.spec_from_file_location("sg_binding_src", os.path.join(ROOT, "paper_1403_4560_b200", "sg.py"))
    src = open(spec.origin).read()
    for n in _declared():
        assert '"%s"' % n in src, "binding lacks %s" % n


def test_workspace_bytes_and_validation_without_gpu():
    lib = _lib()
    lib.sg_workspace_bytes.restype = ctypes.c_size_t
    lib.sg_workspace_bytes.argtypes = [ctypes.c_int] * 5
    assert lib.sg_workspace_bytes(5, 1, 4, 8, 0) == 0          # odd L
    assert lib.sg_workspace_bytes(4, 0, 4, 8, 0) == 0          # no samples
    assert lib.sg_workspace_bytes(4, 1, 3, 8, 0) == 0          # replicas not in {2,4}
    assert lib.sg_workspace_bytes(4, 1, 4, 0, 0) == 0
    assert lib.sg_workspace_bytes(4, 1, 4, 8, 3) == 0          # unknown coupling_kind (0, 1, 2 exist)
    # SG_PMJ_TPACK keeps the sample-packed state AND its own temperature-packed copy; SG_PMJ (L <= 16, L = 32) keeps a
    # second sample-packed buffer instead (overlapped measurements / swap on load): both exceed one state (4096 B here)
    one_state = 1 * 4 * 8 * 64 * 4
    assert lib.sg_workspace_bytes(4, 1, 4, 8, 2) > one_state and lib.sg_workspace_bytes(4, 1, 4, 8, 0) > 2 * one_state
    assert lib.sg_workspace_bytes(4, 1, 4, 8, 2) != lib.sg_workspace_bytes(4, 1, 4, 8, 0)
    c1 = lib.sg_workspace_bytes(4, 1, 4, 8, 0)
    assert c1 >= 8 * 1024 and c1 % 256 == 0
    # config 5: 2 x ~4.3 GB bit-packed state (double-buffered for the L = 32 kernel) + couplings + scratch, far below 180 GB
    c5 = lib.sg_workspace_bytes(32, 8192, 4, 32, 0)
    assert 2 * 4.29e9 < c5 < 1.0e10
    c4 = lib.sg_workspace_bytes(16, 512, 4, 32, 1)
    assert 2.68e8 < c4 < 1e9
    # invalid arguments are rejected before any CUDA call
    lib.sg_create.restype = ctypes.c_int
    out = ctypes.c_void_p()
    temps = (ctypes.c_double * 2)(2.0, 1.0)
    rc = lib.sg_create(ctypes.byref(out), 4, ctypes.c_double(0.1), 1, 4, temps, 2, 0, ctypes.c_uint64(1), None,
                       ctypes.c_size_t(0), None)
    assert rc == -1 and not out.value
    lib.sg_last_error.restype = ctypes.c_char_p
    assert b"non-decreasing" in lib.sg_last_error(None)
    # the message for a bad coupling_kind names all three kinds (SG_PMJ_TPACK = 2 exists)
    temps = (ctypes.c_double * 2)(1.0, 2.0)
    rc = lib.sg_create(ctypes.byref(out), 4, ctypes.c_double(0.1), 1, 4, temps, 2, 3, ctypes.c_uint64(1), None,
                       ctypes.c_size_t(0), None)
    assert rc == -1 and not out.value
    assert b"SG_PMJ_TPACK" in lib.sg_last_error(None)
