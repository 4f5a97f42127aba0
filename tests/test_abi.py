"""CPU-side checks of the boundary: the C-ABI library loads without a GPU and exports every symbol that
include/dode.h declares; argument errors are reported without touching a device."""
import ctypes as C
import os
import re

import paper_1901_09266_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "dode.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dode_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import __graft_entry__ as g
    g.build()
    lib = P.lib()
    names = _declared()
    assert len(names) >= 14
    for n in names:
        assert hasattr(lib, n), f"libdode.so does not export {n}"
    assert sorted(P.EXPORTS) == names


def test_create_rejects_bad_arguments_without_a_device():
    lib = P.lib()
    h = C.c_void_p()
    assert lib.dode_create(C.byref(h), None, None, None, None, C.c_float(1.0), None) == P.DODE_EINVAL
    assert h.value is None
    assert b"null" in lib.dode_last_error(None)
    dims = P.dode_dims(0, 6, 288, 6, 1, 14, 0)
    dar = P.dode_dar()
    lab = (C.c_int32 * 14)()
    fake = C.c_void_p(16)
    assert lib.dode_create(C.byref(h), C.byref(dims), C.byref(dar), lab, fake, C.c_float(1.0), None) == P.DODE_EINVAL
    assert b"positive" in lib.dode_last_error(None)
    assert lib.dode_spgd_step(None, None, 0, C.c_float(0.1)) == P.DODE_EINVAL


def test_oracle_and_cuda_sources_share_nothing():
    """The oracle includes nothing from the package and vice versa."""
    osrc = open(os.path.join(ROOT, "oracle", "dode_oracle.cpp")).read()
    assert not re.search(r"#include\s*[<\"][^>\"]*(dode\.h|kernels_|csrc)", osrc)
    pat = re.compile(r"(^\s*(import|from)\s+oracle\b)|(#include\s*[<\"].*oracle)|liboracle|dode_oracle", re.M)
    for root, _, files in os.walk(os.path.join(ROOT, "paper_1901_09266_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(root, f)).read()), f


def test_library_reads_nothing_from_the_environment():
    """include/dode.h: "no global state" — kernel selection is steered by dode_set_option only."""
    csrc = os.path.join(ROOT, "paper_1901_09266_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f
    lib = P.lib()
    assert lib.dode_set_option(None, 0, 1) == P.DODE_EINVAL
    assert lib.dode_reserve(None, 8) == P.DODE_EINVAL
