"""-m "not gpu": the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/dsmc.h declares (no compute calls without a GPU); host-side argument checks."""
import ctypes as C
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    from paper_2602_21244_b200 import build
    return C.CDLL(build.build())


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "dsmc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(dsmc_[a-z_0-9]+)\s*\(", hdr)))
    assert len(names) >= 15
    lib = _lib()
    for n in names:
        assert hasattr(lib, n), n
    from paper_2602_21244_b200 import dsmc
    assert sorted(dsmc.EXPORTS) == names


def test_strerror_and_host_side_argument_errors():
    lib = _lib()
    lib.dsmc_strerror.restype = C.c_char_p
    assert lib.dsmc_strerror(0) == b"ok"
    assert b"cell" in lib.dsmc_strerror(-2)
    assert lib.dsmc_create(None, 0, C.c_int64(10), 4) == -1  # null out pointer: invalid argument
    assert lib.dsmc_sync_status(None) == -1
    assert lib.dsmc_set_stream(None, None) == -1
    # the section-9 entry points reject a null context before touching anything
    assert lib.dsmc_move_couette(None, C.c_int64(4), None, None, None, None, None, None, None, C.c_uint64(0), 0) == -1
    assert lib.dsmc_gather_f32(None, C.c_int64(4), None, None, None) == -1
    assert lib.dsmc_sample_cells(None, C.c_int64(4), 1, None, None, None, None, None) == -1
    assert lib.dsmc_ntc_counts(None, 1, None, None, C.c_double(1.0), None, None) == -1
    assert lib.dsmc_couette_run(None, C.c_int64(4), None, None, None, None, None, None, None, C.c_uint64(0), 0, 1, 0, None) == -1


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_21244_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "dsmc_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "csrc" not in src.replace("paper_2602_21244_b200/csrc/", "") or f.endswith(".h")
            assert "import paper_2602_21244_b200" not in src and "from paper_2602_21244_b200" not in src
