"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/fdas.h declares,
and rejects bad arguments before touching the device.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fd():
    from paper_1804_05335_b200 import build
    build.build()
    from paper_1804_05335_b200 import fdas
    return fdas


def test_header_symbols_are_exported(fd):
    hdr = open(os.path.join(ROOT, "include", "fdas.h")).read()
    declared = set(re.findall(r"\b(fdas_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(fd.EXPORTS)
    for name in declared:
        assert hasattr(fd.lib, name), name


def test_info_struct_matches_header(fd):
    hdr = open(os.path.join(ROOT, "include", "fdas.h")).read()
    body = re.search(r"typedef struct fdas_info \{(.*?)\} fdas_info;", hdr, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        _, rest = decl.split(None, 1)
        names += [n.strip() for n in rest.split(",")]
    assert names == [n for n, _ in fd.FdasInfo._fields_]
    assert ctypes.sizeof(fd.FdasInfo) == 5 * 8 + 2 * 8 + 14 * 4


def test_argument_errors_without_device(fd):
    h = ctypes.c_void_p()
    lib = fd.lib
    assert lib.fdas_plan_create(None, 1024, 20.0, 2.0, 1024, 0) == 1
    assert lib.fdas_plan_create(ctypes.byref(h), 0, 20.0, 2.0, 1024, 0) == 1
    assert lib.fdas_plan_create(ctypes.byref(h), 1024, -1.0, 2.0, 1024, 0) == 1
    assert lib.fdas_plan_create(ctypes.byref(h), 1024, 20.0, 0.0, 1024, 0) == 1
    assert lib.fdas_plan_create(ctypes.byref(h), 1024, 5.0, 2.0, 1024, 0) == 1       # zmax/dz not integer
    assert lib.fdas_plan_create(ctypes.byref(h), 1024, 20.0, 2.0, 1024, 3) == 1
    assert lib.fdas_plan_create(ctypes.byref(h), 1024, 20.0, 2.0, 1000, 0) == 2      # seglen
    assert lib.fdas_plan_create(ctypes.byref(h), 1024, 2000.0, 2.0, 1024, 0) == 2    # overlap >= seglen/2
    assert lib.fdas_plan_create(ctypes.byref(h), 1 << 20, 8100.0, 2.0, 8192, 1) == 2  # overlap >= seglen/2
    assert h.value is None
    assert lib.fdas_destroy(None) == 0
    assert lib.fdas_execute(None, None, None, None) == 1
    assert lib.fdas_status_string(3) == b"FDAS_ERR_NOT_READY"
    assert lib.fdas_last_error(None) == b""
    assert lib.fdas_launch_count() == 0


def test_product_path_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1804_05335_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|from\s+\.\.?oracle|oracle[./]|libfdas_oracle", src), f
