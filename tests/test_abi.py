"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol that
include/rumd_b200.h declares, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rumd_b200.h")


@pytest.fixture(scope="module")
def libpath():
    from paper_1506_05094_b200 import build

    return build.build()


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rumd_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_mandated_entry_points():
    names = declared_symbols()
    for must in ("rumd_create", "rumd_set_pair_potential", "rumd_build_nblist", "rumd_compute_forces",
                 "rumd_run_steps"):
        assert must in names


def test_library_exports_every_declared_symbol(libpath):
    L = C.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(L, name), name


def test_binding_lists_the_same_names():
    src = open(os.path.join(ROOT, "paper_1506_05094_b200", "rumd.py")).read()
    listed = set(re.findall(r'"(rumd_[a-z_0-9]+)"', src))
    assert listed == set(declared_symbols())


def test_no_cpu_fallback(libpath):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    L = C.CDLL(libpath)
    h = C.c_void_p()
    box = (C.c_float * 3)(10, 10, 10)
    assert L.rumd_create(C.byref(h), 100, 1, box, None) == 3  # RUMD_ERR_CUDA
    from paper_1506_05094_b200 import rumd, workloads as W

    wl = W.lj_fcc(2)
    with pytest.raises(RuntimeError):
        rumd.System(wl.r, wl.v, wl.m, wl.types, wl.box, wl.pot)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1506_05094_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", txt, flags=re.M), f
                assert "rumd_oracle" not in txt, f


def test_binding_constants_match_the_header_enums():
    """Every enumerator of include/rumd_b200.h has the same value in the ctypes binding (RUMD_X -> rumd.X), and
    the tuning struct of the binding has the header's fields in the header's order."""
    from paper_1506_05094_b200 import rumd

    src = open(HEADER).read()
    enums = dict((k, int(v)) for k, v in re.findall(r"\bRUMD_([A-Z][A-Z_0-9]*)\s*=\s*(\d+)", src))
    assert len(enums) >= 24
    for name, value in enums.items():
        assert getattr(rumd, name) == value, name
    body = re.search(r"typedef struct(?:\s+\w+)?\s*\{([^}]*)\}\s*rumd_tuning\s*;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = [m.group(1) for m in re.finditer(r"\b(?:int|float)\s+(\w+)\s*;", body)]
    assert fields == [f[0] for f in rumd.Tuning._fields_]


def test_noalloc_entry_point_rejects_oversize_before_touching_the_device(libpath):
    """rumd_forces_noalloc validates its sizes on the host first: beyond RUMD_NOALLOC_MAX_PARTICLES it returns
    RUMD_ERR_INVALID_ARG with a message that names the limit -- with or without a GPU (no compute call is made)."""
    from paper_1506_05094_b200 import rumd

    src = open(HEADER).read()
    limit = int(re.search(r"#define\s+RUMD_NOALLOC_MAX_PARTICLES\s+(\d+)", src).group(1))
    cap = int(re.search(r"#define\s+RUMD_NOALLOC_NBL_CAPACITY\s+(\d+)", src).group(1))
    assert (limit, cap) == (rumd.NOALLOC_MAX_PARTICLES, rumd.NOALLOC_NBL_CAPACITY)
    L = rumd.lib()
    box = (C.c_float * 3)(20, 20, 20)
    pair = (rumd.NoallocPair * 1)(rumd.NoallocPair(1.0, 1.0, 2.5, 0.0, 0.0))
    err = C.create_string_buffer(256)
    fake = C.c_void_p(256)  # never dereferenced: the size check comes first
    st = L.rumd_forces_noalloc(limit + 1, 1, box, pair, 0.3, fake, fake, fake, fake, None, err, len(err))
    assert st == rumd.ERR_INVALID_ARG
    assert b"RUMD_NOALLOC_MAX_PARTICLES" in err.value and str(limit).encode() in err.value
    st = L.rumd_forces_noalloc(0, 1, box, pair, 0.3, fake, fake, fake, fake, None, err, len(err))
    assert st == rumd.ERR_INVALID_ARG and err.value
    st = L.rumd_forces_noalloc(100, 5, box, pair, 0.3, fake, fake, fake, fake, None, err, len(err))
    assert st == rumd.ERR_INVALID_ARG and b"n_types" in err.value
