"""The C-ABI library loads and exports every symbol include/ss.h declares; host-side argument
logic (no compute calls: this runs without a GPU)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2603_24370_b200 import build
    return C.CDLL(build.build())


def test_every_declared_symbol_is_exported(lib):
    from paper_2603_24370_b200.build import declared_symbols
    names = declared_symbols()
    assert {"ss_create", "ss_set_fields", "ss_step", "ss_energy", "ss_charge",
            "ss_get_fields"} <= set(names)              # north_star's list
    for n in names:
        assert hasattr(lib, n), n


def test_binding_names_match_header():
    from paper_2603_24370_b200 import ss
    from paper_2603_24370_b200.build import declared_symbols
    assert sorted(ss.EXPORTS) == declared_symbols()


def test_params_struct_matches_header():
    from paper_2603_24370_b200 import ss
    text = open(os.path.join(ROOT, "include", "ss.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} ss_params;", text, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            names = re.sub(r"^(const\s+)?\w+(\s*\*)?\s+", "", decl)
            fields += [n.strip().lstrip("*") for n in names.split(",")]
    got = [n for n, _ in ss.ss_params._fields_]
    assert [f.replace("lambda", "lam") for f in fields] == got


def test_workspace_bytes_host_logic():
    from paper_2603_24370_b200 import ss
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 63, 64) == 0       # odd Nx, fp64
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 66, 64, dtype=ss.F32) == 0
    assert ss.workspace_bytes(7, 64, 64) == 0                              # unknown theory
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 4, 64) == 0         # no interior
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 64, 64, batch=0) == 0
    # limits of this build (include/ss.h "Limits")
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 65538, 8) == 0
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 8, 32770) == 0
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 8, 8, batch=65536) == 0
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 65536, 8) > 0
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 8, 32768) > 0
    cm = ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 64, 64)
    ah = ss.workspace_bytes(ss.THEORY_ABELIAN_HIGGS, 64, 64)
    assert cm >= 6 * 3 * 64 * 64 * 8 and ah > cm         # phi, v twice; a1, a2
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 64, 64, batch=3) > 2 * cm
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 64, 64, dtype=ss.F32) < cm
    # config 4 fp64 fits one B200 (180 GB) with room to spare
    assert ss.workspace_bytes(ss.THEORY_CHIRAL_MAGNET, 4096, 4096) < 4 * 2**30


def test_strerror_and_null_handles(lib):
    from paper_2603_24370_b200 import ss
    assert ss.strerror(ss.OK) == "ok" and "argument" in ss.strerror(ss.ERR_ARG)
    assert ss.strerror(12345) == "unknown status"
    lib.ss_step.argtypes = [C.c_void_p, C.c_int64]
    lib.ss_destroy.argtypes = [C.c_void_p]
    lib.ss_launch_count.argtypes = [C.c_void_p]
    lib.ss_launch_count.restype = C.c_int64
    assert lib.ss_step(None, 1) == ss.ERR_ARG
    assert lib.ss_destroy(None) == ss.ERR_ARG
    assert lib.ss_launch_count(None) == 0


def test_no_cpu_fallback_without_device():
    import torch
    from paper_2603_24370_b200 import ss
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    with pytest.raises(ss.SSError) as e:
        ss.Solver(ss.THEORY_CHIRAL_MAGNET, 64, 64, 0.2)
    assert e.value.code == ss.ERR_CUDA
