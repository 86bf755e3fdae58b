"""CPU-side checks of the boundary: the library builds for sm_100a, loads, and exports every symbol that
include/afqmc.h declares.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2209_04015_b200.build import build_library
    return build_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "afqmc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(afqmc_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib_path):
    lib = ctypes.CDLL(lib_path)
    syms = declared_symbols()
    assert {"afqmc_create", "afqmc_local_energy", "afqmc_destroy", "afqmc_last_error"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s


def test_binding_covers_header(lib_path):
    from paper_2209_04015_b200.binding import EXPORTS, load_library
    assert sorted(EXPORTS) == declared_symbols()
    load_library()


def test_info_struct_matches_header():
    from paper_2209_04015_b200.binding import AfqmcInfo
    src = open(os.path.join(ROOT, "include", "afqmc.h")).read()
    body = re.search(r"typedef struct afqmc_info \{(.*?)\} afqmc_info;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        decl = re.sub(r"^(long long|int)\s+", "", decl)
        names += [re.sub(r"\[.*\]", "", x).strip() for x in decl.split(",")]
    assert names == [n for n, _ in AfqmcInfo._fields_]


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2209_04015_b200 import AfqmcError, LocalEnergy
    t = torch.zeros(4, dtype=torch.float64)
    with pytest.raises(AfqmcError):
        LocalEnergy(t, t, t.to(torch.complex128), 2, 1, 0, 1, 0.0, 1)


def test_product_path_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2209_04015_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("CPU oracle", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2209_04015_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_2209_04015_b200/``", "")
