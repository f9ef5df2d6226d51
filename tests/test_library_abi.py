"""CPU-side checks of the C-ABI boundary: libdmfe.so loads without a GPU and exports every symbol
that include/dmfe.h declares; the binding's struct layouts match the header's field order;
the product package never imports the oracle."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_06309_b200 import build, dmfe
    build.build()
    return dmfe.load_library()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "dmfe.h")).read()
    return sorted(set(re.findall(r"DMFE_API\s+[\w\s\*]*?\b(dmfe_\w+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 10 and "dmfe_history_integrals" in names and "dmfe_sparsify" in names
    for n in names:
        assert hasattr(lib, n), "libdmfe.so does not export %s" % n


def test_binding_lists_the_same_symbols():
    from paper_2604_06309_b200 import dmfe
    assert sorted(dmfe.EXPORTS) == _declared_symbols()


def test_strerror_and_null_handling(lib):
    assert lib.dmfe_strerror(0) == b"ok"
    assert lib.dmfe_strerror(-3) == b"history capacity exhausted"
    assert lib.dmfe_destroy(None) == -1                      # DMFE_EINVAL, no crash
    assert lib.dmfe_history_integrals(None, None, None) == -1


def _header_struct_fields(name):
    src = open(os.path.join(ROOT, "include", "dmfe.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    body = re.search(r"typedef struct \{([^}]*)\}\s*%s;" % name, src).group(1)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            fields.append(re.findall(r"(\w+)\s*$", decl)[0])
    return fields


@pytest.mark.parametrize("name", ["dmfe_params", "dmfe_grid", "dmfe_rhs_out", "dmfe_state", "dmfe_advance_result",
                                  "dmfe_policy", "dmfe_run_stats"])
def test_struct_field_order_matches_header(name):
    from paper_2604_06309_b200 import dmfe
    assert [f[0] for f in getattr(dmfe, name)._fields_] == _header_struct_fields(name)


def test_struct_sizes_match_the_c_layout():
    """ctypes lays the mirrored structs out like the C compiler does (natural alignment)."""
    import ctypes
    from paper_2604_06309_b200 import dmfe
    assert ctypes.sizeof(dmfe.dmfe_advance_result) == 5 * 4 + 4 + 3 * 8
    assert ctypes.sizeof(dmfe.dmfe_policy) == 3 * 4 + 4 + 8 + 2 * 4
    assert ctypes.sizeof(dmfe.dmfe_run_stats) == 7 * 8 + 4 * 4 + 3 * 8
    assert dmfe.dmfe_policy.sp_min_gain.offset == 16 and dmfe.dmfe_policy.protect_last.offset == 24


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2604_06309_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, re.M), "%s imports the oracle" % f
                assert "liboracle" not in txt and "dmfe_oracle" not in txt, "%s uses the oracle" % f


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2604_06309_b200 import dmfe
    with pytest.raises(RuntimeError):
        dmfe.dmfe_create(64, 4, 100.0, [0, 0, 0, 1.0], T=1.0)
