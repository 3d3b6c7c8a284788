"""CPU-side checks of the boundary: the C-ABI library builds/loads and exports every symbol include/mbhl.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mbhl.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mbhl_[a-z_]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    names = declared_symbols()
    for required in ("mbhl_init", "mbhl_loglike", "mbhl_loglike_parts", "mbhl_template", "mbhl_sparse",
                     "mbhl_workspace_bytes", "mbhl_set_workspace", "mbhl_strerror", "mbhl_last_error", "mbhl_free"):
        assert required in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2005_01827_b200 import binding, build
    path = build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(L, name), name
    assert sorted(binding.SYMBOLS) == declared_symbols()
    # host-only entry points work without a GPU
    lib = binding.lib()
    assert lib.mbhl_strerror(0) == b"ok" and lib.mbhl_strerror(-1) == b"invalid argument"
    assert lib.mbhl_last_error(None) == b"null context"
    ctx = ctypes.c_void_p()
    assert lib.mbhl_init(ctypes.byref(ctx), None, 0, None, None, None) == -1      # MBHL_EINVAL, no device touched
    assert lib.mbhl_workspace_bytes(None, 4) == 0


def test_model_table_is_baked_in_csv_order():
    from paper_2005_01827_b200 import build
    build.bake_table()
    inc = open(build.TABLE_INC).read()
    rows = [l.strip().split(",") for l in open(build.TABLE_CSV) if l.strip() and not l.startswith("#")]
    assert f"#define MBHL_TABLE_N {len(rows)}" in inc
    for i, (name, value, _) in enumerate(rows[:5] + rows[-5:]):
        idx = i if i < 5 else len(rows) - 10 + i
        assert f"MT_{name.replace('.', '_')} = {idx}," in inc
        assert repr(float(value)) in inc


def test_product_path_has_no_oracle_import():
    pkg = os.path.join(ROOT, "paper_2005_01827_b200")
    for fn in os.listdir(pkg):
        if fn.endswith(".py"):
            src = open(os.path.join(pkg, fn)).read()
            assert "import oracle" not in src and "from oracle" not in src, fn
