"""The C-ABI library builds for sm_100a, loads without a GPU, and exports every symbol include/mkf.h declares."""
import ctypes as C
import os
import re

from paper_2002_06295_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mkf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mkf_[a-z_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    L = C.CDLL(path)
    names = declared_symbols()
    assert {"mkf_build_hit_index", "mkf_fit", "mkf_build_tracks", "mkf_remove_duplicates"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS) == names


def test_create_validates_arguments_without_gpu():
    from workloads import datagen
    g = datagen.geometry_barrel(4, 4.0, 16.0, 50.0, 0.02)
    ctx = binding.Context(g, datagen.default_params())
    assert ctx.max_plan_len == 4
    assert ctx.workspace_bytes(binding.CALL_BUILD_HIT_INDEX, 2, 1000, 0) >= 2 * 4 * 63 * 40 * 4 + 4000
    assert ctx.workspace_bytes(binding.CALL_FIT, 2, 1000, 10) == 0
    ctx.close()
    import pytest
    with pytest.raises(binding.MkfError):
        binding.Context(g, datagen.default_params(max_cand=9))           # > MKF_MAX_CAND -> UNSUPPORTED
    bad = dict(g); bad["plan_layers"] = g["plan_layers"] + 7
    with pytest.raises(binding.MkfError):
        binding.Context(bad, datagen.default_params())                    # layer index out of range -> INVALID_ARG


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2002_06295_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "mkfo" not in txt and "import oracle" not in txt and "from oracle" not in txt, f
