"""The C-ABI library loads and exports every symbol include/tridsk.h declares (no GPU, no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2510_24186_b200 import build
    return ctypes.CDLL(build.build())


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "tridsk.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tridsk_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("tridsk_build_grid", "tridsk_load_ligands", "tridsk_dock", "tridsk_score_grad"):
        assert name in syms


def test_every_declared_symbol_is_exported(built_lib):
    syms = declared_symbols()
    assert len(syms) >= 15
    for name in syms:
        assert hasattr(built_lib, name), name


def test_struct_layouts_match_the_header(built_lib):
    from paper_2510_24186_b200 import binding
    assert ctypes.sizeof(binding.Params) == 21 * 4
    assert binding.TRACE_DTYPE.itemsize == 16
    p = binding.Params()
    built_lib.tridsk_default_params(ctypes.byref(p))
    assert (round(p.w_long, 6), p.w_clash, round(p.w_hbond, 6)) == (0.2, 10.0, 0.6)
    assert (round(p.beta, 6), round(p.lr, 6), round(p.w_tor, 6), p.n_refine) == (0.069, 0.1, 0.01, 1)


def test_no_cpu_fallback(built_lib):
    """Without a CUDA device the library must fail loudly, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    ctx = ctypes.c_void_p()
    assert built_lib.tridsk_create(ctypes.byref(ctx), 0, None) == -3
    from paper_2510_24186_b200 import Engine
    with pytest.raises(RuntimeError):
        Engine()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2510_24186_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "oracle" not in txt.lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2510_24186_b200" not in txt.replace("paper_2510_24186_b200/csrc)", "").replace("(paper_2510_24186_b200/csrc", ""), f
