"""CPU-side checks of the boundary (no compute call is made without a GPU):
the C-ABI library builds for sm_100a, loads, and exports every symbol include/hdc.h declares; the
Python binding lists the same names; the header's enums match the binding's constants; without a
CUDA device hdc_create fails loudly (there is no CPU fallback); the built library carries the
sm_100a tensor-core / TMA instructions the design claims."""
from __future__ import annotations

import ctypes as C
import os
import re
import shutil
import subprocess

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hdc.h")


@pytest.fixture(scope="module")
def libpath():
    from paper_2606_26547_b200 import build
    return build.build()


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    src = re.sub(r"//[^\n]*", "", src)
    return sorted(set(re.findall(r"\b(hdc_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_five_hot_path_calls():
    names = declared_symbols()
    for n in ("hdc_encode_rp", "hdc_encode_levelid", "hdc_similarity", "hdc_classify", "hdc_train_epoch"):
        assert n in names


def test_library_exports_every_declared_symbol(libpath):
    L = C.CDLL(libpath)
    for n in declared_symbols():
        assert hasattr(L, n), f"{n} is declared in include/hdc.h but not exported by libhdc.so"


def test_binding_lists_the_same_names(libpath):
    from paper_2606_26547_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_binding_constants_match_header():
    from paper_2606_26547_b200 import binding
    src = open(HEADER).read()
    pairs = re.findall(r"\b(HDC_[A-Z0-9_]+)\s*=\s*(-?\d+)", src)
    assert len(pairs) >= 20
    for name, val in pairs:
        if hasattr(binding, name):
            assert getattr(binding, name) == int(val), name
    for must in ("HDC_OK", "HDC_F32", "HDC_BF16", "HDC_I8", "HDC_SIM_COS", "HDC_SIM_HAMMING",
                 "HDC_TRAIN_PERCEPTRON", "HDC_OUT_BITS"):
        assert must in dict(pairs) and hasattr(binding, must)


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback_without_a_device(libpath):
    import paper_2606_26547_b200 as hd
    with pytest.raises(Exception):
        hd.Handle(0)


def test_oracle_and_product_do_not_import_each_other():
    pkg = os.path.join(ROOT, "paper_2606_26547_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+(paper_2606_26547_b200|ctypes|torch)\b", s, flags=re.M), f


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not on PATH")
def test_sass_has_tcgen05_tmem_and_tma(libpath):
    sass = subprocess.run(["cuobjdump", "-sass", libpath], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in sass
    assert re.search(r"\bUTC[A-Z]*MMA\b", sass), "no tcgen05.mma (UTC*MMA) in libhdc.so"
    assert "LDTM" in sass, "no tcgen05.ld (LDTM) in libhdc.so"
    assert "UTMALDG" in sass, "no TMA tensor load (UTMALDG) in libhdc.so"


def test_binding_structs_match_header_field_for_field():
    """hdc_knobs_t / hdc_adc_t cross the ABI by value layout: same int32 fields, same order, on both sides."""
    from paper_2606_26547_b200 import binding
    import ctypes as C
    src = open(HEADER).read()
    for cname, cls in (("hdc_knobs_t", binding.hdc_knobs_t), ("hdc_adc_t", binding.hdc_adc_t)):
        m = re.search(r"typedef struct \{([^}]*)\}\s*" + cname + r"\s*;", src)
        assert m, cname
        body = re.sub(r"/\*.*?\*/", "", m.group(1), flags=re.S)
        fields = re.findall(r"int32_t\s+(\w+)\s*;", body)
        assert fields == [f[0] for f in cls._fields_], cname
        assert all(f[1] is C.c_int32 for f in cls._fields_)
        assert C.sizeof(cls) == 4 * len(fields)


@pytest.mark.skipif(shutil.which("gcc") is None, reason="gcc not on PATH")
def test_model_descriptor_layout_matches_the_c_compiler(tmp_path):
    """hdc_model_t is filled by the library and read back by the binding: sizeof and every offsetof, as gcc
    lays the header's struct out, must equal the ctypes Structure's."""
    from paper_2606_26547_b200 import binding
    names = [f[0] for f in binding.hdc_model_t._fields_]
    src = tmp_path / "layout.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "hdc.h"\nint main(void){\n'
                   'printf("%zu\\n", sizeof(hdc_model_t));\n' +
                   "".join(f'printf("%zu\\n", offsetof(hdc_model_t, {n}));\n' for n in names) + "return 0;}\n")
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    assert out[0] == C.sizeof(binding.hdc_model_t)
    assert out[1:] == [getattr(binding.hdc_model_t, n).offset for n in names]
