"""The C-ABI library builds for sm_100a, loads without a GPU and exports every function include/spgpe.h
declares (no compute calls here)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "spgpe.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(spgpe_[a-z0-9_]+)\s*\(", src)))


def test_header_functions_are_exported_and_bound():
    import paper_2010_15069_b200 as sp
    sp.build()
    L = sp.lib()
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"libspgpe.so does not export {n}"
    assert sorted(sp.ABI_SYMBOLS) == names
    # the thin binding carries the same names (spgpe_last_cuda_error / spgpe_strerror are used inside _check)
    for n in names:
        if n in ("spgpe_strerror", "spgpe_last_cuda_error"):
            continue
        assert callable(getattr(sp, n)), f"binding lacks {n}"


def test_no_device_is_an_error_code_not_a_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2010_15069_b200 as sp
    with pytest.raises(sp.SpgpeError) as e:
        sp.spgpe_create(64, 64, 1.0, 1.0)
    assert e.value.code in (-5, -4)
    assert sp.lib().spgpe_strerror(-2).decode().startswith("unsupported")


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2010_15069_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "oracle/" not in text.replace("shares nothing with oracle/", "").replace("Shares nothing with oracle/", ""), f
