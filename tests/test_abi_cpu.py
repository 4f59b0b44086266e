"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/bls.h declares; structural errors are reported without a GPU; there is no CPU fallback."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bls():
    from paper_1112_1701_b200 import build
    build.build()
    import paper_1112_1701_b200 as b
    return b


def test_every_declared_symbol_is_exported(bls):
    hdr = open(os.path.join(ROOT, "include", "bls.h")).read()
    declared = set(re.findall(r"^(?:int|const char \*)\s*\*?(bls_\w+)\s*\(", hdr, flags=re.M))
    assert declared == set(bls.EXPORTS), (declared, bls.EXPORTS)
    L = bls.lib()
    for name in declared:
        assert getattr(L, name) is not None


def test_struct_layouts_match_header(bls):
    assert bls.PEAK_DTYPE.itemsize == 32
    assert bls.PEAK_DTYPE.fields["freq"][1] == 16 and bls.PEAK_DTYPE.fields["epoch"][1] == 24
    assert C.sizeof(bls.binding.BlsConfig) == 88      # gcc sizeof(bls_config) on x86-64
    assert C.sizeof(bls.binding.BlsBatch) == 48
    assert C.sizeof(bls.binding.BlsOutputs) == 40


def test_strerror_and_null_handling(bls):
    L = bls.lib()
    assert L.bls_strerror(0) == b"ok"
    assert b"NULL" in L.bls_strerror(-1)
    assert L.bls_plan_destroy(None) == 0
    assert L.bls_plan_create(None, None) == bls.binding.BLS_ERR_NULL
    v = C.c_int64()
    assert L.bls_plan_query(None, 1, C.byref(v)) == bls.binding.BLS_ERR_NULL


@pytest.mark.parametrize("kw", [dict(n_bins=2), dict(n_bins=5000), dict(q_min=0.0), dict(q_max=0.7),
                                dict(q_min=0.2, q_max=0.1), dict(max_top_k=0), dict(max_top_k=33),
                                dict(n_freq=0), dict(f0=-1.0), dict(freqs=np.array([1.0, np.nan]))])
def test_bad_config_is_rejected_before_any_cuda_call(bls, kw):
    base = dict(n_bins=100, q_min=0.01, q_max=0.1, n_freq=10, f0=0.1, df=0.1, max_top_k=5)
    base.update(kw)
    if "freqs" in kw:
        base.pop("n_freq")
    with pytest.raises(bls.BlsError) as e:
        bls.Plan(**base)
    assert e.value.code == bls.binding.BLS_ERR_CONFIG


def test_no_cpu_fallback(bls):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(bls.BlsError) as e:
        bls.Plan(n_bins=100, q_min=0.01, q_max=0.1, n_freq=10, f0=0.1, df=0.1)
    assert e.value.code == bls.binding.BLS_ERR_CUDA


def test_product_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1112_1701_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), fn
                assert "bls_oracle" not in src, fn
    osrc = open(os.path.join(ROOT, "oracle", "bls_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_1112_1701_b200" not in osrc.replace("paper_1112_1701_b200/", "")  # mentions only in prose
    assert "#include \"../" not in osrc and "bls.h" not in osrc
