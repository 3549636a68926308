"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/lq.h declares; the binding refuses to run without a device (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1911_07045_b200 import build, binding
    build.build()
    return binding.load()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "lq.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lq_[a-zA-Z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(lib):
    from paper_1911_07045_b200 import binding
    declared = _declared_symbols()
    assert len(declared) >= 15
    raw = ctypes.CDLL(binding.lib_path())
    for name in declared:
        assert hasattr(raw, name), "liblq.so does not export %s" % name
    assert sorted(binding.SYMBOLS) == declared        # the binding covers exactly the header
    for name in declared:
        assert callable(getattr(binding, name)), "binding lacks %s" % name


def test_version_and_struct_sizes(lib):
    from paper_1911_07045_b200 import binding
    assert binding.lq_version().startswith("lq ") and "sm_100a" in binding.lq_version()
    assert ctypes.sizeof(binding.lq_fire_params) == 6 * 8 + 3 * 4 + 4     # 6 doubles + 3 ints, padded to 8
    assert ctypes.sizeof(binding.lq_fire_report) == 8 + 8 + 6 * 8 + 2 * 8 + 8


def test_no_cpu_fallback(lib):
    """without a CUDA device lq_create must fail loudly (LQ_ERR_CUDA), never compute on the host"""
    import torch
    from paper_1911_07045_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.LqError) as ei:
        binding.lq_create(8, 8, 8, -0.172, -2.12, 1.73, 2.32)
    assert ei.value.code == binding.LQ_ERR_CUDA
    assert "no CPU fallback" in str(ei.value) or "CUDA" in str(ei.value)


def test_bad_arguments_rejected_before_any_device_work(lib):
    from paper_1911_07045_b200 import binding
    for dims in ((3, 8, 8), (8, 2, 8), (8, 8, 0)):
        with pytest.raises(binding.LqError) as ei:
            binding.lq_create(*dims, -0.172, -2.12, 1.73, 2.32)
        assert ei.value.code == binding.LQ_ERR_ARG
    with pytest.raises(binding.LqError) as ei:       # C <= 0
        binding.lq_create(8, 8, 8, -0.172, -2.12, 0.0, 2.32)
    assert ei.value.code == binding.LQ_ERR_ARG
    with pytest.raises(binding.LqError) as ei:       # B^2 - 24AC < 0: no nematic minimum
        binding.lq_create(8, 8, 8, 1.0, -0.1, 1.0, 2.32)
    assert ei.value.code == binding.LQ_ERR_ARG


def test_product_does_not_import_oracle():
    """the product path must not reach into oracle/ (or _work/)"""
    pkg = os.path.join(ROOT, "paper_1911_07045_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), fn
                assert "lq_oracle" not in txt and "_work" not in txt, fn


def test_workloads_hold_no_method_arithmetic():
    """seeded generators: shapes, masks, anchoring records, initial Q -- and q0 as stored data"""
    from paper_1911_07045_b200 import workloads as wl
    c = wl.make_config("1")
    assert c["q"].shape == (5, 32 ** 3) and c["mask"] is None
    n2 = c["q"][0] + c["q"][3]                       # -Qzz = q0 (1/3 - nz^2) in [-2/3 q0, q0/3]
    assert n2.max() <= wl.Q0_5CB / 3 + 1e-12 and n2.min() >= -2 * wl.Q0_5CB / 3 - 1e-12
    c2 = wl.make_config("1")
    assert np.array_equal(c["q"], c2["q"])           # seeded: identical on every call
    r = wl.make_replica("5p")
    assert set(np.unique(r["kind"])) == {0, 1, 2}
