"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/kf.h declares (no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "kf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kf_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_path():
    syms = declared_symbols()
    for s in ("kf_fit", "kf_bin_hits", "kf_window_lookup", "kf_build", "kf_last_error", "kf_version"):
        assert s in syms


def test_library_builds_loads_and_exports_every_symbol():
    from paper_1711_06571_b200 import build_ext, binding
    so = build_ext.build()
    lib = ctypes.CDLL(so)
    for s in declared_symbols():
        assert hasattr(lib, s), s
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert binding.kf_version() >= 100
    assert binding.lib().kf_last_error() is not None


def test_product_path_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1711_06571_b200 import binding
    with pytest.raises(binding.KfError):
        binding.kf_fit(None, None, None, None, None)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1711_06571_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "kf_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1711_06571_b200\.(binding|build_ext)", txt, flags=re.M), f
            assert "libkf_b200" not in txt and '#include "kf' not in txt and "csrc/" not in txt.replace("paper_1711_06571_b200/csrc/ and", ""), f
