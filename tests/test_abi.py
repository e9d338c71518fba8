"""-m "not gpu": the C-ABI library loads and exports every symbol include/sdp.h declares; host-side
argument checks that need no device."""
import ctypes
import os
import re

import pytest

import paper_1302_5507_b200 as S
from paper_1302_5507_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "sdp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sdp_[a-z_]+)\s*\(", src)))


def test_header_symbols_exported():
    lib = S.load_library()
    syms = declared_symbols()
    assert set(syms) == set(binding.EXPORTS)
    for s in syms:
        assert hasattr(lib, s), s


def test_version_and_null_arguments():
    lib = S.load_library()
    assert S.sdp_version().startswith("sdp ")
    assert lib.sdp_create(None, 0, None) == binding.SDP_EINVAL
    h = ctypes.c_void_p()
    bad = binding.sdp_scoring(1, 1, 5, 2, 0.6)          # mismatch > 0
    assert lib.sdp_create(ctypes.byref(bad), 0, ctypes.byref(h)) == binding.SDP_EINVAL
    bad = binding.sdp_scoring(1, -3, 5, 0, 0.6)         # gap_extend < 1
    assert lib.sdp_create(ctypes.byref(bad), 0, ctypes.byref(h)) == binding.SDP_EINVAL
    bad = binding.sdp_scoring(1, -3, 5, 2, 1.5)         # min_similarity out of [0,1]
    assert lib.sdp_create(ctypes.byref(bad), 0, ctypes.byref(h)) == binding.SDP_EINVAL
    assert lib.sdp_last_error(None) == b"null context"
    lib.sdp_destroy(None)                               # ignored
    assert lib.sdp_align_batch(None, None, None, None) == binding.SDP_EINVAL


def test_struct_layouts_match_header():
    # sizes the C compiler gives the ABI structs (LP64): guards the ctypes mirror against drift
    assert ctypes.sizeof(binding.sdp_scoring) == 24
    assert ctypes.sizeof(binding.sdp_batch) == 112
    assert ctypes.sizeof(binding.sdp_result) == 104
    assert ctypes.sizeof(binding.sdp_stats) == 88


def test_no_cpu_fallback_without_library(tmp_path):
    with pytest.raises(FileNotFoundError):
        binding.load_library(str(tmp_path / "libsdp.so"))
