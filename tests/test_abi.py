"""The C-ABI library loads and exports every symbol include/cp.h declares (no GPU calls)."""
import os
import re

import pytest

from paper_2606_09061_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "cp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cp_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    syms = declared_symbols()
    assert "cp_build_batch" in syms and "cp_attention_step" in syms and "cp_latency_table" in syms
    assert len(syms) >= 19
    for s in syms:
        assert hasattr(lib, s), f"libcp.so does not export {s}"
    assert sorted(binding.EXPORTS) == syms          # the binding mirrors the header, name for name


def test_struct_sizes_match_the_header(lib):
    import ctypes as C
    assert C.sizeof(binding.cp_req_desc) == 32
    assert C.sizeof(binding.cp_latency_row) == 72
    assert C.sizeof(binding.cp_config) == 88


def test_missing_library_fails_loudly(tmp_path):
    with pytest.raises(ImportError):
        binding.load(str(tmp_path / "libcp.so"))


def test_host_side_argument_errors(lib):
    # no GPU here: only the calls that fail before touching CUDA
    import ctypes as C
    assert lib.cp_create(None, None) == binding.CP_EINVAL
    assert b"null" in lib.cp_last_error()
    cfg = binding.cp_config(32, 5, 128, 16, 1, 1024, 0.1, 128, 8, 1024, 0, 0, 0, 0, 0, 0)
    h = C.c_void_p()
    assert lib.cp_create(C.byref(cfg), C.byref(h)) == binding.CP_EINVAL     # Hq % Hkv
    cfg = binding.cp_config(32, 8, 96, 16, 1, 1024, 0.1, 128, 8, 1024, 0, 0, 0, 0, 0, 0)
    assert lib.cp_create(C.byref(cfg), C.byref(h)) == binding.CP_EINVAL     # head_dim
    assert lib.cp_attention_step(None, 0, None, None, None, None, None, None) == binding.CP_EINVAL
