"""-m "not gpu": the C-ABI library builds, loads, and exports every symbol include/mt.h declares
(no compute call is made without a GPU)."""
import ctypes
import os
import re

from paper_2107_05364_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mt_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_four_north_star_calls():
    syms = declared_symbols()
    for name in ("mt_assemble_tensor", "mt_demag_field", "mt_llg_rhs", "mt_integrate"):
        assert name in syms


def test_library_builds_and_exports_every_declared_symbol():
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in mt.h but not exported"
    assert set(declared_symbols()) == set(binding.EXPORTS)
    lib.mt_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.mt_version()


def test_library_carries_sm100a_code():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_binding_struct_layouts_match_header_sizes():
    # mt_tiles: int64 + 5 pointers; mt_problem and friends are plain C structs with natural alignment
    assert ctypes.sizeof(binding._Tiles) == 8 + 5 * 8
    assert ctypes.sizeof(binding._Opts) == 80
    assert ctypes.sizeof(binding._Result) == 56
    assert ctypes.sizeof(binding._Problem) == 8 + 8 + 8 + 8 + 8 + 8 + 24 + 16 + 16 + 8 + 24 + 8 + 24 + 16 + 8 + 8 + 8 + 8
    assert ctypes.sizeof(binding._Shard) == 4 + 4 + 8 + 8 + 8 + 8 + 8  # rank, world, slice_pad, pack, scal, exchange, user
    assert ctypes.sizeof(binding._Sym) == 24
    assert ctypes.sizeof(binding._SelectState) == 64  # int, double, int, 3 x u64, int, double (8-byte aligned)
    assert ctypes.sizeof(binding._Sparse) == 8 + 8 + 8 + 8 + 5 * 8  # int dtype padded to 8; + cols16, panel_ptr


def test_no_cpu_fallback_without_device():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.MtError):
        binding.mt_create(0)
    # and the raw entry point reports MT_ERR_CUDA rather than computing anything
    lib = binding.load()
    h = ctypes.c_void_p()
    assert lib.mt_create(ctypes.byref(h), 0, None) == binding.MT_ERR_CUDA
