"""CPU-side checks of the C-ABI boundary (include/wd.h): the library builds for sm_100a, loads,
exports every declared symbol, and its host-only entry points validate their arguments.
No compute call is made here (no GPU in this container)."""
import ctypes
import os
import re

import pytest

from paper_0912_2186_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "wd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(wd_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree():
    assert declared_symbols() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), name


def test_library_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", binding.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_create_lattice_and_queries(lib):
    lat = binding.wd_create_lattice((4, 6, 2, 3))
    assert binding.wd_lattice_dims(lat) == (4, 6, 2, 3)
    assert binding.wd_lattice_volume(lat) == 144
    # native buffers pad the volume to a multiple of 32 sites (144 -> 160)
    assert binding.wd_spinor_bytes(lat, 1, 32) == 160 * 24 * 4
    assert binding.wd_spinor_bytes(lat, 24, 64) == 24 * 160 * 24 * 8
    assert binding.wd_spinor_bytes(lat, 0, 32) == 0
    assert binding.wd_spinor_bytes(lat, 1, 16) == 52 * ((binding.wd_lattice_volume(lat) + 31) // 32 * 32)  # half storage
    binding.wd_destroy(lat)
    binding.wd_destroy(None)  # NULL destroy is a no-op
    binding.wd_destroy_gauge(None)


@pytest.mark.parametrize("dims", [(0, 4, 4, 4), (4, -1, 4, 4), (4, 4, 4, 0)])
def test_create_lattice_rejects_bad_extents(lib, dims):
    with pytest.raises(binding.WdError) as e:
        binding.wd_create_lattice(dims)
    assert e.value.code == -2
    assert "extents" in binding.wd_last_error()


def test_null_arguments(lib):
    h = ctypes.c_void_p()
    assert lib.wd_create_lattice(None, ctypes.byref(h)) == -1
    assert lib.wd_create_lattice((ctypes.c_int * 4)(4, 4, 4, 4), None) == -1
    d = (ctypes.c_int * 4)(4, 4, 4, 4)
    assert lib.wd_apply(None, None, None, 0.1, d, 1, 32) == -1
    assert lib.wd_apply_host(None, None, None, 0.1, d, 1, 32) == -1
    assert lib.wd_pack_spinor(None, None, None, 1, 32, None) == -1
    assert lib.wd_set_stream(None, None) == -1
    assert lib.wd_set_kernel(None, 0) == -1
    assert lib.wd_lattice_volume(None) == -1


def test_load_gauge_validates_before_touching_the_device(lib):
    lat = binding.wd_create_lattice((4, 4, 4, 4))
    h = ctypes.c_void_p()
    fake = ctypes.c_void_p(0x1000)
    assert lib.wd_load_gauge(lat, fake, 24, 18, None, ctypes.byref(h)) == -3   # (16 = half storage, 32, 64 are valid)
    assert lib.wd_load_gauge(lat, fake, 32, 10, None, ctypes.byref(h)) == -4   # (18, 12, 8 are valid)
    assert lib.wd_load_gauge(lat, None, 32, 18, None, ctypes.byref(h)) == -1
    assert not h.value
    binding.wd_destroy(lat)


def test_no_cpu_fallback_without_a_device(lib):
    """Without a CUDA device wd_load_gauge must fail with WD_ERR_CUDA/ALLOC -- never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lat = binding.wd_create_lattice((4, 4, 4, 4))
    h = ctypes.c_void_p()
    rc = lib.wd_load_gauge(lat, ctypes.c_void_p(0x1000), 32, 18, None, ctypes.byref(h))
    assert rc in (-8, -9)
    assert not h.value
    binding.wd_destroy(lat)


def test_product_does_not_import_the_oracle():
    """The product path and the oracle share no code and neither imports the other."""
    pkg = os.path.join(ROOT, "paper_0912_2186_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith(".py"):
                for line in open(os.path.join(dirpath, f)):
                    assert not re.match(r"\s*(from|import)\s+.*oracle", line), (f, line)
            if f.endswith((".cu", ".cuh", ".h")):
                for line in open(os.path.join(dirpath, f)):
                    assert not re.match(r"\s*#\s*include.*oracle", line), (f, line)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            for line in open(os.path.join(ROOT, "oracle", f)):
                assert not re.match(r"\s*(from|import)\s+.*paper_0912_2186_b200", line), (f, line)
        if f.endswith(".c"):
            for line in open(os.path.join(ROOT, "oracle", f)):
                assert not re.match(r"\s*#\s*include\s*\"", line), (f, line)
