"""CPU-side checks of the boundary: the C-ABI library loads without a GPU and exports every symbol that
include/rflbm.h declares; host-only argument validation (no compute calls)."""
import ctypes as C
import os
import re

import pytest

from paper_2507_08820_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "rflbm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rflbm_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_all_exported_and_bound(lib):
    names = declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.SYMBOLS) == names


def test_create_validation_and_workspace_size(lib):
    h = C.c_void_p()
    bad = [(0, 4, 4, 1.0, 0.0, 1.0), (4, 4, 4, 0.5, 0.0, 1.0), (4, 4, 4, float("nan"), 0.0, 1.0),
           (4, 4, 4, 1.0, -1e-9, 1.0), (4, 4, 4, 1.0, 0.0, 0.0), (2048, 2048, 2048, 1.0, 0.0, 1.0)]
    for nx, ny, nz, tau, kT, rho0 in bad:
        assert lib.rflbm_create(nx, ny, nz, tau, kT, rho0, 0, binding.F64, C.byref(h)) == binding.EINVAL
    assert lib.rflbm_create(4, 4, 4, 1.0, 0.0, 1.0, 0, 5, C.byref(h)) == binding.EINVAL
    assert lib.rflbm_create(4, 4, 4, 1.0, 0.0, 1.0, 0, binding.F64, None) == binding.EINVAL
    assert lib.rflbm_create(16, 16, 16, 1.0, 1e-4, 1.0, 42, binding.F64, C.byref(h)) == binding.OK
    assert lib.rflbm_workspace_bytes(h) == 2 * 27 * 4096 * 8 + 4096 + 12288
    # state machine, host side only
    assert lib.rflbm_step(h, 1) == binding.ESTATE
    assert b"before init" in lib.rflbm_last_error(h)
    assert lib.rflbm_init(h, None, None) == binding.ESTATE
    assert lib.rflbm_set_workspace(h, 0x1000, 16) == binding.ENOMEM
    assert lib.rflbm_set_workspace(h, 0x1001, 1 << 30) == binding.ENOMEM      # misaligned
    assert lib.rflbm_set_force(h, float("inf"), 0.0, 0.0) == binding.EINVAL
    assert lib.rflbm_set_scheme(h, 7) == binding.EINVAL
    assert lib.rflbm_set_scheme(h, binding.SCHEME_AA) == binding.OK
    assert lib.rflbm_workspace_bytes(h) == 27 * 4096 * 8 + 4096 + 12288          # one buffer
    assert lib.rflbm_set_scheme(h, binding.SCHEME_AB) == binding.OK
    assert lib.rflbm_set_model(h, 9) == binding.EINVAL and lib.rflbm_set_model(h, binding.MODEL_BGK) == binding.OK
    assert lib.rflbm_set_force(h, 1e-6, 0.0, 0.0) == binding.EINVAL              # BGK-FLBM carries no force
    assert lib.rflbm_set_model(h, binding.MODEL_REG) == binding.OK
    assert lib.rflbm_step_count(h) == 0 and lib.rflbm_launch_count(h) == 0
    assert lib.rflbm_destroy(h) == binding.OK
    h32 = C.c_void_p()
    assert lib.rflbm_create(4, 4, 2, 1.0, 0.0, 1.0, 0, binding.F32, C.byref(h32)) == binding.OK
    assert lib.rflbm_workspace_bytes(h32) == 2 * 3584 + 4096 + 12288                  # 27*32*4 = 3456 -> 256-aligned 3584
    assert lib.rflbm_set_walls_z(h32, 1) == binding.EINVAL                     # nz < 3
    lib.rflbm_destroy(h32)


def test_slab_and_grid_validation_host_side(lib):
    """rflbm_set_slab / halo argument checks and the launch-grid limits of rflbm_create: host only, no GPU work."""
    h = C.c_void_p()
    # padded row pitch: nx = 33 fp64 rows are 48 elements (whole 128-byte lines), slab adds two ghost layers
    assert lib.rflbm_create(33, 4, 5, 1.0, 1e-4, 1.0, 0, binding.F64, C.byref(h)) == binding.OK
    plain = lib.rflbm_workspace_bytes(h)
    assert plain == 2 * 27 * (48 * 4 * 5) * 8 + 4096 + 12288
    assert lib.rflbm_halo_bytes(h) == 9 * 33 * 4 * 8
    assert lib.rflbm_halo_pending(h) == 0
    assert lib.rflbm_halo_pack(h, binding.SIDE_LOW, 0x1000) == binding.ESTATE          # not in slab mode
    assert lib.rflbm_set_slab(h, -1, 20) == binding.EINVAL
    assert lib.rflbm_set_slab(h, 16, 20) == binding.EINVAL                                # [16, 21) does not fit
    assert lib.rflbm_set_slab(h, 0, 1 << 30) == binding.EINVAL                            # 2^32 global sites or more
    assert lib.rflbm_workspace_bytes(h) == plain                                          # failed calls change nothing
    assert lib.rflbm_set_slab(h, 15, 20) == binding.OK
    assert lib.rflbm_workspace_bytes(h) == 2 * 27 * (48 * 4 * 7) * 8 + 4096 + 12288
    assert lib.rflbm_halo_pack(h, binding.SIDE_LOW, 0x1000) == binding.ESTATE          # before init
    assert lib.rflbm_halo_pack(h, 2, 0x1000) == binding.EINVAL
    assert lib.rflbm_halo_unpack(h, binding.SIDE_HIGH, None) == binding.EINVAL
    assert lib.rflbm_set_walls_z(h, 1) == binding.OK                                      # walls look at nz_global = 20
    assert lib.rflbm_last_kernel(h) == b""
    lib.rflbm_destroy(h)
    assert lib.rflbm_create(4, 4, 2, 1.0, 0.0, 1.0, 0, binding.F64, C.byref(h)) == binding.OK
    assert lib.rflbm_set_walls_z(h, 1) == binding.EINVAL                                  # nz = 2
    assert lib.rflbm_set_slab(h, 3, 8) == binding.OK
    assert lib.rflbm_set_walls_z(h, 1) == binding.OK                                      # nz_global = 8
    lib.rflbm_destroy(h)
    # gridDim.y <= 65535 blocks: nx >= 128 -> one row per block row; nx = 8 -> 16 rows per block
    assert lib.rflbm_create(128, 70000, 1, 1.0, 0.0, 1.0, 0, binding.F64, C.byref(h)) == binding.EINVAL
    assert lib.rflbm_create(128, 65535, 1, 1.0, 0.0, 1.0, 0, binding.F64, C.byref(h)) == binding.OK
    lib.rflbm_destroy(h)
    assert lib.rflbm_create(8, 70000, 1, 1.0, 0.0, 1.0, 0, binding.F64, C.byref(h)) == binding.OK
    lib.rflbm_destroy(h)
    assert lib.rflbm_create(1, 1, 70000, 1.0, 0.0, 1.0, 0, binding.F64, C.byref(h)) == binding.EINVAL
    # row offsets are 32-bit: 27 x the padded row (nx rounded up by at most 31 elements) must fit an int, i.e.
    # nx <= RFLBM_MAX_NX = INT_MAX/27 - 32.  80 000 000 x 2 x 1 has fewer than 2^32 sites and was accepted before.
    max_nx = (2 ** 31 - 1) // 27 - 32
    hdr = open(os.path.join(ROOT, "include", "rflbm.h")).read()
    assert "#define RFLBM_MAX_NX (2147483647 / 27 - 32)" in hdr
    assert lib.rflbm_create(80_000_000, 2, 1, 1.0, 0.0, 1.0, 0, binding.F64, C.byref(h)) == binding.EINVAL
    assert lib.rflbm_create(max_nx + 1, 1, 1, 1.0, 0.0, 1.0, 0, binding.F32, C.byref(h)) == binding.EINVAL
    for prec in (binding.F64, binding.F32):
        assert lib.rflbm_create(max_nx, 2, 1, 1.0, 0.0, 1.0, 0, prec, C.byref(h)) == binding.OK
        es = 8 if prec == binding.F64 else 4
        line = 128 // es
        px = (max_nx + line - 1) // line * line
        assert 27 * px <= 2 ** 31 - 1                                                 # what Geom::px holds
        assert lib.rflbm_workspace_bytes(h) == 2 * ((27 * px * 2 * es + 255) // 256 * 256) + 4096 + 12288
        lib.rflbm_destroy(h)


def test_no_environment_knobs_in_the_product():
    """the C-ABI's layout and launch shape must not depend on the caller's environment"""
    pkg = os.path.join(ROOT, "paper_2507_08820_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h", ".py")) and f != "build.py":
                s = open(os.path.join(dirpath, f)).read()
                assert "getenv" not in s and "os.environ" not in s, f


def test_binding_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.Rflbm(4, 4, 4, 1.0, 0.0)


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (or read _work/)."""
    pkg = os.path.join(ROOT, "paper_2507_08820_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", s, flags=re.M), f
                assert "rflbm_ref" not in s and "_work/" not in s, f
