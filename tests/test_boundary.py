"""Host-side checks of the C-ABI boundary -- CPU only (no compute calls without a GPU)."""
import ctypes
import os
import re

import pytest

from paper_1808_01309_b200 import build as psbuild
from paper_1808_01309_b200 import psfft

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    psbuild.build_library()
    return psfft.lib()


def test_library_exports_every_declared_symbol(lib):
    """Every function include/psfft.h declares is exported by libpsfft.so, and the binding names them all."""
    hdr = open(os.path.join(ROOT, "include", "psfft.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(psfft_[a-z0-9_]+)\s*\(", hdr)))
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(psfft.EXPORTS) == declared


def test_plan_query_sizes(lib):
    lay = psfft.plan_query(512, psfft.F64, 3)
    assert (lay.N, lay.ldk, lay.batch) == (512, 257, 3)
    assert lay.real_bytes == 1073741824 and lay.spec_bytes == 1077936128      # SURVEY §8 size table
    assert 512 * 16 <= lay.table_bytes <= 4 * 512 * 16 and lay.work_bytes_fft == 3 * lay.spec_bytes
    lay = psfft.plan_query(768, psfft.F32, 1)
    assert lay.ldk == 385 and lay.real_bytes == 1811939328 and lay.spec_bytes == 1816657920
    lay = psfft.plan_query(1024, psfft.F32, 1)
    assert lay.real_bytes == 4294967296 and lay.spec_bytes == 4303355904
    assert lay.work_bytes_mhd + 12 * lay.spec_bytes < 180e9                    # config 5 fits one B200


def test_mask_integers_fit_int32_for_every_supported_grid(lib):
    """DESIGN.md reading G25: the 2/3-rule test 9 sum (n_i L / N_i)^2 < L^2, L = lcm(Nx, Ny, Nz), is evaluated in int32 on
    the device.  For every triple of supported sizes the largest sum, 3 (L/2)^2, must stay below 2^31."""
    import math
    lay = psfft.Layout()
    sizes = [n for n in range(1, 4097) if lib.psfft_plan_query(n, psfft.F32, 1, ctypes.byref(lay)) == 0]
    assert sizes == [8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024, 2048]
    worst = max(math.lcm(a, b, c) for a in sizes for b in sizes for c in sizes)
    assert worst == 6144 and 3 * (worst // 2) ** 2 < 2 ** 31 and (worst * worst + 8) // 9 < 2 ** 31


def test_error_codes(lib):
    lay = psfft.Layout()
    assert lib.psfft_plan_query(500, psfft.F64, 1, ctypes.byref(lay)) == -2     # unsupported N
    assert lib.psfft_plan_query(4096, psfft.F64, 1, ctypes.byref(lay)) == -2
    assert lib.psfft_plan_query(1536, psfft.F64, 1, ctypes.byref(lay)) == -2
    assert lib.psfft_plan_query3(2048, 2048, 512, psfft.F32, 1, ctypes.byref(lay)) == 0 and lay.ldk == 1025
    assert lib.psfft_plan_query(512, 7, 1, ctypes.byref(lay)) == -3
    assert lib.psfft_plan_query(512, psfft.F64, 0, ctypes.byref(lay)) == -2
    assert lib.psfft_plan_query(512, psfft.F64, 1, None) == -1
    h = ctypes.c_void_p()
    assert lib.psfft_plan_create(ctypes.byref(h), 64, psfft.F64, 1, None, 1 << 20, None) == -1
    assert lib.psfft_plan_create(ctypes.byref(h), 64, psfft.F64, 1, ctypes.c_void_p(0x1008), 1 << 20, None) == -4
    assert lib.psfft_plan_create(ctypes.byref(h), 64, psfft.F64, 1, ctypes.c_void_p(0x1000), 8, None) == -5
    assert lib.psfft_plan_destroy(None) == -6
    assert lib.psfft_fft3d_r2c(None, None, None, None, None) == -6
    assert lib.psfft_plan_query(1024, psfft.F64, 64, ctypes.byref(lay)) == -7   # batch * Nz > 65535 (y-pass grid)
    assert lib.psfft_plan_query(1024, psfft.F64, 63, ctypes.byref(lay)) == 0
    for code in (0, -1, -2, -3, -4, -5, -6, -7, -8, -9):
        assert psfft.strerror(code)
    assert "overlap" in psfft.strerror(-8)
    assert "psfft" in psfft.strerror(-2)
    with pytest.raises(psfft.PsfftError):
        psfft.plan_query(10, psfft.F64, 1)
    assert psfft.version() == "0.1"


def test_stale_and_invented_handles_are_rejected_without_dereferencing(lib):
    """Handles are looked up in the library's registry of live plans: an address that was never a plan (here:
    unmapped memory, which a read of a magic word would fault on) is answered with PSFFT_E_PLAN."""
    lay = psfft.Layout()
    for bogus in (0x10, 0xDEAD0000, 0x7FFFFFFFF000):
        assert lib.psfft_plan_layout(ctypes.c_void_p(bogus), ctypes.byref(lay)) == -6
        assert lib.psfft_plan_destroy(ctypes.c_void_p(bogus)) == -6
        assert lib.psfft_hd_rhs(ctypes.c_void_p(bogus), None, None, 0.0, None, None) == -6
        assert lib.psfft_last_launch_count(ctypes.c_void_p(bogus)) == -6


def test_every_supported_size_is_accepted(lib):
    for N in (8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024):
        for dt in (psfft.F32, psfft.F64):
            lay = psfft.plan_query(N, dt, 2)
            assert lay.ldk == N // 2 + 1 and lay.spec_elems == lay.ldk * N * N


def test_product_never_imports_the_oracle():
    """The CUDA path and its binding may not import, read or run anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1808_01309_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "psfft_oracle" not in src and "liboracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "psfft_oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_1808_01309_b200", osrc, flags=re.M)
    assert "psfft.h" not in osrc and "csrc" not in osrc.replace("paper_1808_01309_b200/csrc/", "")


def test_plan_query3_anisotropic_sizes(lib):
    """Anisotropic plans (PAPER.md:370 runs 1024 x 1024 x 256): sizes per axis; RHS workspace = 11 (HD) / 16
    (Boussinesq) compact fields [Nz][Ny][kx pitch] whose pitch is the retained kx count of Nx rounded up to a tile."""
    lay = psfft.plan_query3(1024, 1024, 256, psfft.F32, 1)
    assert (lay.N, lay.Ny, lay.Nz, lay.ldk) == (1024, 1024, 256, 513)
    assert lay.real_elems == 1024 * 1024 * 256 and lay.spec_elems == 513 * 1024 * 256
    assert lay.work_bytes_fft == lay.spec_bytes
    pitch = lay.work_bytes_hd // (11 * 256 * 1024 * 8)
    assert lay.work_bytes_hd == 11 * 256 * 1024 * pitch * 8 and 342 <= pitch <= 342 + 32 and pitch % 16 == 0
    assert lay.work_bytes_boussinesq * 11 == lay.work_bytes_hd * 16 and lay.work_bytes_mhd == 2 * lay.work_bytes_hd
    cub = psfft.plan_query3(512, 512, 512, psfft.F64, 3)
    ref = psfft.plan_query(512, psfft.F64, 3)
    assert (cub.table_bytes, cub.work_bytes_hd, cub.Ny, cub.Nz) == (ref.table_bytes, ref.work_bytes_hd, 512, 512)
    assert psfft.plan_query3(64, 64, 16, psfft.F64, 1).table_bytes > psfft.plan_query3(64, 64, 64, psfft.F64, 1).table_bytes - 16 * 64
    bad = psfft.Layout()
    assert lib.psfft_plan_query3(512, 500, 512, psfft.F64, 1, ctypes.byref(bad)) == -2
