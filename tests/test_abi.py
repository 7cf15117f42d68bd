"""Boundary checks that need no GPU: libfd6.so loads, exports every symbol include/fd6.h declares, and
validates its arguments before touching CUDA.  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fd6():
    from paper_1707_08900_b200 import build
    build.build()
    from paper_1707_08900_b200 import fd6 as mod
    return mod


def declared_functions(header="fd6.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fd_[a-z0-9_]+)\s*\(", src)) - {"fd_alloc_fn", "fd_free_fn"})


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for must in ("fd_create", "fd_load", "fd_store", "fd_rhs", "fd_rk3_step", "fd_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(fd6):
    for name in declared_functions():
        assert hasattr(fd6.lib, name), f"libfd6.so does not export {name}"
    assert sorted(fd6.EXPORTS) == declared_functions()


def test_test_hooks_live_in_their_own_header(fd6):
    """include/fd6.h is the product ABI; the NaN-poison hooks are declared in include/fd6_testing.h only."""
    from paper_1707_08900_b200 import fd6_testing
    hooks = declared_functions("fd6_testing.h")
    assert hooks == sorted(fd6_testing.TEST_EXPORTS) and hooks
    assert not set(hooks) & set(declared_functions())
    assert not any("debug" in n for n in declared_functions())
    for name in hooks:
        assert hasattr(fd6.lib, name), f"libfd6.so does not export {name}"


def test_every_dynamic_fd_symbol_is_declared_in_a_header(fd6):
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", os.path.join(ROOT, "paper_1707_08900_b200", "libfd6.so")],
                         capture_output=True, text=True).stdout
    syms = sorted({ln.split()[-1] for ln in out.splitlines() if ln.split() and ln.split()[-1].startswith("fd_")})
    assert syms == sorted(declared_functions() + declared_functions("fd6_testing.h"))


def test_library_does_not_link_torch_or_the_oracle(fd6):
    import subprocess
    out = subprocess.run(["ldd", os.path.join(ROOT, "paper_1707_08900_b200", "libfd6.so")], capture_output=True, text=True).stdout
    assert "torch" not in out and "c10" not in out and "fd_oracle" not in out


def test_product_sources_never_reference_the_oracle():
    pkg = os.path.join(ROOT, "paper_1707_08900_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "fd_oracle" not in text and "from oracle" not in text and "import oracle" not in text, f


def test_argument_validation_happens_before_any_cuda_call(fd6):
    h = C.c_void_p()
    L = fd6.lib
    assert L.fd_create(None, 32, 32, 32, 0.1, 0.0, 1.0, fd6.FD_F32) == fd6.FD_EINVAL
    assert L.fd_create(C.byref(h), 4, 32, 32, 0.1, 0.0, 1.0, fd6.FD_F32) == fd6.FD_EINVAL
    assert b"n >= 8" in L.fd_last_error()
    assert L.fd_create(C.byref(h), 32, 32, 7, 0.1, 0.0, 1.0, fd6.FD_F32) == fd6.FD_EINVAL
    assert L.fd_create(C.byref(h), 32, 32, 32, 0.0, 0.0, 1.0, fd6.FD_F32) == fd6.FD_EINVAL
    assert L.fd_create(C.byref(h), 32, 32, 32, float("nan"), 0.0, 1.0, fd6.FD_F32) == fd6.FD_EINVAL
    assert L.fd_create(C.byref(h), 32, 32, 32, 0.1, -1.0, 1.0, fd6.FD_F32) == fd6.FD_EINVAL
    assert L.fd_create(C.byref(h), 32, 32, 32, 0.1, 0.0, -1.0, fd6.FD_F32) == fd6.FD_EINVAL
    assert L.fd_create(C.byref(h), 32, 32, 32, 0.1, 0.0, 1.0, 7) == fd6.FD_EINVAL
    assert L.fd_create(C.byref(h), 30, 32, 32, 0.1, 0.0, 1.0, fd6.FD_F32) == fd6.FD_EUNSUPPORTED
    # launch-grid limits (rows in gridDim.y, (field, plane) in gridDim.z): refused up front, not at the first launch
    assert L.fd_create(C.byref(h), 32, 70000, 8, 0.1, 0.0, 1.0, fd6.FD_F64) == fd6.FD_EUNSUPPORTED
    assert L.fd_create(C.byref(h), 32, 8, 16384, 0.1, 0.0, 1.0, fd6.FD_F64) == fd6.FD_EUNSUPPORTED
    assert b"launch-grid" in L.fd_last_error()
    assert L.fd_set_tile_shape(None, 0) == fd6.FD_EINVAL and L.fd_set_graphs(None, 1) == fd6.FD_EINVAL
    assert h.value is None
    # NULL context
    assert L.fd_rk3_step(None, 0.1, 1) == fd6.FD_EINVAL
    assert L.fd_load(None, None, None, None, None, 0) == fd6.FD_EINVAL
    assert L.fd_set_path(None, 0) == fd6.FD_EINVAL
    assert L.fd_destroy(None) == fd6.FD_OK
    assert L.fd_kernel_launches(None) == 0
    assert L.fd_set_forcing(None, None, None, 0.0, 0.0, 1.0) == fd6.FD_EINVAL


def test_fd_rhs_static_validates_before_any_cuda_call(fd6):
    """The no-allocation entry point checks pointers, parameters and the size limit of its built-in array first."""
    L = fd6.lib
    p = C.c_void_p(256)  # never dereferenced: every call below fails on its arguments
    ok = [p] * 8
    assert L.fd_rhs_static(32, 32, 32, 0.1, 0.0, 1.0, fd6.FD_F32, None, p, p, p, p, p, p, p, None) == fd6.FD_EINVAL
    assert L.fd_rhs_static(32, 32, 32, 0.1, 0.0, 1.0, fd6.FD_F32, p, p, p, p, p, p, p, None, None) == fd6.FD_EINVAL
    assert L.fd_rhs_static(32, 4, 32, 0.1, 0.0, 1.0, fd6.FD_F32, *ok, None) == fd6.FD_EINVAL
    assert L.fd_rhs_static(32, 32, 32, -0.1, 0.0, 1.0, fd6.FD_F32, *ok, None) == fd6.FD_EINVAL
    assert L.fd_rhs_static(32, 32, 32, 0.1, float("nan"), 1.0, fd6.FD_F32, *ok, None) == fd6.FD_EINVAL
    assert L.fd_rhs_static(32, 32, 32, 0.1, 0.0, 1.0, 2, *ok, None) == fd6.FD_EINVAL
    assert L.fd_rhs_static(30, 32, 32, 0.1, 0.0, 1.0, fd6.FD_F32, *ok, None) == fd6.FD_EUNSUPPORTED
    # the limit: 64^3 fp32 and 48^3 fp64 fit the 8 MiB array (run on the GPU in tests/test_zz_no_alloc.py); these do not
    for shape, dtype in (((64, 64, 64), fd6.FD_F64), ((128, 128, 128), fd6.FD_F32), ((2**30, 2**30, 2**30), fd6.FD_F32)):
        assert L.fd_rhs_static(*shape, 0.1, 0.0, 1.0, dtype, *ok, None) == fd6.FD_EUNSUPPORTED
        msg = L.fd_last_error().decode()
        assert "built-in scratch" in msg and str(fd6.FD_RHS_STATIC_MAX_BYTES) in msg
    header = open(os.path.join(ROOT, "include", "fd6.h")).read()
    assert re.search(r"#define\s+FD_RHS_STATIC_MAX_BYTES\s+\(8u \* 1024u \* 1024u\)", header)
    assert fd6.FD_RHS_STATIC_MAX_BYTES == 8 * 1024 * 1024


def test_no_cpu_fallback_without_a_device(fd6):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    assert fd6.lib.fd_create(C.byref(h), 32, 32, 32, 0.1, 0.0, 1.0, fd6.FD_F32) == fd6.FD_ECUDA
    assert b"no CPU fallback" in fd6.lib.fd_last_error()
    with pytest.raises(fd6.FdError):
        fd6.Fd(32, 32, 32, 0.1, 0.0, 1.0)


def _items(wl):
    """Enumerate (tile, plane range) of every launch-grid item exactly as fd6.h documents it."""
    tiles = wl.tiles_x * wl.tiles_y
    for b in range(wl.items):
        if wl.split_plane > 0:
            yield (b, 0, wl.split_plane) if b < tiles else (b - tiles, wl.split_plane, wl.planes)
        elif b < wl.full_tiles:
            yield b, 0, wl.planes
        else:
            j = b - wl.full_tiles
            zs = (j % wl.chunks) * wl.chunk_planes
            yield wl.full_tiles + j // wl.chunks, zs, min(zs + wl.chunk_planes, wl.planes)


@pytest.mark.parametrize("shape", [(512, 512, 512), (256, 256, 256), (128, 128, 128), (32, 32, 32), (1024, 1024, 1024),
                                   (40, 13, 9), (8, 8, 8), (132, 70, 20), (72, 33, 41), (512, 96, 30), (2048, 8, 8)])
@pytest.mark.parametrize("dtype", [0, 1])
@pytest.mark.parametrize("sms", [148, 1, 132, 7])
def test_work_list_covers_every_tile_plane_exactly_once(fd6, shape, dtype, sms):
    nx, ny, nz = shape
    wl = fd6.fd_plan_work_list(nx, ny, nz, dtype, sms)
    tiles = wl.tiles_x * wl.tiles_y
    assert wl.tiles_x * wl.tile_x >= nx > (wl.tiles_x - 1) * wl.tile_x
    assert wl.tiles_y * wl.tile_y >= ny > (wl.tiles_y - 1) * wl.tile_y
    paired = dtype == 0 and nz % 2 == 0
    assert wl.planes == (nz // 2 if paired else nz)
    if wl.split_plane > 0:  # every tile cut once, the long part first
        assert wl.items == 2 * tiles and wl.full_tiles == 0 and wl.planes / 2 <= wl.split_plane <= wl.planes - 2
    else:
        assert wl.full_tiles % sms == 0 and 0 <= tiles - wl.full_tiles < sms
        assert wl.items == wl.full_tiles + (tiles - wl.full_tiles) * wl.chunks
    covered = [0] * (tiles * wl.planes)
    for tile, zs, ze in _items(wl):
        assert 0 <= tile < tiles
        for z in range(zs, ze):  # an empty range (zs >= ze) is an item that returns at once
            covered[tile * wl.planes + z] += 1
    assert min(covered) == 1 and max(covered) == 1


def test_work_list_of_the_headline_config(fd6):
    wl = fd6.fd_plan_work_list(512, 512, 512, fd6.FD_F32, 148)
    # enough tiles for the tall shape: 16 x 32 tiles of 32 x 16 pairs; three full waves of columns, the remaining 68
    # tiles cut in z
    assert (wl.tile_x, wl.tile_y, wl.tiles_x, wl.tiles_y, wl.planes, wl.full_tiles) == (32, 16, 16, 32, 256, 444)
    assert wl.chunks >= 2 and wl.items == 444 + 68 * wl.chunks
    # a grid with few tiles keeps the wide shape (32 x 12 values): more, smaller work items
    wl = fd6.fd_plan_work_list(128, 128, 128, fd6.FD_F32, 148)
    assert (wl.tile_x, wl.tile_y, wl.tiles_x, wl.tiles_y, wl.planes) == (32, 12, 4, 11, 64)
    wl = fd6.fd_plan_work_list(256, 256, 256, fd6.FD_F64, 148)
    assert (wl.tile_x, wl.tile_y, wl.tiles_x, wl.tiles_y, wl.planes) == (32, 16, 8, 16, 256)
    # C3: 128 tiles on 148 SMs.  Full columns would leave 20 SMs idle for the whole launch (266 plane-times with the
    # warm-up); the split list gives every SM work: 128 long parts, and the 128 short parts packed 6-7 deep on 20 SMs
    assert wl.split_plane > 0 and wl.items == 256 and wl.full_tiles == 0
    long_cost, short_cost = wl.split_plane + 10, wl.planes - wl.split_plane + 10
    assert max(long_cost, 7 * short_cost) <= 245


def test_work_list_cuts_thin_grids_into_short_chunks(fd6):
    """Few tiles and few stored planes: the remainder is cut down to chunks of a few planes (>= 2) so that its items fill
    the SMs, in the paired layout too (round 1 capped the chunk count at planes / 8)."""
    wl = fd6.fd_plan_work_list(132, 70, 20, fd6.FD_F32, 148)   # paired: 10 stored planes, 5 x 6 tiles
    assert (wl.planes, wl.tiles_x * wl.tiles_y, wl.full_tiles) == (10, 30, 0)
    assert wl.chunks >= 3 and 2 <= wl.chunk_planes <= 4 and wl.items <= 148
    wl = fd6.fd_plan_work_list(2048, 100, 9, fd6.FD_F32, 148)  # plain fp32 (odd nz): 32 x 24 cells per tile
    assert (wl.tile_x, wl.tile_y, wl.planes) == (32, 24, 9) and wl.chunks >= 2
    wl = fd6.fd_plan_work_list(64, 64, 64, fd6.FD_F32, 148)
    assert wl.chunks >= 8 and wl.chunk_planes >= 2


def test_work_list_rejects_bad_arguments(fd6):
    wl = fd6.FdWorkList()
    assert fd6.lib.fd_plan_work_list(512, 512, 512, 0, 148, None) == fd6.FD_EINVAL
    assert fd6.lib.fd_plan_work_list(4, 512, 512, 0, 148, C.byref(wl)) == fd6.FD_EINVAL
    assert fd6.lib.fd_plan_work_list(512, 512, 512, 0, 0, C.byref(wl)) == fd6.FD_EINVAL
    assert fd6.lib.fd_plan_work_list(512, 512, 512, 5, 148, C.byref(wl)) == fd6.FD_EINVAL
