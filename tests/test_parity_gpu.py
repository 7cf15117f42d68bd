"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded
inputs.  Bars (BASELINE.json north_star): max relative L-inf <= 1e-12 (fp64), <= 2e-5 (fp32)
after one full RK3 step; each stencil path against the oracle of the SAME path (reading G7); fp32 results
against the DOUBLE oracle on the same fp32-representable inputs (reading G15)."""
import math

import numpy as np
import pytest

from paper_1707_08900_b200 import fd6_testing as T  # include/fd6_testing.h: NaN-poison hooks (tests only)

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}
TWO_PI = 2.0 * math.pi


@pytest.fixture(scope="module")
def mods():
    from oracle import oracle as O
    from paper_1707_08900_b200 import fd6, inputs
    return O, fd6, inputs


def relinf(A, B):
    """reading G14: per field max|A-B| / max|B| (absolute if max|B| == 0), max over fields."""
    worst = 0.0
    for a, b in zip(A, B):
        den = float(np.abs(b).max())
        err = float(np.abs(a.astype(np.float64) - b).max())
        worst = max(worst, err / den if den > 0 else err)
    return worst


def variants(fd6):
    return [fd6.FD_VARIANT_DIRECT, fd6.FD_VARIANT_TILED, fd6.FD_VARIANT_PAIRED]


def make_ctx(fd6, shape_xyz, dx, nu, cs, dtype, path, variant):
    nx, ny, nz = shape_xyz
    ctx = fd6.Fd(nx, ny, nz, dx, nu, cs, fd6.FD_F32 if dtype == "f32" else fd6.FD_F64)
    ctx.fd_set_path(path)
    try:
        ctx.fd_set_variant(variant)
    except fd6.FdError as e:
        if e.code == fd6.FD_EUNSUPPORTED:
            ctx.fd_destroy()
            pytest.skip("variant does not support this grid")
        raise
    return ctx


def smooth_state(rng, shape_xyz, amp, dtype):
    """A few random low-wavenumber modes per field on a (possibly non-cubic) periodic box."""
    nx, ny, nz = shape_xyz
    i = np.arange(nx)[None, None, :] / nx
    j = np.arange(ny)[None, :, None] / ny
    k = np.arange(nz)[:, None, None] / nz
    F = np.zeros((4, nz, ny, nx))
    for q in range(4):
        for _ in range(4):
            kv = rng.integers(-2, 3, 3)
            F[q] += amp * rng.uniform(0.3, 1.0) * np.cos(TWO_PI * (kv[0] * i + kv[1] * j + kv[2] * k) + rng.uniform(0, TWO_PI))
    return F.astype(np.float32 if dtype == "f32" else np.float64)


# ------------------------------------------------------------------ layout: load / store / halo
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("where", ["host", "device"])
def test_load_store_round_trip_is_bit_exact(mods, dtype, where):
    import torch
    O, fd6, I = mods
    rng = np.random.default_rng(1)
    shape = (40, 13, 9)
    F = rng.standard_normal((4, 9, 13, 40)).astype(np.float32 if dtype == "f32" else np.float64)
    ctx = make_ctx(fd6, shape, 0.1, 0.01, 1.0, dtype, fd6.FD_PATH_55, fd6.FD_VARIANT_DIRECT)
    if where == "host":
        ctx.load_state(F)
        out = ctx.store_state()
    else:
        d = torch.from_numpy(F).cuda()
        ctx.load_state(d)
        o = torch.empty_like(d)
        ctx.store_state(o)
        ctx.fd_sync()
        out = o.cpu().numpy()
    assert np.array_equal(out, F)
    assert ctx.fd_kernel_launches() > 0
    ctx.fd_destroy()


# ------------------------------------------------------------ config C1: full grid, both paths
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_c1_one_step_and_rhs_full_grid_fp64(mods, path, variant):
    O, fd6, I = mods
    cfg = I.CONFIGS["C1"]
    F = I.make_state(cfg)
    ctx = make_ctx(fd6, (cfg.n,) * 3, cfg.dx, cfg.nu, cfg.cs, "f64", path, variant)
    ctx.load_state(F)
    R = ctx.rhs_state()
    assert relinf(R, O.rhs(F, cfg.dx, cfg.nu, cfg.cs, path)) <= TOL["f64"]
    assert np.array_equal(ctx.store_state(), F)  # fd_rhs leaves the state untouched
    T.fd_debug_poison_w(ctx)                        # stale w must not matter: alpha^(1) = 0
    ctx.fd_rk3_step(cfg.dt, 1)
    got = ctx.store_state()
    ref = O.rk3_step(F, cfg.dx, cfg.nu, cfg.cs, cfg.dt, 1, path)
    assert relinf(got, ref) <= TOL["f64"]
    ctx.fd_destroy()


# ------------------------------------------- ragged sizes spanning several tiles plus a tail
@pytest.mark.parametrize("shape", [(40, 13, 9), (8, 8, 8), (132, 70, 20), (72, 33, 41), (44, 9, 11)])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_ragged_grids_three_steps(mods, shape, dtype, path, variant):
    O, fd6, I = mods
    rng = np.random.default_rng(shape[0] * 1000 + shape[1] * 10 + path)
    dx, nu, cs = 0.2, 0.02, 1.0
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.1, dtype)
    ctx = make_ctx(fd6, shape, dx, nu, cs, dtype, path, variant)
    T.fd_debug_poison_ghosts(ctx)  # every ghost that is read must have been filled by the library
    ctx.load_state(F)
    ctx.fd_rk3_step(dt, 1)
    one = ctx.store_state()
    ref1 = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 1, path)
    assert relinf(one, ref1) <= TOL[dtype]
    ctx.fd_rk3_step(dt, 2)
    three = ctx.store_state()
    ref3 = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 3, path)
    assert relinf(three, ref3) <= 3 * TOL[dtype]
    ctx.fd_destroy()


# --------------------------------------- config C2 (128^3 fp32): one step, full grid, both paths
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_c2_one_step_full_grid_fp32(mods, path, variant):
    O, fd6, I = mods
    cfg = I.CONFIGS["C2"]
    F = I.make_state(cfg)
    assert F.dtype == np.float32
    ctx = make_ctx(fd6, (cfg.n,) * 3, cfg.dx, cfg.nu, cfg.cs, "f32", path, variant)
    ctx.load_state(F)
    ctx.fd_rk3_step(cfg.dt, 1)
    got = ctx.store_state()
    ref = O.rk3_step(F.astype(np.float64), cfg.dx, cfg.nu, cfg.cs, cfg.dt, 1, path)
    assert relinf(got, ref) <= TOL["f32"]
    ctx.fd_destroy()


# ----------------------------------------------------------- degenerate and invariant cases
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_uniform_state_at_rest_is_a_fixed_point(mods, dtype, path, variant):
    O, fd6, I = mods
    shape = (32, 16, 24)
    F = np.zeros((4, 24, 16, 32), dtype=np.float32 if dtype == "f32" else np.float64)
    F[0] = 0.731
    ctx = make_ctx(fd6, shape, 0.1, 5e-3, 1.0, dtype, path, variant)
    ctx.load_state(F)
    assert np.all(ctx.rhs_state() == 0.0)
    ctx.fd_rk3_step(0.01, 2)
    assert np.array_equal(ctx.store_state(), F)
    ctx.fd_rk3_step(0.01, 0)  # nsteps = 0 is a no-op
    assert np.array_equal(ctx.store_state(), F)
    ctx.fd_destroy()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_periodic_shift_equivariance_is_bitwise(mods, dtype, path, variant):
    """step(roll(F)) == roll(step(F)) bit for bit: no cell's arithmetic may depend on its position in a tile."""
    O, fd6, I = mods
    rng = np.random.default_rng(5)
    shape = (64, 40, 24)
    F = smooth_state(rng, shape, 0.1, dtype)
    sh = (5, 17, 30)
    outs = []
    for G in (F, np.roll(F, sh, (1, 2, 3))):
        ctx = make_ctx(fd6, shape, 0.15, 0.01, 1.0, dtype, path, variant)
        ctx.load_state(np.ascontiguousarray(G))
        ctx.fd_rk3_step(0.01, 1)
        outs.append(ctx.store_state())
        ctx.fd_destroy()
    assert np.array_equal(np.roll(outs[0], sh, (1, 2, 3)), outs[1])


@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_shear_mode_decay_closed_form_on_gpu(mods, path, variant):
    """P6 on the GPU: the discrete twin of the paper's Eq. 22 test."""
    O, fd6, I = mods
    n, k, u0, nu, nsteps = 32, 5, 1e-2, 5e-3, 10
    dx = TWO_PI / n
    dt = 0.1 * dx
    X = (np.arange(n) * dx)[None, None, :] * np.ones((n, n, 1))
    F = np.zeros((4, n, n, n))
    F[2] = u0 * np.sin(k * X)
    a = k * dx
    s2 = (490 - 540 * np.cos(a) + 54 * np.cos(2 * a) - 4 * np.cos(3 * a)) / 180
    z = -nu * dt * s2 / dx ** 2
    G = 1 + z + z * z / 2 + z ** 3 / 6
    ctx = make_ctx(fd6, (n,) * 3, dx, nu, 1.0, "f64", path, variant)
    ctx.load_state(F)
    ctx.fd_rk3_step(dt, nsteps)
    out = ctx.store_state()
    np.testing.assert_allclose(out[2], G ** nsteps * u0 * np.sin(k * X), atol=1e-13 * u0)
    assert max(np.abs(out[q]).max() for q in (0, 1, 3)) < 1e-15
    ctx.fd_destroy()


# ------------------------------- big grids: windowed oracle on sampled blocks
def _sample_origins(n, size, rng, extra, count=8):
    pts = [(0, 0, 0), (n - size // 2, n - size // 2, n - size // 2), (n - 7, 3, n // 2)] + list(extra)
    while len(pts) < count:
        pts.append(tuple(int(v) for v in rng.integers(0, n, 3)))
    return pts


def _windowed_check(mods, cfg_name, path, variant, n_override=None, inner=16, nblocks=8, before_step=None):
    import torch
    O, fd6, I = mods
    cfg = I.CONFIGS[cfg_name]
    n = n_override or cfg.n
    dx = TWO_PI / n
    dt = 0.1 * dx / cfg.cs
    F = I.make_state(cfg, device="cuda", n_override=n_override)
    ctx = make_ctx(fd6, (n,) * 3, dx, cfg.nu, cfg.cs, cfg.dtype, path, variant)
    ctx.load_state(F)
    if before_step:
        before_step(ctx)
    ctx.fd_rk3_step(dt, 1)
    out = torch.empty_like(F)
    ctx.store_state(out)
    ctx.fd_sync()
    m = O.window_margin(path)
    size = inner + 2 * m
    rng = np.random.default_rng(cfg.seed)
    # blocks at the periodic seam, at the origin, across tile boundaries (multiples of 64/16) and random ones
    extra = [(64 - m - 3, 16 - m - 2, n // 2 - m), (n // 2 - m - 1, n - m - 5, 5)]
    worst = 0.0
    for origin in _sample_origins(n, size, rng, extra, nblocks)[:nblocks]:
        sub = I.gather_block(F, origin, size).astype(np.float64)
        ref, mm = O.rk3_step_window(sub, dx, cfg.nu, cfg.cs, dt, 1, path)
        got = I.gather_block(out, tuple(o + m for o in origin), inner)
        worst = max(worst, relinf(got, ref))
    ctx.fd_destroy()
    del F, out
    torch.cuda.empty_cache()
    return worst


@pytest.mark.parametrize("path", [0, 1])
def test_c3_256_fp64_sampled_blocks(mods, path):
    assert _windowed_check(mods, "C3", path, 0) <= TOL["f64"]


@pytest.mark.parametrize("path", [0, 1])
def test_c4_512_fp32_sampled_blocks_in_the_bench_configuration(mods, path):
    """Full headline size, default (AUTO) variant = the launch configuration bench.py times; 16 blocks of 32^3
     at the periodic seam, the z-pairing seam, tile edges and random places."""
    assert _windowed_check(mods, "C4", path, 0, inner=32, nblocks=16) <= TOL["f32"]


@pytest.mark.parametrize("path", [0, 1])
def test_c5_1024_fp32_sampled_blocks(mods, path):
    import torch
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.skip("needs ~80 GB of free device memory")
    fd6 = mods[1]

    def rejected_switch(ctx):
        """The plain-layout tiled kernel cannot address 1024^3 (32-bit store offsets): an explicit request is refused
        BEFORE anything is converted, and the context keeps stepping with the variant it had."""
        assert ctx.fd_get_info().variant == fd6.FD_VARIANT_PAIRED
        with pytest.raises(fd6.FdError) as e:
            ctx.fd_set_variant(fd6.FD_VARIANT_TILED)
        assert e.value.code == fd6.FD_EUNSUPPORTED and "2^32" in str(e.value)
        assert ctx.fd_get_info().variant == fd6.FD_VARIANT_PAIRED

    assert _windowed_check(mods, "C5", path, 0, inner=32, nblocks=16, before_step=rejected_switch if path == 0 else None) <= TOL["f32"]


def test_c3_256_fp64_full_grid_55(mods):
    O, fd6, I = mods
    cfg = I.CONFIGS["C3"]
    F = I.make_state(cfg, device="cpu").numpy()
    ctx = make_ctx(fd6, (cfg.n,) * 3, cfg.dx, cfg.nu, cfg.cs, "f64", 0, 0)
    ctx.load_state(F)
    ctx.fd_rk3_step(cfg.dt, 1)
    got = ctx.store_state()
    ref = O.rk3_step(F, cfg.dx, cfg.nu, cfg.cs, cfg.dt, 1, 0)
    assert relinf(got, ref) <= TOL["f64"]
    ctx.fd_destroy()


# ------------------------------------------------- fd_rhs against the oracle: every kernel that can produce it
@pytest.mark.parametrize("shape", [(132, 70, 20), (72, 33, 41)])
@pytest.mark.parametrize("variant", [1, 2, 3])
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_fd_rhs_on_ragged_multi_tile_grids(mods, dtype, path, variant, shape):
    """fd_rhs is one of the six calls north_star names: right-hand side of Eq. 1-3 from the direct kernels (write_f = 0),
    the staged kernels in update mode 2 (plain fp32 = y pairs, fp64, paired fp32) and, on the 19-point path, pass 1 +
    pass 2 with write_f = 0, on shapes with several tiles per axis, ragged tails and (41 planes) an odd plane count."""
    O, fd6, I = mods
    rng = np.random.default_rng(1000 + 7 * path + variant)
    dx, nu, cs = 0.1, 0.02, 1.0
    F = smooth_state(rng, shape, 0.1, dtype)
    ctx = make_ctx(fd6, shape, dx, nu, cs, dtype, path, variant)
    ctx.load_state(F)
    T.fd_debug_poison_w(ctx)  # the w scratch fd_rhs writes through must not be read
    R = ctx.rhs_state()
    assert np.array_equal(ctx.store_state(), F)
    ctx.fd_destroy()
    assert relinf(R, O.rhs(F.astype(np.float64), dx, nu, cs, path)) <= TOL[dtype]


@pytest.mark.parametrize("variant", [1, 2, 3])
@pytest.mark.parametrize("path", [0, 1])
def test_fd_rhs_c2_full_grid_fp32(mods, path, variant):
    O, fd6, I = mods
    cfg = I.CONFIGS["C2"]
    F = I.make_state(cfg)
    ctx = make_ctx(fd6, (cfg.n,) * 3, cfg.dx, cfg.nu, cfg.cs, "f32", path, variant)
    ctx.load_state(F)
    R = ctx.rhs_state()
    ctx.fd_destroy()
    assert relinf(R, O.rhs(F.astype(np.float64), cfg.dx, cfg.nu, cfg.cs, path)) <= TOL["f32"]


@pytest.mark.parametrize("cfg_name,variant", [("C3", 2), ("C4", 0)])
@pytest.mark.parametrize("path", [0, 1])
def test_fd_rhs_big_grids_sampled_blocks(mods, cfg_name, variant, path):
    """fd_rhs on grids with more than one wave of tiles and a z-chunked remainder (C3 fp64 staged kernels, C4 fp32 in the
    bench configuration).  The right-hand side is local (radius 3; 6 on the 19-point path, whose pass 2 differentiates
    div u again), so the oracle runs on a periodic sub-block and only the cells further than that from its faces count."""
    import torch
    O, fd6, I = mods
    cfg = I.CONFIGS[cfg_name]
    n = cfg.n
    F = I.make_state(cfg, device="cuda")
    ctx = make_ctx(fd6, (n,) * 3, cfg.dx, cfg.nu, cfg.cs, cfg.dtype, path, variant)
    ctx.load_state(F)
    R = torch.empty_like(F)
    ctx.rhs_state(R)
    ctx.fd_sync()
    m = 3 if path == 0 else 6
    inner = 32
    size = inner + 2 * m
    rng = np.random.default_rng(cfg.seed + 17)
    extra = [(64 - m - 3, 16 - m - 2, n // 2 - m), (n // 2 - m - 1, n - m - 5, 5)]
    worst = 0.0
    for origin in _sample_origins(n, size, rng, extra, 16):
        sub = I.gather_block(F, origin, size).astype(np.float64)
        ref = O.rhs(sub, cfg.dx, cfg.nu, cfg.cs, path)[:, m:-m, m:-m, m:-m]
        got = I.gather_block(R, tuple(o + m for o in origin), inner)
        worst = max(worst, relinf(got, ref))
    ctx.fd_destroy()
    del F, R
    torch.cuda.empty_cache()
    assert worst <= TOL[cfg.dtype]


# ------------------------------------------------------------------------ error behaviour
def test_error_codes_on_a_live_context(mods):
    O, fd6, I = mods
    ctx = fd6.Fd(32, 32, 32, 0.1, 0.01, 1.0, fd6.FD_F32)
    L = fd6.lib
    assert L.fd_rk3_step(ctx._h, 0.1, -1) == fd6.FD_EINVAL
    assert L.fd_rk3_step(ctx._h, float("inf"), 1) == fd6.FD_EINVAL
    assert L.fd_set_path(ctx._h, 5) == fd6.FD_EINVAL
    assert L.fd_set_variant(ctx._h, 9) == fd6.FD_EINVAL
    assert L.fd_load(ctx._h, None, None, None, None, fd6.FD_HOST) == fd6.FD_EINVAL
    a = np.zeros(32 ** 3, dtype=np.float32)
    p = a.ctypes.data
    assert L.fd_load(ctx._h, p, p, p, p, 3) == fd6.FD_EINVAL
    assert L.fd_get_profile(ctx._h, 99, None, None) == fd6.FD_EINVAL
    info = ctx.fd_get_info()
    assert (info.nx, info.ny, info.nz) == (32, 32, 32) and info.ghost_y == 3 and info.pitch_x >= 32 + 6
    assert info.device_bytes >= 12 * 32 ** 3 * 4
    ctx.fd_destroy()


def test_fd_get_info_reports_what_the_context_launches(mods):
    """variant, prepared tile shape, tile extents and work items come from the context, not from a planner call."""
    O, fd6, I = mods
    ctx = fd6.Fd(32, 32, 32, 0.1, 0.01, 1.0, fd6.FD_F64)  # AUTO on a tiny grid: the one-thread-per-cell kernels
    info = ctx.fd_get_info()
    assert info.variant == fd6.FD_VARIANT_DIRECT and (info.tile_shape, info.tile_x, info.tile_y, info.work_items) == (-1, 0, 0, 0)
    assert info.graph_state == fd6.FD_GRAPH_WAITING and info.graph_note == b""
    ctx.fd_set_graphs(False)
    assert ctx.fd_get_info().graph_state == fd6.FD_GRAPH_OFF
    ctx.fd_destroy()
    sms = __import__("torch").cuda.get_device_properties(0).multi_processor_count
    ctx = fd6.Fd(256, 256, 64, 0.1, 0.01, 1.0, fd6.FD_F64)  # 8 x 16 tall tiles
    info = ctx.fd_get_info()
    wl = fd6.fd_plan_work_list(256, 256, 64, fd6.FD_F64, sms)
    assert info.variant == fd6.FD_VARIANT_TILED and (info.tile_shape, info.tile_x, info.tile_y) == (1, 32, 16)
    assert info.work_items == wl.items and (wl.split_plane > 0) == (wl.items == 2 * wl.tiles_x * wl.tiles_y)
    ctx.fd_set_tile_shape(0)
    info = ctx.fd_get_info()
    assert (info.tile_shape, info.tile_x, info.tile_y) == (0, 32, 12) and info.work_items > 0
    ctx.fd_destroy()


def test_profile_counters_count_the_launches(mods):
    O, fd6, I = mods
    ctx = fd6.Fd(64, 64, 64, 0.1, 0.01, 1.0, fd6.FD_F32)
    ctx.load_state(np.zeros((4, 64, 64, 64), dtype=np.float32))
    ctx.fd_set_profiling(True)
    ctx.fd_reset_profile()
    before = ctx.fd_kernel_launches()
    ctx.fd_rk3_step(0.01, 2)
    ms, n = ctx.fd_get_profile(fd6.FD_K_FUSED55)
    assert n == 6 and ms > 0
    total = sum(ctx.fd_get_profile(k)[1] for k in range(fd6.FD_K_COUNT))
    assert total == ctx.fd_kernel_launches() - before
    ctx.fd_destroy()


# ------------------------------------------------- layout conversion when the variant changes
def test_variant_switch_carries_a_loaded_state_across_layouts(mods):
    """PAIRED stores cells k and k+nz/2 side by side; switching variants converts the resident state.  Every
    variant, entered from either layout, must continue the same trajectory (each compared with the oracle)."""
    O, fd6, I = mods
    shape = (40, 24, 18)
    rng = np.random.default_rng(77)
    dx, nu, cs = 0.2, 0.02, 1.0
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.1, "f32")
    ctx = fd6.Fd(*shape, dx, nu, cs, fd6.FD_F32)
    assert ctx.fd_get_info().variant == fd6.FD_VARIANT_DIRECT  # AUTO on a tiny grid
    ctx.fd_set_variant(fd6.FD_VARIANT_PAIRED)                   # fp32, even nz: the paired layout takes it
    ctx.load_state(F)
    order = [fd6.FD_VARIANT_TILED, fd6.FD_VARIANT_DIRECT, fd6.FD_VARIANT_PAIRED, fd6.FD_VARIANT_DIRECT, fd6.FD_VARIANT_TILED]
    for n, v in enumerate(order, start=1):
        ctx.fd_set_variant(v)
        assert ctx.fd_get_info().variant == v
        assert np.array_equal(ctx.store_state(), F) or n > 1  # the conversion itself is exact
        ctx.fd_rk3_step(dt, 1)
        got = ctx.store_state()
        ref = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, n, 0)
        assert relinf(got, ref) <= n * TOL["f32"]
    # fd_rhs through the paired layout, host and device destinations agree with the oracle
    ctx.fd_set_variant(fd6.FD_VARIANT_PAIRED)
    ctx.load_state(F)
    R = ctx.rhs_state()
    assert relinf(R, O.rhs(F.astype(np.float64), dx, nu, cs, 0)) <= TOL["f32"]
    assert np.array_equal(ctx.store_state(), F)
    import torch
    Rd = torch.empty((4,) + shape[::-1], dtype=torch.float32, device="cuda")
    ctx.rhs_state(Rd)
    ctx.fd_sync()
    assert np.array_equal(Rd.cpu().numpy(), R)
    ctx.fd_destroy()


def test_paired_variant_is_refused_where_it_cannot_run(mods):
    O, fd6, I = mods
    ctx = fd6.Fd(16, 16, 9, 0.1, 0.01, 1.0, fd6.FD_F32)   # odd nz
    assert ctx.fd_get_info().variant == fd6.FD_VARIANT_DIRECT  # AUTO on a tiny grid
    ctx.fd_destroy()
    ctx = fd6.Fd(96, 96, 45, 0.1, 0.01, 1.0, fd6.FD_F32)  # odd nz, large enough for the staged kernels
    assert ctx.fd_get_info().variant == fd6.FD_VARIANT_TILED
    with pytest.raises(fd6.FdError) as e:
        ctx.fd_set_variant(fd6.FD_VARIANT_PAIRED)
    assert e.value.code == fd6.FD_EUNSUPPORTED
    ctx.fd_destroy()
    ctx = fd6.Fd(16, 16, 16, 0.1, 0.01, 1.0, fd6.FD_F64)  # fp64
    with pytest.raises(fd6.FdError) as e:
        ctx.fd_set_variant(fd6.FD_VARIANT_PAIRED)
    assert e.value.code == fd6.FD_EUNSUPPORTED
    ctx.fd_destroy()


# ------------------------------------------------- work-list corners: many tiles, few planes; ragged everything
@pytest.mark.parametrize("shape,dtype", [((512, 500, 16), "f32"), ((512, 500, 16), "f64"), ((1024, 300, 8), "f32"),
                                         ((36, 1000, 10), "f64"), ((2048, 100, 9), "f32"), ((132, 2000, 12), "f32")])
@pytest.mark.parametrize("path", [0, 1])
def test_many_tiles_few_planes(mods, shape, dtype, path):
    """Grids whose tile count exceeds the SM count (full columns AND a z-chunked remainder in one launch) with very
    few planes, odd plane counts (plain fp32 layout) and ragged tiles, one step against the oracle on the full grid."""
    O, fd6, I = mods
    rng = np.random.default_rng(11)
    dx, nu, cs = 0.1, 0.004, 1.0
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.05, dtype)
    ctx = fd6.Fd(*shape, dx, nu, cs, fd6.FD_F32 if dtype == "f32" else fd6.FD_F64)
    ctx.fd_set_path(path)
    wl = fd6.fd_plan_work_list(*shape, fd6.FD_F32 if dtype == "f32" else fd6.FD_F64, 148)
    ctx.load_state(F)
    ctx.fd_rk3_step(dt, 1)
    got = ctx.store_state()
    ctx.fd_destroy()
    ref = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 1, path)
    assert relinf(got, ref) <= TOL[dtype], (wl.full_tiles, wl.chunks, wl.chunk_planes, wl.items)


# ------------------------------------------------- CUDA-graph stepping (fd_set_graphs) against plain launches
@pytest.mark.parametrize("dtype,shape", [("f32", (40, 26, 24)), ("f32", (40, 13, 9)), ("f64", (36, 20, 11))])
@pytest.mark.parametrize("path", [0, 1])
def test_graph_steps_equal_plain_launches_bitwise(mods, dtype, shape, path):
    """One graph launch per step must enqueue exactly the launches of the plain path: same bits and the same launch
    count, across an odd number of steps (the read copy alternates), a change of dt, of the forcing and of the variant
    (each drops the graphs; a new one is captured once the new parameters have held for two steps), and with the oracle
    as the referee of the whole trajectory."""
    O, fd6, I = mods
    rng = np.random.default_rng(77 + path)
    dx, nu, cs = 0.2, 0.02, 1.0
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.1, dtype)
    kf, ef = (TWO_PI / (shape[0] * dx), 0.0, 2 * TWO_PI / (shape[2] * dx)), (0.0, 1.0, 0.0)

    def trajectory(graphs):
        ctx = fd6.Fd(*shape, dx, nu, cs, fd6.FD_F32 if dtype == "f32" else fd6.FD_F64)
        ctx.fd_set_path(path)
        ctx.fd_set_graphs(graphs)
        captured = fd6.FD_GRAPH_CAPTURED if graphs else fd6.FD_GRAPH_OFF
        waiting = fd6.FD_GRAPH_WAITING if graphs else fd6.FD_GRAPH_OFF
        ctx.load_state(F)
        n0 = ctx.fd_kernel_launches()
        ctx.fd_rk3_step(dt, 3)  # two plain steps while the parameters settle, then the first captured step
        assert ctx.fd_get_info().graph_state == captured
        ctx.fd_rk3_step(dt, 2)  # the graph of the other read copy, then the first one again
        a = ctx.store_state()
        ctx.fd_rk3_step(0.5 * dt, 1)
        assert ctx.fd_get_info().graph_state == waiting  # a new dt: plain launches, nothing captured for one step
        ctx.fd_set_forcing(kf, ef, 0.3, 0.02, dt)
        ctx.fd_rk3_step(dt, 4)  # forced steps: two plain, then one graph per read copy
        assert ctx.fd_get_info().graph_state == captured
        ctx.fd_set_forcing(None, None, 0.0, 0.0, dt)
        ctx.fd_set_variant(fd6.FD_VARIANT_DIRECT)
        ctx.fd_rk3_step(dt, 3)
        assert ctx.fd_get_info().graph_state == captured
        b = ctx.store_state()
        n = ctx.fd_kernel_launches() - n0
        assert ctx.fd_get_info().graph_note == b""
        ctx.fd_destroy()
        return a, b, n

    a1, b1, n1 = trajectory(True)
    a0, b0, n0 = trajectory(False)
    assert n1 == n0 and n1 > 0
    assert all(np.array_equal(x, y) for x, y in zip(a1, a0))
    assert all(np.array_equal(x, y) for x, y in zip(b1, b0))
    ref = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 5, path)
    assert relinf(a1, ref) <= 5 * TOL[dtype]


def test_parameters_that_change_every_step_never_pay_for_a_capture(mods):
    """A driver that draws a new forcing wavevector every step or adapts dt every step must run plain
    launches (graph_state stays FD_GRAPH_WAITING: no capture, no instantiation per step) with the bits of graphs-off."""
    O, fd6, I = mods
    shape, dx, nu, cs = (40, 26, 24), 0.2, 0.02, 1.0
    dt = 0.1 * dx
    F = smooth_state(np.random.default_rng(5), shape, 0.1, "f32")
    k1 = TWO_PI / (shape[0] * dx)

    def run(graphs):
        ctx = fd6.Fd(*shape, dx, nu, cs, fd6.FD_F32)
        ctx.fd_set_graphs(graphs)
        ctx.load_state(F)
        states = []
        for s in range(6):
            ctx.fd_set_forcing((k1 * (1 + s % 3), 0.0, 0.0), (0.0, 1.0, 0.0), 0.1 * s, 0.02, dt)
            ctx.fd_rk3_step(dt, 1)
            states.append(ctx.fd_get_info().graph_state)
        for s in range(6):
            ctx.fd_rk3_step(dt * (1.0 + 0.01 * s), 1)
            states.append(ctx.fd_get_info().graph_state)
        out = ctx.store_state()
        n = ctx.fd_kernel_launches()
        ctx.fd_destroy()
        return out, states, n

    g, sg, ng = run(True)
    p, sp, np_ = run(False)
    assert sg == [fd6.FD_GRAPH_WAITING] * 12 and sp == [fd6.FD_GRAPH_OFF] * 12
    assert ng == np_ and all(np.array_equal(x, y) for x, y in zip(g, p))


# ------------------------------------------------- BASELINE config C2 as stated: 100 RK3 steps, both stencil paths
@pytest.mark.parametrize("path", [0, 1])
def test_c2_hundred_steps_full_grid_deviation_reported(mods, path, capsys):
    """after the config's own 100 steps the full-grid deviation from the oracle is REPORTED (printed;
    DESIGN.md section 9 quotes it), not gated at the one-step tolerance: fp32 rounding differences between two correct
    evaluation orders grow along the trajectory.  The gate here only catches a wrong trajectory (100 x the one-step bar)."""
    O, fd6, I = mods
    cfg = I.CONFIGS["C2"]
    F = I.make_state(cfg)
    ctx = fd6.Fd(cfg.n, cfg.n, cfg.n, cfg.dx, cfg.nu, cfg.cs, fd6.FD_F32)
    ctx.fd_set_path(path)
    ctx.load_state(F)
    ctx.fd_rk3_step(cfg.dt, 100)
    got = ctx.store_state()
    variant = ctx.fd_get_info().variant
    ctx.fd_destroy()
    ref = O.rk3_step(F.astype(np.float64), cfg.dx, cfg.nu, cfg.cs, cfg.dt, 100, path)
    dev = relinf(got, ref)
    with capsys.disabled():
        print(f"\nC2 128^3 fp32, 100 RK3 steps, {'55' if path == 0 else '19'}-point path, variant {variant}: "
              f"max relative L-inf deviation from the fp64 oracle = {dev:.3e}")
    assert dev <= 100 * TOL["f32"]


# ------------------------------------------------- the two tile shapes of the staged kernels (fd_set_tile_shape)
@pytest.mark.parametrize("shape", [(40, 13, 10), (132, 70, 20), (72, 33, 42), (512, 500, 16), (36, 1000, 10), (132, 2000, 12)])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("path", [0, 1])
def test_tall_tiles_equal_wide_tiles_bitwise(mods, shape, dtype, path):
    """The tall shape (two vertically adjacent values per thread) loads less but computes every value with the same
    operations in the same order as the wide one: identical bits, on ragged grids, on grids with many tiles and few planes
    (z-chunked remainders), for the paired fp32 and the fp64 kernels, on both paths; and both within the one-step bar."""
    O, fd6, I = mods
    rng = np.random.default_rng(sum(shape) + path)
    dx, nu, cs = 0.2, 0.02, 1.0
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.1, dtype)
    out = []
    for tile_shape in (0, 1):
        ctx = make_ctx(fd6, shape, dx, nu, cs, dtype, path, fd6.FD_VARIANT_PAIRED if dtype == "f32" else fd6.FD_VARIANT_TILED)
        ctx.fd_set_tile_shape(tile_shape)
        T.fd_debug_poison_ghosts(ctx)
        ctx.load_state(F)
        T.fd_debug_poison_w(ctx)
        ctx.fd_rk3_step(dt, 2)
        out.append(ctx.store_state())
        R = ctx.rhs_state()
        out.append(R)
        ctx.fd_destroy()
    assert all(np.array_equal(a, b) for a, b in zip(out[0], out[2]))
    assert all(np.array_equal(a, b) for a, b in zip(out[1], out[3]))
    ref = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 2, path)
    assert relinf(out[2], ref) <= 2 * TOL[dtype]


@pytest.mark.parametrize("shape", [(132, 70, 20), (72, 33, 42), (512, 500, 16)])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("tile_shape", [0, 1])
def test_overlapping_tiles_give_the_same_bits(mods, shape, dtype, tile_shape):
    """fd_debug_set_tile_overlap (the temporal-blocking emulation DESIGN.md section 7 measures): tiles that overlap by a
    radius-3 ring on every side do redundant work but store every value exactly once, with unchanged bits."""
    O, fd6, I = mods
    rng = np.random.default_rng(sum(shape))
    dx, nu, cs = 0.2, 0.02, 1.0
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.1, dtype)
    out = []
    for overlap in (0, 6):
        ctx = make_ctx(fd6, shape, dx, nu, cs, dtype, 0, fd6.FD_VARIANT_PAIRED if dtype == "f32" else fd6.FD_VARIANT_TILED)
        ctx.fd_set_tile_shape(tile_shape)
        T.fd_debug_set_tile_overlap(ctx, overlap)
        ctx.load_state(F)
        ctx.fd_rk3_step(dt, 2)
        out.append(ctx.store_state())
        ctx.fd_destroy()
    assert all(np.array_equal(a, b) for a, b in zip(out[0], out[1]))
    ref = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 2, 0)
    assert relinf(out[1], ref) <= 2 * TOL[dtype]
