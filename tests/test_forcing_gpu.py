"""Forcing term of Eq. 2 (Eq. 24-25) on the CUDA path, through the C ABI, against the
oracle step O11 on the same inputs — same bars as test_parity_gpu.py (1e-12 fp64, 2e-5 fp32, reading G14/G15)."""
import math

import numpy as np
import pytest

from test_parity_gpu import TOL, TWO_PI, make_ctx, relinf, smooth_state

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from oracle import oracle as O
    from paper_1707_08900_b200 import fd6, inputs
    return O, fd6, inputs


def _spec(dt, k=(2, -1, 3), e=(0.36, -0.48, 0.8), phi=0.7, f0=0.05):
    return dict(k=k, e=e, phi=phi, f0=f0, dt=dt)


@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_forced_rhs_and_steps_c1_fp64(mods, path, variant):
    O, fd6, I = mods
    cfg = I.CONFIGS["C1"]
    F = I.make_state(cfg)
    sp = _spec(cfg.dt)
    ctx = make_ctx(fd6, (cfg.n,) * 3, cfg.dx, cfg.nu, cfg.cs, "f64", path, variant)
    ctx.fd_set_forcing(sp["k"], sp["e"], sp["phi"], sp["f0"], sp["dt"])
    ctx.load_state(F)
    assert relinf(ctx.rhs_state(), O.rhs(F, cfg.dx, cfg.nu, cfg.cs, path, force=sp)) <= TOL["f64"]
    ctx.fd_rk3_step(cfg.dt, 3)
    got = ctx.store_state()
    ref = O.rk3_step(F, cfg.dx, cfg.nu, cfg.cs, cfg.dt, 3, path, force=sp)
    assert relinf(got, ref) <= TOL["f64"]
    assert relinf(got, O.rk3_step(F, cfg.dx, cfg.nu, cfg.cs, cfg.dt, 3, path)) > 1e-4  # the forcing did act
    # f0 = 0 switches it off again: bit-identical to a context that never had a forcing
    ctx.fd_set_forcing(None, None, 0.0, 0.0, 1.0)
    ctx.load_state(F)
    ctx.fd_rk3_step(cfg.dt, 1)
    a = ctx.store_state()
    ctx.fd_destroy()
    ctx = make_ctx(fd6, (cfg.n,) * 3, cfg.dx, cfg.nu, cfg.cs, "f64", path, variant)
    ctx.load_state(F)
    ctx.fd_rk3_step(cfg.dt, 1)
    assert np.array_equal(a, ctx.store_state())
    ctx.fd_destroy()


@pytest.mark.parametrize("shape", [(40, 13, 9), (72, 33, 42), (64, 32, 32)])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("variant", [1, 2, 3])
def test_forced_steps_on_ragged_grids(mods, shape, dtype, path, variant):
    O, fd6, I = mods
    rng = np.random.default_rng(5)
    dx, nu, cs = 0.17, 0.01, 1.1
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.05, dtype)
    sp = _spec(dt, k=(1.3, -0.7, 2.1), phi=-2.0, f0=0.08)  # f need not be periodic on the box: it is only evaluated
    ctx = make_ctx(fd6, shape, dx, nu, cs, dtype, path, variant)
    ctx.fd_set_forcing(sp["k"], sp["e"], sp["phi"], sp["f0"], sp["dt"])
    ctx.load_state(F)
    ctx.fd_rk3_step(dt, 2)
    got = ctx.store_state()
    ctx.fd_destroy()
    ref = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 2, path, force=sp)
    assert relinf(got, ref) <= TOL[dtype]


@pytest.mark.parametrize("path", [0, 1])
def test_forced_shear_mode_from_rest_closed_form_on_gpu(mods, path):
    """P13 on the GPU: a_{n+1} = G a_n + N dt (G - 1)/z with the discrete symbol of Eq. 7."""
    O, fd6, I = mods
    n, kk, nu, nsteps = 32, 3, 0.02, 9
    dx = TWO_PI / n
    dt = 0.1 * dx
    f0 = 0.02
    ctx = fd6.Fd(n, n, n, dx, nu, 1.0, fd6.FD_F64)
    ctx.fd_set_path(path)
    ctx.fd_set_forcing((kk, 0, 0), (0, 0, 1), 0.4, f0, dt)  # k x e = (0, -k, 0): f along -y
    ctx.fd_rk3_step(dt, nsteps)  # from the zero state fd_create leaves
    out = ctx.store_state()
    ctx.fd_destroy()
    a = kk * dx
    s2 = (490 - 540 * np.cos(a) + 54 * np.cos(2 * a) - 4 * np.cos(3 * a)) / 180
    z = -nu * dt * s2 / dx ** 2
    G = 1 + z + z * z / 2 + z ** 3 / 6
    N = f0 * math.sqrt(kk / dt)
    amp = 0.0
    for _ in range(nsteps):
        amp = G * amp + N * dt * (1 + z / 2 + z * z / 6)
    expect = -amp * np.cos(kk * np.arange(n) * dx + 0.4)
    np.testing.assert_allclose(out[2], expect[None, None, :] * np.ones((n, n, 1)), atol=1e-13 * amp)
    assert max(float(np.abs(out[q]).max()) for q in (0, 1, 3)) < 1e-15


def test_forced_c4_512_fp32_sampled_blocks(mods):
    """The bench configuration with the forcing on: one step at 512^3 against the windowed oracle on sampled blocks."""
    import torch
    O, fd6, I = mods
    cfg = I.CONFIGS["C4"]
    n, dx = cfg.n, cfg.dx
    dt = cfg.dt
    sp = _spec(dt, k=(3, 2, -4), f0=0.05)
    F = I.make_state(cfg, device="cuda")
    ctx = fd6.Fd(n, n, n, dx, cfg.nu, cfg.cs, fd6.FD_F32)
    ctx.fd_set_forcing(sp["k"], sp["e"], sp["phi"], sp["f0"], sp["dt"])
    ctx.load_state(F)
    ctx.fd_rk3_step(dt, 1)
    out = torch.empty_like(F)
    ctx.store_state(out)
    ctx.fd_sync()
    ctx.fd_destroy()
    m = O.window_margin(0)
    inner, worst = 16, 0.0
    for origin in [(0, 0, 0), (n - 20, n - 20, n - 20), (n - 7, 3, n // 2), (250, 100, 37), (n // 2 - m - 1, n - m - 5, 5), (17, 300, 490)]:
        sub = I.gather_block(F, origin, inner + 2 * m).astype(np.float64)
        ref = O.rk3_step(sub, dx, cfg.nu, cfg.cs, dt, 1, 0, force=sp, origin=origin[::-1])[:, m:-m, m:-m, m:-m]
        got = I.gather_block(out, tuple(o + m for o in origin), inner)
        worst = max(worst, relinf(got, ref))
    assert worst <= TOL["f32"]


def test_forcing_argument_errors_on_a_live_context(mods):
    O, fd6, I = mods
    ctx = fd6.Fd(32, 32, 32, 0.2, 0.01, 1.0, fd6.FD_F32)
    for args in [((0, 0, 2), (0, 0, 1), 0.0, 1.0, 0.01),        # k parallel to e
                 ((1, 0, 0), (0, 1, 0), 0.0, -1.0, 0.01),       # f0 < 0
                 ((1, 0, 0), (0, 1, 0), 0.0, 1.0, 0.0),         # dt_ref <= 0
                 ((1, 0, 0), (0, 1, 0), float("nan"), 1.0, 0.01),
                 ((float("inf"), 0, 0), (0, 1, 0), 0.0, 1.0, 0.01),
                 (None, None, 0.0, 1.0, 0.01)]:                  # NULL vectors with f0 != 0
        with pytest.raises(fd6.FdError) as ei:
            ctx.fd_set_forcing(*args)
        assert ei.value.code == fd6.FD_EINVAL
    ctx.fd_set_forcing(None, None, 0.0, 0.0, 1.0)  # switching off needs no vectors
    ctx.fd_rk3_step(0.01, 1)                       # and a failed call left the context usable
    assert np.array_equal(ctx.store_state(), np.zeros((4, 32, 32, 32), np.float32))
    ctx.fd_destroy()


@pytest.mark.parametrize("path", [0, 1])
def test_forcing_on_a_grid_too_deep_for_the_shared_z_table(mods, path):
    """12000 planes: the forcing's z phase table no longer fits beside the staging rings of the staged kernels.  Under
    FD_VARIANT_AUTO the forced launches fall back to the one-thread-per-cell kernels (no error, oracle parity); a variant
    asked for by name still reports FD_EUNSUPPORTED."""
    O, fd6, I = mods
    shape = (32, 16, 12000)
    rng = np.random.default_rng(12)
    dx, nu, cs = 0.2, 0.02, 1.0
    dt = 0.1 * dx
    F = smooth_state(rng, shape, 0.05, "f32")
    sp = _spec(dt, k=(1.0, 0.5, 0.013), f0=0.05)
    ctx = fd6.Fd(*shape, dx, nu, cs, fd6.FD_F32)
    ctx.fd_set_path(path)
    assert ctx.fd_get_info().variant == fd6.FD_VARIANT_PAIRED
    ctx.load_state(F)
    ctx.fd_set_forcing(sp["k"], sp["e"], sp["phi"], sp["f0"], sp["dt"])
    ctx.fd_rk3_step(dt, 1)
    got = ctx.store_state()
    ref = O.rk3_step(F.astype(np.float64), dx, nu, cs, dt, 1, path, force=sp)
    assert relinf(got, ref) <= TOL["f32"]
    ctx.fd_set_variant(fd6.FD_VARIANT_PAIRED)  # by name: the limit is reported
    with pytest.raises(fd6.FdError) as e:
        ctx.fd_rk3_step(dt, 1)
    assert e.value.code == fd6.FD_EUNSUPPORTED
    ctx.fd_destroy()
