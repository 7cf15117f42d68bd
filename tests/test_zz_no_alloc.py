"""fd_rhs_static (include/fd6.h): the entry point for callers that cannot allocate device memory.

Who needs it: code that runs where cudaMalloc is off limits — a solver plug-in inside an application whose own pool
holds all of the GPU's memory, or a time loop that must not trigger the device-wide synchronisation of cudaMalloc and
cudaFree.  Such callers cannot use fd_create (it allocates the padded field copies and w); fd_rhs_static keeps the padded
copy in an 8 MiB array built into libfd6.so instead, shared by every call on the device.

What is checked here, through the C ABI on a B200:
  * two calls in a row give what the existing path (fd_create + fd_load + fd_rhs, FD_PATH_55) gives for the same
    states, within the bars the parity tests use (1e-12 fp64, 2e-5 fp32; relative L-inf per field);
  * the shared array keeps the previous call's contents and that must not matter: a small grid is run right after a
    larger one whose state was all NaN, and still has to match;
  * the calls do not take device memory (free memory as the driver reports it does not drop);
  * grids beyond the array are refused with a message that says so.
This file is named to be collected last (pytest -x stops at the first failure), and it holds no state that depends on
the tests before it: it passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 2e-5}  # the bars of tests/test_parity_gpu.py


@pytest.fixture(scope="module")
def mods():
    import torch
    from paper_1707_08900_b200 import fd6, inputs
    torch.cuda.set_device(0)
    return torch, fd6, inputs


def relinf(A, B):
    """Per field max|A-B| / max|B| (absolute if max|B| == 0), max over fields (reading G14)."""
    worst = 0.0
    for a, b in zip(A, B):
        den = float(np.abs(b).max())
        err = float(np.abs(a.astype(np.float64) - b.astype(np.float64)).max())
        worst = max(worst, err / den if den > 0 else err)
    return worst


def smooth_state(rng, shape_xyz, amp, np_dtype):
    """A few random low-wavenumber modes per field on a periodic box (inputs only; no method arithmetic)."""
    nx, ny, nz = shape_xyz
    i = np.arange(nx)[None, None, :] / nx
    j = np.arange(ny)[None, :, None] / ny
    k = np.arange(nz)[:, None, None] / nz
    F = np.zeros((4, nz, ny, nx))
    for q in range(4):
        for _ in range(4):
            kv = rng.integers(-2, 3, 3)
            F[q] += amp * rng.uniform(0.3, 1.0) * np.cos(2 * np.pi * (kv[0] * i + kv[1] * j + kv[2] * k) + rng.uniform(0, 2 * np.pi))
    return np.ascontiguousarray(F.astype(np_dtype))


def existing_path_rhs(fd6, F, shape_xyz, dx, nu, cs, dtype):
    """fd_create + fd_load + fd_rhs on FD_PATH_55 with the kernels FD_VARIANT_AUTO picks."""
    nx, ny, nz = shape_xyz
    ctx = fd6.Fd(nx, ny, nz, dx, nu, cs, dtype)
    ctx.fd_set_path(fd6.FD_PATH_55)
    ctx.load_state(F)
    R = ctx.rhs_state()
    ctx.fd_destroy()
    return R


def static_rhs(torch, fd6, F, shape_xyz, dx, nu, cs, dtype, out=None):
    nx, ny, nz = shape_xyz
    dF = torch.from_numpy(F).cuda()
    if out is None:
        out = torch.full_like(dF, float("nan"))  # every element has to be written by the call
    fd6.fd_rhs_static(nx, ny, nz, dx, nu, cs, dtype, [dF[q] for q in range(4)], [out[q] for q in range(4)])
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("dt", ["f64", "f32"])
def test_two_calls_in_a_row_match_the_existing_path(mods, dt):
    torch, fd6, I = mods
    dtype = fd6.FD_F64 if dt == "f64" else fd6.FD_F32
    np_dtype = np.float64 if dt == "f64" else np.float32
    cfg = I.CONFIGS["C1"]
    rng = np.random.default_rng(1707_08900)
    # first call: BASELINE config C1 (32^3); second call, straight after it: another state on a ragged box
    cases = [((cfg.n,) * 3, I.make_state(cfg).astype(np_dtype)), ((44, 21, 19), None)]
    for shape, F in cases:
        if F is None:
            F = smooth_state(rng, shape, 1e-2, np_dtype)
        dx = 2 * np.pi / shape[0]
        got = static_rhs(torch, fd6, F, shape, dx, cfg.nu, cfg.cs, dtype)
        want = existing_path_rhs(fd6, F, shape, dx, cfg.nu, cfg.cs, dtype)
        assert np.isfinite(got).all()
        assert relinf(got, want) <= TOL[dt], (shape, relinf(got, want))


def test_contents_left_by_the_previous_call_do_not_leak(mods):
    torch, fd6, I = mods
    cfg = I.CONFIGS["C1"]
    big, small = (64, 64, 64), (24, 20, 16)
    # call 1 fills the whole padded region of a 64^3 fp32 grid (6.0 of the 8 MiB) with NaN ...
    nanF = np.full((4,) + big[::-1], np.nan, dtype=np.float32)
    static_rhs(torch, fd6, nanF, big, 0.1, cfg.nu, cfg.cs, fd6.FD_F32)
    # ... call 2 runs a small fp64 grid in the same bytes: every value its stencil reads must be its own
    F = smooth_state(np.random.default_rng(7), small, 1e-2, np.float64)
    dx = 2 * np.pi / small[0]
    got = static_rhs(torch, fd6, F, small, dx, cfg.nu, cfg.cs, fd6.FD_F64)
    want = existing_path_rhs(fd6, F, small, dx, cfg.nu, cfg.cs, fd6.FD_F64)
    assert np.isfinite(got).all()
    assert relinf(got, want) <= TOL["f64"]


def test_calls_take_no_device_memory(mods):
    torch, fd6, I = mods
    cfg = I.CONFIGS["C1"]
    shape = (cfg.n,) * 3
    dF = torch.from_numpy(I.make_state(cfg)).cuda()
    out = torch.empty_like(dF)
    args = (*shape, cfg.dx, cfg.nu, cfg.cs, fd6.FD_F64, [dF[q] for q in range(4)], [out[q] for q in range(4)])
    fd6.fd_rhs_static(*args)  # the first call on the device looks the array's address up and loads the kernels
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        fd6.fd_rhs_static(*args)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, f"device free memory dropped by {free0 - free1} bytes across fd_rhs_static calls"


def test_grids_beyond_the_built_in_array_are_refused(mods):
    torch, fd6, I = mods
    x = torch.zeros(8, device="cuda")
    four = [x] * 4
    for shape, dtype in (((64, 64, 64), fd6.FD_F64), ((128, 128, 128), fd6.FD_F32), ((2048, 2048, 2048), fd6.FD_F32)):
        with pytest.raises(fd6.FdError) as ei:
            fd6.fd_rhs_static(*shape, 0.1, 0.0, 1.0, dtype, four, four)
        assert ei.value.code == fd6.FD_EUNSUPPORTED
        assert "built-in scratch" in str(ei.value) and str(fd6.FD_RHS_STATIC_MAX_BYTES) in str(ei.value)
