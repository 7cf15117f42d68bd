"""Seeded synthetic inputs for the five BASELINE.json configs (C1..C5).

This module is the ONLY thing the CUDA path's tests/bench and the CPU oracle share.  It holds
none of the method's arithmetic (no stencil, no RHS, no RK coefficient): it only draws
random wave-vectors / phases / Fourier coefficients and evaluates smooth periodic fields.
The recipe for every config is stated in DESIGN.md "Inputs".  The paper names no dataset
("a test case, which simulated compressible hydrodynamic flow"); these fields
stand in for that generic periodic compressible flow.

State layout: array of shape (4, nz, ny, nx); component 0 = ln rho, 1..3 = u_x, u_y, u_z;
x is the fastest axis (PAPER.md:189 structure of arrays).  Domain is (2*pi)^3.
"""
import math
from dataclasses import dataclass

import numpy as np

SEED0 = 170708900
TWO_PI = 2.0 * math.pi


@dataclass(frozen=True)
class Config:
    name: str
    n: int            # grid points per axis (cubic, periodic)
    dtype: str        # "f32" | "f64"
    nu: float
    cs: float
    nsteps: int       # full RK3 steps the config asks for
    kind: str         # "modes" | "band"
    kmax: int
    amp: float        # modes: field amplitude; band: rms Mach number of u
    lnrho_rms: float  # band only
    seed: int

    @property
    def dx(self) -> float:
        return TWO_PI / self.n

    @property
    def dt(self) -> float:          # reading G18: dt = 0.1 dx / cs for every config
        return 0.1 * self.dx / self.cs

    @property
    def np_dtype(self):
        return np.float32 if self.dtype == "f32" else np.float64


CONFIGS = {
    "C1": Config("C1", 32, "f64", 5e-3, 1.0, 1, "modes", 4, 1e-2, 0.0, SEED0 + 1),
    "C2": Config("C2", 128, "f32", 5e-3, 1.0, 100, "modes", 4, 1e-1, 0.0, SEED0 + 2),
    "C3": Config("C3", 256, "f64", 5e-3, 1.0, 20, "band", 16, 0.1, 0.0, SEED0 + 3),
    "C4": Config("C4", 512, "f32", 1e-3, 1.0, 20, "band", 32, 0.3, 0.1, SEED0 + 4),
    "C5": Config("C5", 1024, "f32", 5e-4, 1.0, 5, "band", 64, 0.3, 0.1, SEED0 + 5),
}


# ------------------------------------------------------------------------------------------
# "modes": each field = amp * sum_{m=1..8} cos(k_m . x + phi_m) / sqrt(8)   (C1, C2)
# ------------------------------------------------------------------------------------------
def draw_modes(seed: int, nmodes: int = 8, kmax: int = 4):
    """Per field: integer wave-vectors uniform in the ball 0 < |k| <= kmax and phases in [0, 2 pi).
    Returns (k, phi): k int array (4, nmodes, 3) in (kx, ky, kz) order, phi (4, nmodes)."""
    rng = np.random.default_rng(seed)
    k = np.zeros((4, nmodes, 3), dtype=np.int64)
    phi = np.zeros((4, nmodes))
    for f in range(4):
        for m in range(nmodes):
            while True:
                kv = rng.integers(-kmax, kmax + 1, 3)
                if 0 < int(kv @ kv) <= kmax * kmax:
                    break
            k[f, m] = kv
            phi[f, m] = rng.uniform(0.0, TWO_PI)
    return k, phi


def mode_sum_state(n: int, k, phi, amp: float, dtype=np.float64):
    """Evaluate the mode sums on the n^3 grid x_i = i * 2 pi / n (in float64, then rounded to dtype)."""
    g = np.arange(n) * (TWO_PI / n)
    Z, Y, X = np.meshgrid(g, g, g, indexing="ij")
    nm = k.shape[1]
    F = np.zeros((4, n, n, n))
    for f in range(4):
        for m in range(nm):
            F[f] += np.cos(k[f, m, 0] * X + k[f, m, 1] * Y + k[f, m, 2] * Z + phi[f, m])
    F *= amp / math.sqrt(nm)
    return F.astype(dtype)


# ------------------------------------------------------------------------------------------
# "band": iid complex Gaussian Fourier coefficients on 0 < |k| <= kmax, zero elsewhere (C3..C5)
# ------------------------------------------------------------------------------------------
def band_limited_state(n: int, kmax: int, seed: int, mach_rms: float, lnrho_rms: float, cs: float = 1.0,
                       dtype="f32", device="cpu"):
    """Returns a torch tensor (4, n, n, n) on `device`.  u is scaled so that sqrt(<|u|^2>) = mach_rms*cs
    (|u|^2 = ux^2+uy^2+uz^2); ln rho has rms lnrho_rms (identically 0 if lnrho_rms == 0).
    The arrays this returns ARE the input: the same bits go to fd_load and to the oracle."""
    import torch

    rdt = torch.float32 if dtype == "f32" else torch.float64
    cdt = torch.complex64 if dtype == "f32" else torch.complex128
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    kfull = torch.fft.fftfreq(n, d=1.0 / n, device=device)
    khalf = torch.fft.rfftfreq(n, d=1.0 / n, device=device)
    k2 = kfull[:, None, None] ** 2 + kfull[None, :, None] ** 2 + khalf[None, None, :] ** 2
    mask = ((k2 > 0) & (k2 <= float(kmax * kmax))).to(rdt)
    out = torch.empty((4, n, n, n), dtype=rdt, device=device)
    for f in range(4):
        re = torch.randn((n, n, n // 2 + 1), generator=gen, dtype=rdt, device=device)
        im = torch.randn((n, n, n // 2 + 1), generator=gen, dtype=rdt, device=device)
        coef = torch.complex(re * mask, im * mask).to(cdt)
        del re, im
        out[f] = torch.fft.irfftn(coef, s=(n, n, n))
        del coef
    if lnrho_rms > 0.0:
        out[0] *= lnrho_rms / out[0].double().pow(2).mean().sqrt().to(rdt)
    else:
        out[0].zero_()
    u2 = (out[1].double().pow(2) + out[2].double().pow(2) + out[3].double().pow(2)).mean().sqrt()
    out[1:] *= (mach_rms * cs / u2).to(rdt)
    return out


def make_state(cfg: Config, device="cpu", n_override=None):
    """The config's initial state. "modes" configs return numpy (float64-evaluated, rounded to the config
    dtype); "band" configs return a torch tensor on `device`.  n_override shrinks the grid (same spectrum
    recipe) for tests that cannot afford the full size."""
    n = n_override or cfg.n
    if cfg.kind == "modes":
        k, phi = draw_modes(cfg.seed, 8, cfg.kmax)
        return mode_sum_state(n, k, phi, cfg.amp, cfg.np_dtype)
    return band_limited_state(n, cfg.kmax, cfg.seed, cfg.amp, cfg.lnrho_rms, cfg.cs, cfg.dtype, device)


def gather_block(F, origin, size):
    """Periodic gather of a cubic sub-block: F is (4, nz, ny, nx) numpy or torch; origin = (k0, j0, i0)
    may be negative or cross the seam.  Returns a numpy array (4, size, size, size) with the same bits."""
    nz, ny, nx = F.shape[1:]
    kk = (np.arange(size) + origin[0]) % nz
    jj = (np.arange(size) + origin[1]) % ny
    ii = (np.arange(size) + origin[2]) % nx
    if isinstance(F, np.ndarray):
        return np.ascontiguousarray(F[:, kk[:, None, None], jj[None, :, None], ii[None, None, :]])
    import torch
    dev = F.device
    tk = torch.as_tensor(kk, device=dev)[:, None, None]
    tj = torch.as_tensor(jj, device=dev)[None, :, None]
    ti = torch.as_tensor(ii, device=dev)[None, None, :]
    return F[:, tk, tj, ti].contiguous().cpu().numpy()
