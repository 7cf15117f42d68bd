"""ctypes front end of the CPU oracle (oracle/fd_oracle.cpp) — TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module; the product package never does.  It holds no
arithmetic of the method: every number comes out of fd_oracle.cpp.

Array convention: a state is a numpy array of shape (4, nz, ny, nx), C-contiguous, so that
the flat index of component q is i + nx*(j + ny*k) (x fastest), q = 0: ln rho, 1..3: u_x,u_y,u_z
(PAPER.md:61-63, 189).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
PATH_55, PATH_19 = 0, 1
_lib = None


def lib():
    global _lib
    if _lib is None:
        import importlib.util
        spec = importlib.util.spec_from_file_location("_fd_oracle_build", os.path.join(_HERE, "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        _lib = C.CDLL(mod.build())
        d, i = C.c_double, C.c_int
        pd, pf = C.POINTER(C.c_double), C.POINTER(C.c_float)
        _lib.fdo_num_threads.restype = i
        _lib.fdo_set_num_threads.argtypes = [i]
        _lib.fdo_stencil_d1.restype = d
        _lib.fdo_stencil_d1.argtypes = [pd, d]
        _lib.fdo_stencil_d2.restype = d
        _lib.fdo_stencil_d2.argtypes = [pd, d]
        _lib.fdo_stencil_dmix.restype = d
        _lib.fdo_stencil_dmix.argtypes = [pd, pd, pd, pd, d]
        _lib.fdo_deriv_f64.argtypes = [i, i, i, i, i, i, d, pd, pd]
        _lib.fdo_rhs_f64.argtypes = [i, i, i, i, d, d, d] + [pd] * 8
        _lib.fdo_rhs_f32.argtypes = [i, i, i, i, d, d, d] + [pf] * 8
        _lib.fdo_rk3_step_f64.argtypes = [i, i, i, i, d, d, d, d, i] + [pd] * 8
        _lib.fdo_rk3_step_f32.argtypes = [i, i, i, i, d, d, d, d, i] + [pf] * 8
        _lib.fdo_rk3_linear.argtypes = [d, d, d, i, pd, pd]
        _lib.fdo_set_forcing.argtypes = [pd, pd, d, d, d, pd]
    return _lib


def num_threads() -> int:
    return int(lib().fdo_num_threads())


def set_num_threads(n: int) -> None:
    lib().fdo_set_num_threads(int(n))


def _p(a):
    ct = C.c_double if a.dtype == np.float64 else C.c_float
    return a.ctypes.data_as(C.POINTER(ct))


def _vec(v, n):
    a = np.ascontiguousarray(np.asarray(v, dtype=np.float64))
    assert a.shape == (n,)
    return a


def stencil_d1(v7, dx):
    """Eq. 6 on f(-3..3) supplied by the caller (non-periodic use)."""
    a = _vec(v7, 7)
    return float(lib().fdo_stencil_d1(_p(a), float(dx)))


def stencil_d2(v7, dx):
    """Eq. 7 on f(-3..3) supplied by the caller."""
    a = _vec(v7, 7)
    return float(lib().fdo_stencil_d2(_p(a), float(dx)))


def stencil_dmix(pp, mp, mm, pm, dx):
    """Eq. 8 on the 12 diagonal values: pp[m-1]=f(+m,+m), mp=f(-m,+m), mm=f(-m,-m), pm=f(+m,-m)."""
    a, b, c, d = (_vec(x, 3) for x in (pp, mp, mm, pm))
    return float(lib().fdo_stencil_dmix(_p(a), _p(b), _p(c), _p(d), float(dx)))


def deriv(f, kind, a, b=-1, dx=1.0):
    """One periodic derivative of a (nz,ny,nx) float64 field. Axis numbering: 0 = x (fastest), 1 = y, 2 = z."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    nz, ny, nx = f.shape
    out = np.empty_like(f)
    rc = lib().fdo_deriv_f64(kind, a, b, nx, ny, nz, float(dx), _p(f), _p(out))
    if rc:
        raise ValueError("fdo_deriv_f64: bad arguments")
    return out


class forcing:
    """Context manager: the forcing term of Eq. 2 (Eq. 24-25) for the oracle calls inside it.
    spec = dict(k=(kx,ky,kz), e=(ex,ey,ez), phi=..., f0=..., dt=...) or None; origin = cell offset of index 0."""

    def __init__(self, spec, origin=(0, 0, 0)):
        self.spec, self.origin = spec, origin

    def __enter__(self):
        if self.spec is not None:
            sp = self.spec
            rc = lib().fdo_set_forcing(_p(_vec(sp["k"], 3)), _p(_vec(sp["e"], 3)), float(sp["phi"]), float(sp["f0"]),
                                       float(sp["dt"]), _p(_vec(self.origin, 3)))
            if rc:
                raise ValueError("fdo_set_forcing: bad arguments")
        return self

    def __exit__(self, *a):
        z = _vec((0, 0, 0), 3)
        lib().fdo_set_forcing(_p(z), _p(z), 0.0, 0.0, 1.0, _p(z))


def _state(F, dtype):
    F = np.ascontiguousarray(F, dtype=dtype)
    assert F.ndim == 4 and F.shape[0] == 4, "state must have shape (4, nz, ny, nx)"
    return F


def rhs(F, dx, nu, cs, path=PATH_55, dtype=np.float64, force=None):
    """Full right-hand side (Eq. 1-3, including nu/3 grad div u, plus the forcing `force` if given) of state F;
    returns (4,nz,ny,nx)."""
    F = _state(F, dtype)
    _, nz, ny, nx = F.shape
    R = np.empty_like(F)
    fn = lib().fdo_rhs_f64 if dtype == np.float64 else lib().fdo_rhs_f32
    with forcing(force):
        rc = fn(path, nx, ny, nz, float(dx), float(nu), float(cs), *[_p(F[q]) for q in range(4)], *[_p(R[q]) for q in range(4)])
    if rc:
        raise ValueError("fdo_rhs: bad arguments")
    return R


def rk3_step(F, dx, nu, cs, dt, nsteps=1, path=PATH_55, dtype=np.float64, W=None, return_w=False, force=None,
             origin=(0, 0, 0)):
    """nsteps full 2N-RK3 steps (Eq. 10, Alg. 2 / Alg. 3), with the frozen forcing `force` if given.
    Returns the new state (a copy)."""
    F = _state(F, dtype).copy()
    _, nz, ny, nx = F.shape
    W = np.zeros_like(F) if W is None else _state(W, dtype).copy()
    fn = lib().fdo_rk3_step_f64 if dtype == np.float64 else lib().fdo_rk3_step_f32
    with forcing(force, origin):
        rc = fn(path, nx, ny, nz, float(dx), float(nu), float(cs), float(dt), int(nsteps),
                *[_p(F[q]) for q in range(4)], *[_p(W[q]) for q in range(4)])
    if rc:
        raise ValueError("fdo_rk3_step: bad arguments")
    return (F, W) if return_w else F


def rk3_linear(lam, dt, nsteps, y0):
    """y' = lam*y advanced with the oracle's own RK3 update; complex in, complex out."""
    lam, y0 = complex(lam), complex(y0)
    yr, yi = C.c_double(y0.real), C.c_double(y0.imag)
    rc = lib().fdo_rk3_linear(lam.real, lam.imag, float(dt), int(nsteps), C.byref(yr), C.byref(yi))
    if rc:
        raise ValueError("fdo_rk3_linear: bad arguments")
    return complex(yr.value, yi.value)


def window_margin(path, nsteps=1, substeps=3):
    """Domain-of-dependence radius (cells) of `nsteps` RK3 steps: 3 per substep on the 55-point
    path, 6 on the 19-point path (div u with radius 3, then Eq. 6 on it with radius 3)."""
    return (3 if path == PATH_55 else 6) * substeps * nsteps


def rk3_step_window(Fsub, dx, nu, cs, dt, nsteps=1, path=PATH_55, dtype=np.float64):
    """Step a sub-block gathered (periodically) out of a large grid as if it were a small periodic
    box and return only the cells whose domain of dependence lies inside the block: the result
    there is identical to stepping the whole grid (the update is local).
    Returns (interior_result, margin)."""
    m = window_margin(path, nsteps)
    out = rk3_step(Fsub, dx, nu, cs, dt, nsteps, path, dtype)
    assert min(out.shape[1:]) > 2 * m, "window too small for its margin"
    return out[:, m:-m, m:-m, m:-m], m
