"""ctypes binding of libfd6 (include/fd6.h): same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used for two things only:
device memory (its caching allocator is installed as the library's allocator hook) and streams (the
current torch stream is handed to fd_set_stream before every call).  There is no CPU fallback: if
libfd6.so is missing this module raises at import; without a CUDA device fd_create fails (FD_ECUDA).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libfd6.so")

FD_F32, FD_F64 = 0, 1
FD_PATH_55, FD_PATH_19 = 0, 1
FD_HOST, FD_DEVICE = 0, 1
FD_OK, FD_EINVAL, FD_ENOMEM, FD_ECUDA, FD_EUNSUPPORTED = 0, 1, 2, 3, 4
FD_VARIANT_AUTO, FD_VARIANT_DIRECT, FD_VARIANT_TILED, FD_VARIANT_PAIRED = 0, 1, 2, 3
FD_GRAPH_OFF, FD_GRAPH_WAITING, FD_GRAPH_CAPTURED, FD_GRAPH_FAILED = 0, 1, 2, 3
FD_K_PACK, FD_K_UNPACK, FD_K_HALO, FD_K_FUSED55, FD_K_PASS1, FD_K_PASS2, FD_K_COUNT = range(7)
KERNEL_NAMES = ["pack", "unpack", "halo", "fused55", "pass1_19", "pass2_19"]

EXPORTS = [
    "fd_set_allocator", "fd_create", "fd_set_path", "fd_set_variant", "fd_set_stream", "fd_load", "fd_store",
    "fd_rhs", "fd_rk3_step", "fd_sync", "fd_destroy", "fd_last_error", "fd_get_info", "fd_kernel_launches",
    "fd_set_profiling", "fd_get_profile", "fd_reset_profile",
    "fd_plan_work_list", "fd_set_forcing", "fd_set_graphs", "fd_set_tile_shape", "fd_rhs_static",
]

if not os.path.exists(_LIB_PATH):
    raise ImportError(
        f"{_LIB_PATH} is missing: build it with `python -m paper_1707_08900_b200.build` "
        "(libfd6 is CUDA-only; there is no CPU fallback)")

lib = C.CDLL(_LIB_PATH)


class FdInfo(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("dtype", C.c_int), ("path", C.c_int),
                ("variant", C.c_int), ("pitch_x", C.c_int), ("pitch_y", C.c_int), ("pitch_z", C.c_int),
                ("ghost_x", C.c_int), ("ghost_y", C.c_int), ("ghost_z", C.c_int),
                ("field_stride", C.c_size_t), ("device_bytes", C.c_size_t),
                ("tile_shape", C.c_int), ("tile_x", C.c_int), ("tile_y", C.c_int), ("work_items", C.c_int),
                ("graph_state", C.c_int), ("graph_note", C.c_char * 160)]


class FdWorkList(C.Structure):
    _fields_ = [(n, C.c_int) for n in ("tile_x", "tile_y", "tiles_x", "tiles_y", "planes", "full_tiles", "chunks",
                                       "chunk_planes", "items", "split_plane")]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_vp, _i, _d = C.c_void_p, C.c_int, C.c_double
lib.fd_set_allocator.argtypes = [ALLOC_FN, FREE_FN, _vp]
lib.fd_create.argtypes = [C.POINTER(_vp), _i, _i, _i, _d, _d, _d, _i]
lib.fd_set_path.argtypes = [_vp, _i]
lib.fd_set_variant.argtypes = [_vp, _i]
lib.fd_set_stream.argtypes = [_vp, _vp]
lib.fd_load.argtypes = [_vp, _vp, _vp, _vp, _vp, _i]
lib.fd_store.argtypes = [_vp, _vp, _vp, _vp, _vp, _i]
lib.fd_rhs.argtypes = [_vp, _vp, _vp, _vp, _vp, _i]
lib.fd_rk3_step.argtypes = [_vp, _d, _i]
lib.fd_sync.argtypes = [_vp]
lib.fd_destroy.argtypes = [_vp]
lib.fd_last_error.restype = C.c_char_p
lib.fd_get_info.argtypes = [_vp, C.POINTER(FdInfo)]
lib.fd_kernel_launches.argtypes = [_vp]
lib.fd_kernel_launches.restype = C.c_ulonglong
lib.fd_set_profiling.argtypes = [_vp, _i]
lib.fd_get_profile.argtypes = [_vp, _i, C.POINTER(_d), C.POINTER(C.c_ulonglong)]
lib.fd_reset_profile.argtypes = [_vp]
lib.fd_set_graphs.argtypes = [_vp, _i]
lib.fd_set_tile_shape.argtypes = [_vp, _i]
lib.fd_set_forcing.argtypes = [_vp, C.POINTER(_d), C.POINTER(_d), _d, _d, _d]
lib.fd_plan_work_list.argtypes = [_i, _i, _i, _i, _i, C.POINTER(FdWorkList)]
lib.fd_rhs_static.argtypes = [_i, _i, _i, _d, _d, _d, _i] + [_vp] * 9
FD_RHS_STATIC_MAX_BYTES = 8 * 1024 * 1024


def fd_plan_work_list(nx, ny, nz, dtype, sm_count):
    """Work list of the tiled kernels for a grid (host arithmetic only; needs no CUDA device)."""
    wl = FdWorkList()
    code = lib.fd_plan_work_list(nx, ny, nz, dtype, sm_count, C.byref(wl))
    if code != FD_OK:
        raise FdError(code, lib.fd_last_error().decode())
    return wl


class FdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libfd6 error {code}: {msg}")
        self.code = code


def _check(rc):
    if rc != FD_OK:
        raise FdError(rc, lib.fd_last_error().decode())


def fd_last_error() -> str:
    return lib.fd_last_error().decode()


# -- PyTorch as the device-memory provider --------------------------------------------------------
_hooks = None


def use_torch_allocator():
    """Install torch's CUDA caching allocator as the library's allocator (idempotent)."""
    global _hooks
    if _hooks is not None:
        return
    import torch

    def _alloc(nbytes, stream, _user):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return None

    def _free(ptr, _user):
        torch.cuda.caching_allocator_delete(int(ptr))

    _hooks = (ALLOC_FN(_alloc), FREE_FN(_free))
    _check(lib.fd_set_allocator(_hooks[0], _hooks[1], None))


def _ptr(a, where):
    """Pointer of one field given as numpy array (host), torch tensor (host or device) or int."""
    if isinstance(a, (int, np.integer)):
        return int(a)
    if isinstance(a, np.ndarray):
        assert where == FD_HOST and a.flags.c_contiguous
        return a.ctypes.data
    assert a.is_contiguous()
    assert (a.device.type == "cuda") == (where == FD_DEVICE)
    return a.data_ptr()


def fd_rhs_static(nx, ny, nz, dx, nu, cs, dtype, state, out):
    """fd_rhs_static of include/fd6.h: the 55-point right-hand side for callers that cannot allocate device memory
    (a plug-in inside an application that owns all of the GPU's memory, a loop that must stay clear of cudaMalloc's
    device-wide synchronisation).  No context, no allocation: the padded copy of the state lives in an 8 MiB array
    built into libfd6.so, which limits the grid (about 64^3 fp32 / 48^3 fp64) and is shared by all calls on a device,
    so calls that could overlap on the GPU must be ordered by the caller.  `state` and `out` are four dense CUDA
    tensors each (or device addresses) on the current device; the work is enqueued on torch's current stream."""
    import torch
    ptrs = [_ptr(a, FD_DEVICE) for a in tuple(state) + tuple(out)]
    _check(lib.fd_rhs_static(int(nx), int(ny), int(nz), float(dx), float(nu), float(cs), int(dtype), *ptrs,
                             torch.cuda.current_stream().cuda_stream))


class Fd:
    """One libfd6 context.  Methods mirror the C entry points one to one."""

    def __init__(self, nx, ny, nz, dx, nu, cs, dtype=FD_F32, torch_allocator=True):
        if torch_allocator:
            import torch
            if torch.cuda.is_available():
                torch.cuda.init()
                use_torch_allocator()
        self._h = _vp()
        self.dtype = dtype
        self.shape = (nz, ny, nx)
        _check(lib.fd_create(C.byref(self._h), nx, ny, nz, float(dx), float(nu), float(cs), dtype))

    # stream plumbing: the library works on torch's current stream
    def _stream(self):
        import torch
        _check(lib.fd_set_stream(self._h, torch.cuda.current_stream().cuda_stream))

    def fd_set_path(self, path):
        self._stream()
        _check(lib.fd_set_path(self._h, path))

    def fd_set_variant(self, variant):
        self._stream()  # a switch of layout converts the resident state on the stream
        _check(lib.fd_set_variant(self._h, variant))

    def fd_set_tile_shape(self, shape):
        self._stream()
        _check(lib.fd_set_tile_shape(self._h, int(shape)))

    def fd_set_graphs(self, on):
        _check(lib.fd_set_graphs(self._h, int(bool(on))))

    def fd_set_forcing(self, k, e, phi, f0, dt_ref):
        """Forcing term of Eq. 2 (Eq. 24-25); f0 = 0 switches it off (k, e may then be None)."""
        self._stream()
        kv = (C.c_double * 3)(*[float(v) for v in k]) if k is not None else None
        ev = (C.c_double * 3)(*[float(v) for v in e]) if e is not None else None
        _check(lib.fd_set_forcing(self._h, kv, ev, float(phi), float(f0), float(dt_ref)))

    def fd_load(self, lnrho, ux, uy, uz, where):
        self._stream()
        _check(lib.fd_load(self._h, *[_ptr(a, where) for a in (lnrho, ux, uy, uz)], where))

    def fd_store(self, lnrho, ux, uy, uz, where):
        self._stream()
        _check(lib.fd_store(self._h, *[_ptr(a, where) for a in (lnrho, ux, uy, uz)], where))

    def fd_rhs(self, r0, r1, r2, r3, where):
        self._stream()
        _check(lib.fd_rhs(self._h, *[_ptr(a, where) for a in (r0, r1, r2, r3)], where))

    def fd_rk3_step(self, dt, nsteps=1):
        self._stream()
        _check(lib.fd_rk3_step(self._h, float(dt), int(nsteps)))

    def fd_sync(self):
        _check(lib.fd_sync(self._h))

    def fd_get_info(self):
        info = FdInfo()
        _check(lib.fd_get_info(self._h, C.byref(info)))
        return info

    def fd_kernel_launches(self):
        return int(lib.fd_kernel_launches(self._h))

    def fd_set_profiling(self, on):
        _check(lib.fd_set_profiling(self._h, int(bool(on))))

    def fd_get_profile(self, kernel_id):
        ms, n = _d(), C.c_ulonglong()
        _check(lib.fd_get_profile(self._h, kernel_id, C.byref(ms), C.byref(n)))
        return ms.value, int(n.value)

    def fd_reset_profile(self):
        _check(lib.fd_reset_profile(self._h))

    def fd_destroy(self):
        if self._h:
            lib.fd_destroy(self._h)
            self._h = _vp()

    # conveniences (marshalling only): whole state as one (4,nz,ny,nx) array
    def np_dtype(self):
        return np.float32 if self.dtype == FD_F32 else np.float64

    def load_state(self, F):
        """F: numpy (host) or torch tensor (host or device) of shape (4,nz,ny,nx), C-contiguous, library dtype."""
        where = FD_DEVICE if (not isinstance(F, np.ndarray) and F.device.type == "cuda") else FD_HOST
        assert tuple(F.shape) == (4,) + self.shape
        self.fd_load(F[0], F[1], F[2], F[3], where)

    def store_state(self, out=None):
        if out is None:
            out = np.empty((4,) + self.shape, dtype=self.np_dtype())
        where = FD_DEVICE if (not isinstance(out, np.ndarray) and out.device.type == "cuda") else FD_HOST
        self.fd_store(out[0], out[1], out[2], out[3], where)
        return out

    def rhs_state(self, out=None):
        if out is None:
            out = np.empty((4,) + self.shape, dtype=self.np_dtype())
        where = FD_DEVICE if (not isinstance(out, np.ndarray) and out.device.type == "cuda") else FD_HOST
        self.fd_rhs(out[0], out[1], out[2], out[3], where)
        return out

    def __del__(self):
        try:
            self.fd_destroy()
        except Exception:
            pass
