"""Out-of-bounds WRITE check without compute-sanitizer (the GPU pool refuses it): every device allocation of a context
is served by a hook that pads it with 64 KB of canary bytes on both sides; after stepping, fd_rhs and fd_store on
ragged and many-tile shapes, on every variant, path and dtype, the canaries must be untouched.  (Stale READS are
covered by the NaN-poisoned ghosts and w of test_parity_gpu.py.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

PAD = 64 * 1024
CANARY = 0xA5


class GuardAllocator:
    """fd_set_allocator hooks: torch owns the memory, the library gets the middle of a padded block."""

    def __init__(self, fd6, torch):
        self.fd6, self.torch = fd6, torch
        self.blocks = {}
        self.alloc_fn = fd6.ALLOC_FN(self._alloc)
        self.free_fn = fd6.FREE_FN(self._free)
        self.freed_dirty = []

    def _alloc(self, nbytes, _stream, _user):
        t = self.torch.full((int(nbytes) + 2 * PAD,), CANARY, dtype=self.torch.uint8, device="cuda")
        p = t.data_ptr() + PAD
        assert p % 256 == 0
        self.blocks[p] = (t, int(nbytes))
        return p

    def _dirty(self, t, n):
        lo, hi = t[:PAD], t[PAD + n:]
        return int((lo != CANARY).sum().item()), int((hi != CANARY).sum().item())

    def _free(self, ptr, _user):
        t, n = self.blocks.pop(int(ptr))
        self.torch.cuda.synchronize()
        d = self._dirty(t, n)
        if d != (0, 0):
            self.freed_dirty.append((n, d))

    def check(self):
        self.torch.cuda.synchronize()
        bad = [(n, self._dirty(t, n)) for t, n in self.blocks.values()]
        return [b for b in bad if b[1] != (0, 0)] + self.freed_dirty

    def install(self):
        self.fd6.use_torch_allocator()  # so that Fd() does not install torch's hooks over ours
        assert self.fd6.lib.fd_set_allocator(self.alloc_fn, self.free_fn, None) == self.fd6.FD_OK

    def uninstall(self):
        assert self.fd6.lib.fd_set_allocator(self.fd6._hooks[0], self.fd6._hooks[1], None) == self.fd6.FD_OK


SHAPES = [(40, 13, 9), (8, 8, 8), (132, 70, 20), (72, 33, 41), (44, 9, 11),  # the ragged shapes of test_parity_gpu
          (512, 500, 16), (1024, 300, 8), (36, 1000, 10), (2048, 100, 9), (132, 2000, 12)]  # many tiles, few planes


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_no_write_outside_allocations(shape, dtype):
    import torch
    from paper_1707_08900_b200 import fd6
    guard = GuardAllocator(fd6, torch)
    guard.install()
    ran = 0
    try:
        nx, ny, nz = shape
        rng = np.random.default_rng(nx + ny + nz)
        F = (0.05 * rng.standard_normal((4, nz, ny, nx))).astype(np.float32 if dtype == "f32" else np.float64)
        ctx = fd6.Fd(nx, ny, nz, 0.2, 0.02, 1.0, fd6.FD_F32 if dtype == "f32" else fd6.FD_F64)
        assert guard.blocks, "the context did not allocate through the hook"
        for variant in (fd6.FD_VARIANT_DIRECT, fd6.FD_VARIANT_TILED, fd6.FD_VARIANT_PAIRED):
            try:
                ctx.fd_set_variant(variant)
            except fd6.FdError as e:
                assert e.code == fd6.FD_EUNSUPPORTED
                continue
            for path in (fd6.FD_PATH_55, fd6.FD_PATH_19):
                ctx.fd_set_path(path)
                for graphs in (True, False):
                    ctx.fd_set_graphs(graphs)
                    ctx.load_state(F)
                    ctx.fd_rk3_step(0.02, 3)  # with graphs on: two plain steps, then one captured step
                    ctx.rhs_state()
                    ctx.store_state()
                    ran += 1
                    assert guard.check() == [], f"canary overwritten: variant {variant}, path {path}, shape {shape}"
        ctx.fd_set_forcing((0.5, 0.25, 1.0), (0.0, 1.0, 0.0), 0.3, 0.02, 0.02)
        ctx.fd_rk3_step(0.02, 1)
        assert guard.check() == []
        ctx.fd_destroy()
        assert guard.check() == [] and not guard.blocks
    finally:
        guard.uninstall()
    assert ran >= 4


def test_guard_detects_a_stray_write():
    """Negative control: one byte written just outside an allocation is reported."""
    import torch
    from paper_1707_08900_b200 import fd6
    guard = GuardAllocator(fd6, torch)
    guard.install()
    try:
        ctx = fd6.Fd(16, 16, 16, 0.2, 0.02, 1.0, fd6.FD_F64)
        assert guard.check() == []
        t, n = next(iter(guard.blocks.values()))
        t[PAD + n] = 0  # first byte past the end
        bad = guard.check()
        assert len(bad) == 1 and bad[0][1] == (0, 1)
        t[PAD + n] = CANARY
        ctx.fd_destroy()
    finally:
        guard.uninstall()
