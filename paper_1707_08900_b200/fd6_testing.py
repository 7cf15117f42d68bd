"""ctypes binding of include/fd6_testing.h: the library's test hooks.  Not part of the product API; imported by tests/ only."""
import ctypes as C

from . import fd6

TEST_EXPORTS = ["fd_debug_poison_w", "fd_debug_poison_ghosts", "fd_debug_set_tile_overlap"]

fd6.lib.fd_debug_poison_w.argtypes = [C.c_void_p]
fd6.lib.fd_debug_poison_ghosts.argtypes = [C.c_void_p]
fd6.lib.fd_debug_set_tile_overlap.argtypes = [C.c_void_p, C.c_int]


def fd_debug_poison_w(ctx: "fd6.Fd") -> None:
    """NaN into the w arrays (alpha_1 = 0: must not reach a result)."""
    ctx._stream()
    fd6._check(fd6.lib.fd_debug_poison_w(ctx._h))


def fd_debug_poison_ghosts(ctx: "fd6.Fd") -> None:
    """NaN into every ghost cell of both field copies (the library must refill every ghost it reads)."""
    ctx._stream()
    fd6._check(fd6.lib.fd_debug_poison_ghosts(ctx._h))


def fd_debug_set_tile_overlap(ctx: "fd6.Fd", overlap: int) -> None:
    """Overlapping tiles (same results, redundant halo-ring work): the temporal-blocking emulation of DESIGN.md section 7."""
    ctx._stream()
    fd6._check(fd6.lib.fd_debug_set_tile_overlap(ctx._h, int(overlap)))
