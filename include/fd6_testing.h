/* fd6_testing.h — test hooks of libfd6.  NOT part of the product ABI (include/fd6.h): nothing on the hot path calls
 * them; they exist so that the GPU tests can prove two properties of the kernels from outside the library.
 * The symbols are exported by the same libfd6.so; only tests/ and the testing module of the Python binding
 * (paper_1707_08900_b200/fd6_testing.py) declare them. */
#ifndef FD6_TESTING_H
#define FD6_TESTING_H

#include "fd6.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Overwrite the four w arrays with a quiet NaN: a following fd_rk3_step must still give finite, correct fields,
 * because alpha_1 = 0 means w is not read on the first substep (Eq. 10; reading G4).
 * Enqueued on the context's stream.  FD_EINVAL: ctx == NULL. */
int fd_debug_poison_w(fd_ctx* ctx);

/* Overwrite every ghost cell of both field copies with a quiet NaN: every ghost a kernel reads must have been
 * filled by the library's own periodic halo fill.  Enqueued on the context's stream; marks the
 * context as holding a non-zero state.  FD_EINVAL: ctx == NULL. */
int fd_debug_poison_ghosts(fd_ctx* ctx);

/* Measurement aid for DESIGN.md section 7 ("temporal blocking"): let neighbouring tiles of the staged kernels overlap by
 * `overlap` values in x and y (even, smaller than the tile; 0 = off, the product setting).  Every tile is still evaluated
 * in full, a value is stored by the tile that holds it furthest from its edge, so results are unchanged (bitwise) while
 * the launch does the redundant halo-ring work that the first of two fused substeps would have to do (overlap 6 = a
 * radius-3 ring).  fp64 and the paired fp32 layout only.  FD_EINVAL / FD_ECUDA with a message otherwise. */
int fd_debug_set_tile_overlap(fd_ctx* ctx, int overlap);

#ifdef __cplusplus
}
#endif
#endif /* FD6_TESTING_H */
