/* fd6.h — C ABI of libfd6: the hot path of arXiv 1707.08900 on one B200 (sm_100a).
 *
 * One 2N-storage RK3 step of isothermal compressible hydrodynamics,
 *     D ln(rho)/Dt = -div u                                              (Eq. 1)
 *     D u/Dt = -cs^2 grad ln(rho) + nu (lap u + 1/3 grad div u + 2 S.grad ln(rho))   (Eq. 2-3; f = 0)
 * on a periodic nx*ny*nz grid with cubic cells of size dx, sixth-order central differences
 * (Eq. 6-8), in one of the paper's two stencil paths:
 *     FD_PATH_55  single fused pass per substep, mixed derivatives by Eq. 8   (Alg. 2)
 *     FD_PATH_19  two passes per substep, grad(div u) by Eq. 6 applied twice  (Alg. 3, Eq. 14-18)
 * and the update  w <- alpha_s w + dt*rhs ; F <- F + beta_s w,  s = 1..3, alpha_1 = 0   (Eq. 10)
 * with Williamson's coefficients alpha = (0,-5/9,-153/128), beta = (1/3,15/16,8/15) (reading G2).
 *
 * Conventions for every call
 *   - Caller arrays are dense, no ghost zone, x fastest: element (i,j,k) at i + nx*(j + ny*k); one array per
 *     field (structure of arrays); field order ln(rho), u_x, u_y, u_z; element type float
 *     (FD_F32) or double (FD_F64) as given to fd_create; nx*ny*nz elements each.
 *   - `where` says where the caller's pointers live: FD_HOST (pageable or pinned host memory; the call copies
 *     through the context's stream) or FD_DEVICE (device memory of the context's device).
 *   - Ownership: the caller owns its arrays; the context owns all device state (two ghost-padded copies of the
 *     four fields, four dense w arrays, one ghost-padded div array once FD_PATH_19 is selected).  w is scratch
 *     between steps: fd_load, fd_store(FD_HOST) and fd_rhs overwrite it (legal because alpha_1 = 0).
 *   - Work is enqueued on the context's stream (fd_set_stream; default: the legacy default stream).  Calls with
 *     FD_HOST pointers return after their copies completed; fd_rk3_step and calls with FD_DEVICE pointers may
 *     return before the work finished: use fd_sync or the stream.
 *   - Every function returns FD_OK or an error code, never throws, never aborts; fd_last_error() gives a
 *     thread-local message for the last failure.  There is no CPU fallback: without a CUDA device fd_create
 *     fails with FD_ECUDA.
 *   - A context is not thread-safe; distinct contexts are independent.
 */
#ifndef FD6_H
#define FD6_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fd_ctx fd_ctx; /* opaque, owned by the library */

enum { FD_F32 = 0, FD_F64 = 1 };          /* dtype */
enum { FD_PATH_55 = 0, FD_PATH_19 = 1 };  /* stencil path */
enum { FD_HOST = 0, FD_DEVICE = 1 };      /* where caller pointers live */
enum { FD_OK = 0, FD_EINVAL = 1, FD_ENOMEM = 2, FD_ECUDA = 3, FD_EUNSUPPORTED = 4 };

/* Kernel implementations of the derivative/update step (fd_set_variant).  All compute the same path;
 * FD_VARIANT_AUTO picks the fastest one that supports the grid (PAIRED for fp32 with an even nz, else TILED).
 * The device layout is private to the library: PAIRED stores cells (i,j,k) and (i,j,k+nz/2) side by side so
 * that one packed fp32x2 instruction works on both; switching variants converts a loaded state in place. */
enum {
    FD_VARIANT_AUTO = 0,
    FD_VARIANT_DIRECT = 1, /* one thread per cell (or pair), neighbours through L1/L2 (simple, any layout)    */
    FD_VARIANT_TILED = 2,  /* TMA-staged xy tiles in shared memory, register sliding window along z            */
    FD_VARIANT_PAIRED = 3  /* TILED on the paired fp32 layout with packed FFMA2 arithmetic (fp32, nz even)     */
};

/* Kernel ids for fd_get_profile. */
enum {
    FD_K_PACK = 0,    /* dense -> padded interior */
    FD_K_UNPACK = 1,  /* padded interior -> dense                         (a0)             */
    FD_K_HALO = 2,    /* periodic ghost fill: all faces and edges         (a1, a7)         */
    FD_K_FUSED55 = 3, /* Eq. 6-8 + Eq. 1-3 + Eq. 10, one pass             (a2-a4)          */
    FD_K_PASS1 = 4,   /* 19-pt pass 1: div u, partial update Eq. 14-16    (a6)             */
    FD_K_PASS2 = 5,   /* 19-pt pass 2: grad div by Eq. 6, Eq. 17-18       (a8)             */
    FD_K_COUNT = 6
};

/* Device-memory hooks.  alloc returns a device pointer aligned to >= 256 bytes or NULL; `stream` is the
 * context's stream handle (a cudaStream_t passed as void*).  Installed process-wide; a context keeps the pair
 * that was installed when it was created.  Passing NULLs restores cudaMalloc/cudaFree. */
typedef void* (*fd_alloc_fn)(size_t bytes, void* stream, void* user);
typedef void (*fd_free_fn)(void* ptr, void* user);
int fd_set_allocator(fd_alloc_fn alloc, fd_free_fn release, void* user);

/* Create a context for an nx*ny*nz periodic grid, cell size dx (= dy = dz), viscosity nu, sound speed cs.
 * FD_EINVAL: out == NULL, any n < 8, dx <= 0, nu < 0, cs < 0, non-finite parameter, bad dtype.
 * FD_EUNSUPPORTED: nx % 4 != 0, ny > 65535, nz > 16383 or more than 2^33 cells.  FD_ENOMEM / FD_ECUDA: allocation or CUDA
 * failure (message in fd_last_error).
 * The fields are zero (a uniform state at rest) until fd_load. */
int fd_create(fd_ctx** out, int nx, int ny, int nz, double dx, double nu, double cs, int dtype);

/* Select the stencil path (default FD_PATH_55) / kernel variant (default FD_VARIANT_AUTO) / stream.
 * fd_set_path(FD_PATH_19) allocates the div array on first use.  FD_EUNSUPPORTED if the variant cannot run this
 * grid.  `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream). */
int fd_set_path(fd_ctx* ctx, int path);
int fd_set_variant(fd_ctx* ctx, int variant);
int fd_set_stream(fd_ctx* ctx, void* cuda_stream);

/* Tile shape of the staged kernels (FD_VARIANT_TILED / FD_VARIANT_PAIRED): -1 automatic (default:
 * by the number of tiles the grid gives), 0 "wide" (12 warps, one value per thread), 1 "tall" (8 warps, two vertically
 * adjacent values per thread: fewer shared-memory loads per value, fewer and larger work items).  Results are bitwise
 * identical; plain fp32 grids (odd nz) have the wide shape only and ignore the request.  Re-prepares the launches of the
 * current variant.  FD_EINVAL: shape outside -1..1. */
int fd_set_tile_shape(fd_ctx* ctx, int shape);

/* Forcing term f of Eq. 2 (Eq. 24-25), frozen until the next call:
 *     f(x) = Re{ N f_k exp(i k.x + i phi) } = N f_k cos(k.x + phi),   x = (i, j, k) * dx (cell (0,0,0) at the origin),
 *     N = f0 cs sqrt(|k| cs / dt_ref),   f_k = (k x e) / sqrt(|k|^2 - (k.e)^2).
 * k, e: 3 doubles each (host); k should be 2 pi / (n dx) times integers for f to be periodic on the grid; dt_ref is the
 * step size N is formed with (normally the dt later given to fd_rk3_step).  f is added to the momentum right-hand side
 * on all three substeps of every following fd_rk3_step and to fd_rhs, on both stencil paths.  f0 = 0 switches the
 * forcing off (the default, and the setting of the paper's performance runs); k and e may then be NULL.
 * FD_EINVAL: f0 < 0 or not finite, NULL or non-finite k/e/phi, dt_ref <= 0, k parallel to e.  Synchronises the stream. */
int fd_set_forcing(fd_ctx* ctx, const double* k, const double* e, double phi, double f0, double dt_ref);

/* Copy the caller's four fields in (and fill the ghost zones) / copy the current fields out. */
int fd_load(fd_ctx* ctx, const void* lnrho, const void* ux, const void* uy, const void* uz, int where);
int fd_store(fd_ctx* ctx, void* lnrho, void* ux, void* uy, void* uz, int where);

/* Right-hand side of Eq. 1-3 of the current state with the selected path, into the caller's arrays.  The
 * state is not changed. */
int fd_rhs(fd_ctx* ctx, void* d_lnrho, void* d_ux, void* d_uy, void* d_uz, int where);

/* fd_rhs_static — the right-hand side of Eq. 1-3 by the fused 55-point stencil (Eq. 6-8, Alg. 2,
 * PAPER.md:97-108, 207-213) for callers that cannot allocate device memory.
 *
 * Why it exists.  Everything else in this header goes through fd_create, which allocates the ghost-padded field copies
 * and the w arrays (cudaMalloc, or the fd_set_allocator hook).  Some users of the library are not in a position to do
 * that: a solver plug-in inside an application that has given all device memory to its own pool and forbids further
 * driver allocations; a time loop that may not touch cudaMalloc / cudaFree because both synchronise the whole device and
 * stall every other stream; a job running so close to the memory limit that a late allocation could fail.  For them
 * this one call needs no context and allocates nothing — no cudaMalloc, no cudaFree, no allocating library routine:
 * the ghost-padded copy of the state that the stencil kernel reads lives in a fixed array inside libfd6.so itself.
 *
 * The price.  That array is FD_RHS_STATIC_MAX_BYTES (8 MiB) of device memory which every GPU that loads the library
 * keeps until the process exits, used or not, and it bounds the grid: the padded state, 4 fields of
 * px * (ny + 6) * (nz + 6) values (rounded up to a multiple of 256 bytes per field) with
 * px = nx + 16 rounded up to a multiple of 8 (FD_F32) or nx + 8 rounded up to a multiple of 4 (FD_F64), must fit —
 * e.g. up to 64^3 in FD_F32 or 48^3 in FD_F64 (BASELINE config C1, 32^3 FD_F64, takes 1.8 MiB).  Larger grids are
 * refused with FD_EUNSUPPORTED and a message that states both sizes; use fd_create + fd_rhs for them.
 *
 * Arguments.  nx, ny, nz, dx, nu, cs, dtype as for fd_create (same checks, same error codes).  lnrho, ux, uy, uz: the
 * state, and d_lnrho, d_ux, d_uy, d_uz: the result, are eight dense DEVICE arrays of nx*ny*nz elements in the layout
 * of "Conventions" above, owned by the caller, on the CURRENT device (the caller makes the device of its pointers and
 * of `cuda_stream` current before the call); the result arrays must not overlap each other or the state.  cuda_stream
 * is a cudaStream_t passed as void* (NULL = legacy default stream).  Three kernels are enqueued on it (copy into the
 * padded scratch, periodic halo fill, stencil + assembly straight into the result arrays) and the call returns without
 * waiting.  No forcing term.  Results agree with fd_rhs on FD_PATH_55 to rounding (same formulas and coefficients).
 *
 * First call on a device.  The first call on each device looks up the device address of the built-in array (once; this
 * may load the library's kernels onto that device).  Make that first call before starting any stream capture.
 *
 * Sharing.  All calls on a device use the same array, and it keeps whatever the last call left in it.  Nothing in it
 * has to start from zero: every value the stencil kernel reads is rewritten by the copy-in and the halo fill of the
 * same call (a test runs a small grid after a large one to show stale contents do not leak).  But two calls whose
 * kernels can overlap on the GPU — different streams without an ordering between them, or different host threads —
 * race on the array and give wrong results: keep the calls of one device on one stream, or order them with events.
 *
 * FD_EINVAL: a NULL pointer, any n < 8, dx <= 0, nu < 0, cs < 0, a non-finite parameter, bad dtype.
 * FD_EUNSUPPORTED: nx % 4 != 0, or the padded state exceeds FD_RHS_STATIC_MAX_BYTES.  FD_ECUDA: no device, the address
 * look-up or a launch failed (message in fd_last_error).  Argument errors are reported before any CUDA call. */
#define FD_RHS_STATIC_MAX_BYTES (8u * 1024u * 1024u)
int fd_rhs_static(int nx, int ny, int nz, double dx, double nu, double cs, int dtype,
                  const void* lnrho, const void* ux, const void* uy, const void* uz,
                  void* d_lnrho, void* d_ux, void* d_uy, void* d_uz, void* cuda_stream);

/* Advance nsteps full RK3 steps (3 substeps each) of size dt.  FD_EINVAL: nsteps < 0 or dt not finite. */
int fd_rk3_step(fd_ctx* ctx, double dt, int nsteps);

/* fd_rk3_step enqueues each step as ONE CUDA graph launch instead of its 6 (FD_PATH_55) or 15 (FD_PATH_19) kernel
 * launches: the launch rate is what bounds small grids (BASELINE configs C1, C2).  The graph is captured once dt, the
 * path, the variant and the forcing have been the same for 2 consecutive steps (those 2 steps run as plain launches) and
 * dropped when one of them changes; fd_get_info().graph_state tells which regime is active.  on = 0 switches to plain
 * launches; results are identical.  With profiling on (fd_set_profiling) plain launches are used regardless.  Default: on. */
int fd_set_graphs(fd_ctx* ctx, int on);

/* Block until everything enqueued by this context has finished; returns FD_ECUDA if a kernel faulted. */
int fd_sync(fd_ctx* ctx);

/* Release the context and its device memory.  fd_destroy(NULL) is FD_OK. */
int fd_destroy(fd_ctx* ctx);

/* Message of the last failing call on this thread ("" if none); static thread-local storage. */
const char* fd_last_error(void);

/* Introspection (read-only). */
typedef struct fd_info {
    int nx, ny, nz, dtype, path, variant; /* variant: the one AUTO resolved to            */
    int pitch_x, pitch_y, pitch_z;        /* padded array extents in values (a value = one cell, or a pair of
                                             cells in the paired layout, where pitch_z covers nz/2 planes)       */
    int ghost_x, ghost_y, ghost_z;        /* offset of cell (0,0,0) inside a padded array */
    size_t field_stride;                  /* elements between consecutive padded fields   */
    size_t device_bytes;                  /* device memory owned by the context           */
    /* what fd_rk3_step launches right now (appended fields; the ones above keep their offsets) */
    int tile_shape;                       /* staged kernels (TILED / PAIRED): 0 wide, 1 tall; -1: the direct kernels run   */
    int tile_x, tile_y;                   /* tile extents in stored values (0 for the direct kernels)                      */
    int work_items;                       /* launch grid of the staged main kernel = items of its work list (0: direct)    */
    int graph_state;                      /* FD_GRAPH_* below                                                               */
    char graph_note[160];                 /* FD_GRAPH_FAILED: why the capture failed ("" otherwise)                         */
} fd_info;
/* graph_state: how the NEXT fd_rk3_step with the same dt would be enqueued.  A step is captured into a CUDA graph only
 * after dt and every setting a step depends on have stayed the same for 2 consecutive steps, so that a driver which
 * changes dt or calls fd_set_forcing every step runs plain launches and never pays for a capture. */
enum {
    FD_GRAPH_OFF = 0,      /* fd_set_graphs(0): plain launches                                                   */
    FD_GRAPH_WAITING = 1,  /* on, parameters not yet stable for 2 steps (or profiling on): plain launches         */
    FD_GRAPH_CAPTURED = 2, /* one graph launch per step                                                          */
    FD_GRAPH_FAILED = 3    /* capture or instantiation failed for the current parameters: plain launches, not
                              retried until dt or a setting changes; fd_rk3_step still returns FD_OK              */
};
int fd_get_info(const fd_ctx* ctx, fd_info* out);

/* Work list of the STAGED kernels only (FD_VARIANT_TILED / FD_VARIANT_PAIRED; host arithmetic only,
 * needs no CUDA device).  It is a planning aid: it does not say which variant FD_VARIANT_AUTO resolves to (small grids
 * run the one-thread-per-cell kernels, which have no work list) nor which shape fd_set_tile_shape forced — for what a
 * context really launches read fd_get_info (variant, tile_shape, tile_x, tile_y, work_items).  The grid is cut
 * into tiles_x * tiles_y columns of tile_x * tile_y values and `planes` stored planes (nz, or nz/2 in the paired
 * fp32 layout, which is planned for fp32 with an even nz >= 8).  Item b of the 1-D launch grid is, for b < full_tiles, tile b
 * over all planes; otherwise, with j = b - full_tiles, tile full_tiles + j / chunks over planes
 * [(j % chunks) * chunk_planes, min(that + chunk_planes, planes)) — unless split_plane > 0, see below.  Every (tile,
 * plane) is covered exactly once.
 * FD_EINVAL: out == NULL, n < 8, sm_count < 1, bad dtype. */
typedef struct fd_work_list {
    int tile_x, tile_y, tiles_x, tiles_y, planes;
    int full_tiles, chunks, chunk_planes, items;
    int split_plane; /* 0, or the split list (grids with about as many tiles as SMs): full_tiles = 0, items = 2 * tiles;
                        item b < tiles is tile b over planes [0, split_plane), item tiles + b is tile b over
                        [split_plane, planes): the long parts are dispatched first, the short ones fill the idle SMs */
} fd_work_list;
int fd_plan_work_list(int nx, int ny, int nz, int dtype, int sm_count, fd_work_list* out);

/* Number of kernels this context has launched since creation (every kernel of the library counts). */
unsigned long long fd_kernel_launches(const fd_ctx* ctx);

/* Per-kernel device timing: with profiling on, every launch is bracketed by CUDA events on the context's
 * stream.  fd_get_profile synchronises, then returns the accumulated device milliseconds and launch count of
 * kernel `kernel_id` since the last fd_reset_profile. */
int fd_set_profiling(fd_ctx* ctx, int on);
int fd_get_profile(fd_ctx* ctx, int kernel_id, double* total_ms, unsigned long long* launches);
int fd_reset_profile(fd_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* FD6_H */
