// fd6.cu — the C ABI of libfd6 (include/fd6.h): context, HBM layout, launch sequencing.
// Every step of the path runs in the kernels of fd6_kernels_*.cuh; this file only allocates, orders
// launches on the context's stream and swaps pointers.
#include "../../include/fd6.h"
#include "../../include/fd6_testing.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <type_traits>
#include <vector>

#include "fd6_common.cuh"
#include "fd6_kernels_direct.cuh"
#include "fd6_tiled_host.cuh"

using namespace fd6;

// ------------------------------------------------------------------------------------------------
// errors
// ------------------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define FD_CUDA(expr)                                                                                      \
    do {                                                                                                   \
        cudaError_t e__ = (expr);                                                                          \
        if (e__ != cudaSuccess) return fail(FD_ECUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

// ------------------------------------------------------------------------------------------------
// allocator hooks
// ------------------------------------------------------------------------------------------------
static fd_alloc_fn g_alloc = nullptr;
static fd_free_fn g_free = nullptr;
static void* g_alloc_user = nullptr;

extern "C" int fd_set_allocator(fd_alloc_fn alloc, fd_free_fn release, void* user) {
    if ((alloc == nullptr) != (release == nullptr)) return fail(FD_EINVAL, "fd_set_allocator: give both hooks or neither");
    g_alloc = alloc;
    g_free = release;
    g_alloc_user = user;
    return FD_OK;
}

// ------------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------------
struct ProfRec {
    int id;
    cudaEvent_t a, b;
};

struct StepGraph {
    cudaGraphExec_t exec = nullptr;
    unsigned long long launches = 0;  // kernels in the graph
};

struct fd_ctx {
    Geom g{};  // geometry in VALUES: cells, or V2 pairs of cells when `paired` (then g.nz = nz / 2)
    int nx = 0, ny = 0, nz = 0;  // the caller's grid
    bool paired = false;         // fp32 paired layout: value (i,j,k) = cells (i,j,k) and (i,j,k+nz/2)
    bool loaded = false;         // a state other than the all-zero one is resident
    int dtype = FD_F32, path = FD_PATH_55, variant_req = FD_VARIANT_AUTO, variant = FD_VARIANT_DIRECT;
    double dx = 0, nu = 0, cs = 0;
    size_t esize = 4;            // bytes per value
    size_t f_bytes = 0, div_bytes = 0;  // allocation sizes (cover both layouts)
    cudaStream_t stream = nullptr;
    void* F[2] = {nullptr, nullptr};  // two ghost-padded copies of the four fields (read / write)
    void* W = nullptr;                // four dense w arrays
    void* Div = nullptr;              // ghost-padded div u (19-point path only)
    int cur = 0;                      // F[cur] holds the current state with valid ghosts
    size_t bytes = 0;
    fd_alloc_fn alloc = nullptr;
    fd_free_fn release = nullptr;
    void* alloc_user = nullptr;
    unsigned long long launches = 0;
    bool profiling = false;
    std::vector<ProfRec> pending;
    std::vector<cudaEvent_t> pool;
    double prof_ms[FD_K_COUNT] = {};
    unsigned long long prof_n[FD_K_COUNT] = {};
    TiledState tiled;  // tensor maps etc. of the tiled variant
    // forcing term of Eq. 2 (fd_set_forcing): amplitude N f_k and the device table of the separable phase
    bool force_on = false;
    double famp[3] = {0, 0, 0};
    void* ftab = nullptr;
    // CUDA graphs of one full RK3 step (fd_set_graphs): graph[b] starts from read copy b and ends on
    // copy 1 - b.  Captured on a stream of the library's own (the caller's may be the legacy default stream, which
    // cannot capture) and launched on the context's stream; rebuilt when dt or anything the launches depend on changes.
    bool graphs_on = true;
    StepGraph graph[2];
    double graph_dt = 0;
    unsigned long long epoch = 0, graph_epoch = ~0ULL;  // epoch: bumped by every setter that changes what a step launches
    cudaStream_t cap_stream = nullptr;
    // A graph is captured only once (dt, epoch) have held for kGraphAfterSteps consecutive steps: a driver that changes dt or
    // the forcing every step (PAPER.md:460 draws a new forcing wavevector each step) would otherwise pay a capture and an
    // instantiation per step, which on small grids costs more than the plain launches the graph replaces.
    int stable_steps = 0;       // steps run with plain launches under (graph_dt, graph_epoch)
    bool graph_failed = false;  // capture or instantiation failed under (graph_dt, graph_epoch): plain launches, no retry
    char graph_note[160] = "";  // why, for fd_get_info
};

static const int kGraphAfterSteps = 2;

static int ctx_alloc(fd_ctx* c, void** p, size_t bytes) {
    *p = nullptr;
    if (c->alloc) {
        *p = c->alloc(bytes, (void*)c->stream, c->alloc_user);
        if (!*p) return fail(FD_ENOMEM, "allocator hook returned NULL for %zu bytes", bytes);
    } else {
        cudaError_t e = cudaMalloc(p, bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(e == cudaErrorMemoryAllocation ? FD_ENOMEM : FD_ECUDA, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e));
        }
    }
    c->bytes += bytes;
    return FD_OK;
}

static void ctx_free(fd_ctx* c, void* p) {
    if (!p) return;
    if (c->release)
        c->release(p, c->alloc_user);
    else
        cudaFree(p);
}

// RAII bracket that counts a launch and, with profiling on, times it with events on the context's stream.
struct LaunchScope {
    fd_ctx* c;
    int id;
    cudaEvent_t a = nullptr, b = nullptr;
    LaunchScope(fd_ctx* c_, int id_) : c(c_), id(id_) {
        c->launches++;
        if (!c->profiling) return;
        auto get = [&]() {
            cudaEvent_t e;
            if (!c->pool.empty()) {
                e = c->pool.back();
                c->pool.pop_back();
            } else {
                cudaEventCreate(&e);
            }
            return e;
        };
        a = get();
        b = get();
        cudaEventRecord(a, c->stream);
    }
    ~LaunchScope() {
        if (!a) return;
        cudaEventRecord(b, c->stream);
        c->pending.push_back({id, a, b});
    }
};

static int drain_profile(fd_ctx* c) {
    if (c->pending.empty()) return FD_OK;
    FD_CUDA(cudaStreamSynchronize(c->stream));
    for (auto& r : c->pending) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, r.a, r.b);
        c->prof_ms[r.id] += ms;
        c->prof_n[r.id]++;
        c->pool.push_back(r.a);
        c->pool.push_back(r.b);
    }
    c->pending.clear();
    return FD_OK;
}

// One RK substep as the host sees it (Eq. 10); see Sub<T> for the flags.
struct SubD {
    double alpha, beta, dt;
    int read_w, write_f, write_w;
};

template <class T>
static Coef<T> make_coef(const fd_ctx* c) {
    // Coefficients are formed in double and rounded once to the scalar type (reading G13: constant folding is free).
    typedef typename Scalar<T>::type S;
    const double dx = c->dx, dx2 = dx * dx;
    Coef<T> k;
    k.a1 = T(S(45.0 / (60.0 * dx)));
    k.a2 = T(S(-9.0 / (60.0 * dx)));
    k.a3 = T(S(1.0 / (60.0 * dx)));
    k.b0 = T(S(-490.0 / (180.0 * dx2)));
    k.b1 = T(S(270.0 / (180.0 * dx2)));
    k.b2 = T(S(-27.0 / (180.0 * dx2)));
    k.b3 = T(S(2.0 / (180.0 * dx2)));
    k.m1 = T(S(270.0 / (720.0 * dx2)));
    k.m2 = T(S(-27.0 / (720.0 * dx2)));
    k.m3 = T(S(2.0 / (720.0 * dx2)));
    k.nu = T(S(c->nu));
    k.nu3 = T(S(c->nu / 3.0));
    k.cs2 = T(S(c->cs * c->cs));
    for (int a = 0; a < 3; ++a) k.fa[a] = T(S(c->force_on ? c->famp[a] : 0.0));
    return k;
}

template <class T>
static Sub<T> make_sub(const SubD& d) {
    typedef typename Scalar<T>::type S;
    Sub<T> s;
    s.alpha = T(S(d.alpha));
    s.beta = T(S(d.beta));
    s.dt = T(S(d.dt));
    s.read_w = d.read_w;
    s.write_f = d.write_f;
    s.write_w = d.write_w;
    return s;
}

// Williamson 2N-RK3 (reading G2); written here and in the oracle independently.
static const double kAlpha[3] = {0.0, -5.0 / 9.0, -153.0 / 128.0};
static const double kBeta[3] = {1.0 / 3.0, 15.0 / 16.0, 8.0 / 15.0};

// Run `expr` with T = the value type of the context (float, double, or V2 in the paired layout).
#define FD_DISPATCH(c, expr)                   \
    ((c)->dtype == FD_F64 ? [&]() {            \
        typedef double T;                      \
        return (expr);                         \
    }()                                        \
     : (c)->paired ? [&]() {                   \
           typedef V2 T;                       \
           return (expr);                      \
       }()                                     \
                   : [&]() {                   \
                         typedef float T;      \
                         return (expr);        \
                     }())

// ------------------------------------------------------------------------------------------------
// geometry
// ------------------------------------------------------------------------------------------------
// HBM layout: 32-byte ghost pad in x so interior rows start sector-aligned and 16-byte vector /
// TMA accesses are legal; row pitch a multiple of 32 bytes; 3 ghost rows / planes in y and z.
static Geom make_geom(int nx, int ny, int nz, size_t esize, bool paired) {
    Geom g;
    const int e32 = (int)(32 / esize);
    g.nx = nx;
    g.ny = ny;
    g.nz = paired ? nz / 2 : nz;
    g.gx = e32;
    g.gy = R;
    g.gz = R;
    g.px = ((nx + 2 * g.gx + e32 - 1) / e32) * e32;
    g.py = ny + 2 * R;
    g.pz = g.nz + 2 * R;
    g.n = (long long)nx * ny * g.nz;
    long long fs = (long long)g.px * g.py * g.pz;
    const long long e256 = (long long)(256 / esize);
    g.fs = ((fs + e256 - 1) / e256) * e256;
    return g;
}

static bool pair_ok(const fd_ctx* c) { return c->dtype == FD_F32 && c->nz % 2 == 0 && c->nz / 2 >= 4; }

// ------------------------------------------------------------------------------------------------
// launch helpers (typed)
// ------------------------------------------------------------------------------------------------
template <class T>
static int launch_halo(fd_ctx* c, T* F, int nfields) {
    const Geom& g = c->g;
    LaunchScope ls(c, FD_K_HALO);
    const int yz_rows = 2 * R * g.py + 2 * R * g.nz;
    const long long xthreads = 2LL * g.ny * g.nz * nfields;
    // several ghost rows per block when a row has fewer 32-byte sectors than a block has threads (narrow grids)
    const int nsec = g.nx / g.gx + 2;
    int rpb = 1;
    while (rpb < 8 && 128 / (2 * rpb) >= nsec) rpb *= 2;
    const long long row_blocks = ((long long)nfields * yz_rows + rpb - 1) / rpb;
    const long long blocks = row_blocks + (xthreads + 127) / 128;
    k_halo<T><<<(unsigned)blocks, 128, 0, c->stream>>>(F, g, nfields, yz_rows, rpb, (int)row_blocks);
    FD_CUDA(cudaGetLastError());
    return FD_OK;
}

// One substep of the selected path: F[cur] (valid ghosts) -> F[1-cur] (+ghosts if write_f), w updated.
template <class T>
static int launch_substep(fd_ctx* c, const SubD& sd) {
    const Geom& g = c->g;
    const Coef<T> k = make_coef<T>(c);
    Sub<T> s = make_sub<T>(sd);
    const T* Fin = (const T*)c->F[c->cur];
    T* Fout = (T*)c->F[1 - c->cur];
    T* W = (T*)c->W;
    T* Div = (T*)c->Div;
    const bool p55 = c->path == FD_PATH_55;
    bool tiled = c->variant == FD_VARIANT_TILED || c->variant == FD_VARIANT_PAIRED;
    // forcing on a grid whose z phase table does not fit beside the rings in shared memory: under AUTO the
    // one-thread-per-cell kernels (which run on either layout) take the forced launches
    if (tiled && c->force_on && !c->tiled.force_fits && c->variant_req == FD_VARIANT_AUTO) tiled = false;
    ForceTab<T> ft;
    ft.tab = c->force_on ? (const typename Scalar<T>::type*)c->ftab : nullptr;
    ft.nx = c->nx;
    ft.ny = c->ny;
    ft.nzc = c->nz;
    const double no_force[3] = {0, 0, 0};
    dim3 block(64, 4, 1), grid((g.nx + 63) / 64, (g.ny + 3) / 4, g.nz);
    {
        LaunchScope ls(c, p55 ? FD_K_FUSED55 : FD_K_PASS1);
        if (tiled) {
            typedef typename Arith<T>::type A;  // the arithmetic type of the tiled kernels (V2 for plain fp32)
            const KC<A> kc = make_kc<A>(c->dx, c->nu, c->cs, p55, sd.dt, sd.alpha, sd.beta, sd.read_w, sd.write_f, sd.write_w,
                                        c->force_on ? c->famp : no_force);
            const int lrc = tiled_launch_main<T>(c->tiled, p55, c->cur, Fout, W, Div, g, kc, ft, c->stream);
            if (lrc == 4) return fail(FD_EUNSUPPORTED, "forcing on a grid with this many planes needs FD_VARIANT_DIRECT");
            if (lrc) return fail(FD_ECUDA, "tiled kernel launch failed: %s", tiled_error_of(c->tiled));
        } else if (p55) {
            k_direct_main<T, true><<<grid, block, 0, c->stream>>>(Fin, Fout, W, nullptr, g, k, s, ft);
        } else {
            k_direct_main<T, false><<<grid, block, 0, c->stream>>>(Fin, Fout, W, Div, g, k, s, ft);
        }
    }
    if (!p55) {
        int rc = launch_halo<T>(c, Div, 1);  // "Compute boundary conditions for (div u)" (Alg. 3)
        if (rc) return rc;
        if (tiled) s.dt = T(typename Scalar<T>::type(1));  // the tiled pass 1 leaves dt * div u in Div
        LaunchScope ls(c, FD_K_PASS2);
        // y bands of 16 block rows once seven div planes no longer fit comfortably in L2 (see k_direct_pass2)
        const int brows = (g.ny + 3) / 4;
        const bool banded = 7.0 * g.px * g.py * (double)c->esize > 32e6 && brows > 16 && (long long)((brows + 15) / 16) * g.nz <= 65535;
        const int band_rows = banded ? 16 : brows, bands = (brows + band_rows - 1) / band_rows;
        if constexpr (std::is_same<T, float>::value) {  // plain fp32: two x-adjacent cells per thread
            dim3 grid2((g.nx + 127) / 128, band_rows, bands * g.nz);
            k_direct_pass2_x2<<<grid2, block, 0, c->stream>>>(Div, Fout, W, g, k, s);
        } else if (const int zc = 16;  // planes per thread: 6 warm-up div loads per 16 planes, 16 chunk layers at C4
                   tiled && g.nx >= 128 &&
                   (long long)((g.nx + 127) / 128) * ((g.ny + 3) / 4) * ((g.nz + zc - 1) / zc) >= 4LL * std::max(c->tiled.sm_count, 1)) {
            // staged variants on rows wide enough to fill the block and grids that give every SM several blocks (C2's 128
            // blocks would not: 11887 -> 11264 Mcell/s, it keeps the kernel below): value pairs, z-marching (the seven div
            // planes of the z derivative stay in registers, so no y banding is needed to keep them in L2)
            dim3 grid2((g.nx + 127) / 128, (g.ny + 3) / 4, (g.nz + zc - 1) / zc);
            if (s.write_w)
                k_pass2_march<T, true><<<grid2, block, 0, c->stream>>>(Div, Fout, W, g, k, s, zc);
            else
                k_pass2_march<T, false><<<grid2, block, 0, c->stream>>>(Div, Fout, W, g, k, s, zc);
        } else {
            dim3 grid2((g.nx + 63) / 64, band_rows, bands * g.nz);
            k_direct_pass2<T><<<grid2, block, 0, c->stream>>>(Div, Fout, W, g, k, s);
        }
    }
    FD_CUDA(cudaGetLastError());
    if (s.write_f) {
        int rc = launch_halo<T>(c, Fout, 4);  // ghosts of the new state, ready for the next RHS (reading G12)
        if (rc) return rc;
        c->cur = 1 - c->cur;  // "swapped efficiently using pointers"
    }
    return FD_OK;
}

// The three substeps of one full RK3 step (Alg. 2 / Alg. 3), enqueued on the context's stream.
template <class T>
static int one_step(fd_ctx* c, double dt) {
    for (int s = 0; s < 3; ++s) {
        SubD sub;
        sub.alpha = kAlpha[s];
        sub.beta = kBeta[s];
        sub.dt = dt;
        sub.read_w = s != 0;   // alpha^(1) = 0: w is not read
        sub.write_w = s != 2;  // ... so the w of the last substep is never read either: not written
        sub.write_f = 1;
        int rc = launch_substep<T>(c, sub);
        if (rc) return rc;
    }
    return FD_OK;
}

static void drop_graphs(fd_ctx* c) {
    for (auto& g : c->graph) {
        if (g.exec) cudaGraphExecDestroy(g.exec);
        g = StepGraph();
    }
    c->graph_epoch = ~0ULL;
}

// Capture one step that starts from read copy `cur0` into c->graph[cur0].  Nothing runs; the context is unchanged.
// Returns FD_OK, or an error after which the caller falls back to plain launches.
template <class T>
static int build_graph(fd_ctx* c, double dt, int cur0) {
    if (!c->cap_stream) FD_CUDA(cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking));
    cudaStream_t user = c->stream;
    const int cur_save = c->cur;
    const unsigned long long launches0 = c->launches;
    const bool prof = c->profiling;
    FD_CUDA(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed));
    c->stream = c->cap_stream;
    c->cur = cur0;
    c->profiling = false;
    const int rc = one_step<T>(c, dt);
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    c->stream = user;
    c->cur = cur_save;
    c->profiling = prof;
    const unsigned long long n = c->launches - launches0;
    c->launches = launches0;
    if (rc != FD_OK || e != cudaSuccess || !g) {
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        return rc != FD_OK ? rc : fail(FD_ECUDA, "stream capture of an RK3 step failed: %s", cudaGetErrorString(e));
    }
    cudaGraphExec_t exec = nullptr;
    const cudaError_t ei = cudaGraphInstantiate(&exec, g, 0);
    cudaGraphDestroy(g);
    if (ei != cudaSuccess) {
        cudaGetLastError();
        return fail(FD_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(ei));
    }
    c->graph[cur0].exec = exec;
    c->graph[cur0].launches = n;
    return FD_OK;
}

template <class T>
static int do_rk3(fd_ctx* c, double dt, int nsteps) {
    int n = 0;
    // One graph launch per step instead of 6 (55-point) or 15 (19-point) kernel launches: what bounds small grids is
    // the launch rate.  Per-launch profiling needs the individual launches.
    if (c->graphs_on && !c->profiling && nsteps > 0) {
        if (c->graph_epoch != c->epoch || c->graph_dt != dt) {
            drop_graphs(c);  // nothing to destroy unless the previous parameters had lasted long enough to be captured
            c->graph_epoch = c->epoch;
            c->graph_dt = dt;
            c->stable_steps = 0;
            c->graph_failed = false;
            c->graph_note[0] = 0;
        }
        for (; n < nsteps && !c->graph_failed; ++n) {
            if (c->stable_steps < kGraphAfterSteps) {  // parameters not settled yet: plain launches, no capture cost
                int rc = one_step<T>(c, dt);
                if (rc) return rc;
                c->stable_steps++;
                continue;
            }
            StepGraph& g = c->graph[c->cur];
            if (!g.exec) {
                char keep[sizeof(g_err)];
                memcpy(keep, g_err, sizeof(keep));
                if (build_graph<T>(c, dt, c->cur) != FD_OK) {
                    // plain launches take over for as long as these parameters last (no retry per call); the failure is kept
                    // in the context (fd_get_info: graph_state, graph_note), and since this call still succeeds it
                    // does not leave a message in fd_last_error
                    c->graph_failed = true;
                    snprintf(c->graph_note, sizeof(c->graph_note), "%s", g_err);
                    memcpy(g_err, keep, sizeof(keep));
                    break;
                }
            }
            FD_CUDA(cudaGraphLaunch(g.exec, c->stream));
            c->launches += g.launches;
            c->cur = 1 - c->cur;  // three pointer swaps
        }
    }
    for (; n < nsteps; ++n) {
        int rc = one_step<T>(c, dt);
        if (rc) return rc;
    }
    if (nsteps > 0) c->loaded = true;
    return FD_OK;
}

// dense caller-layout arrays (4 x N scalars at src) -> F[cur] interior, then ghosts
template <class T>
static int do_pack(fd_ctx* c, const typename Scalar<T>::type* const src[4]) {
    const Geom& g = c->g;
    T* F = (T*)c->F[c->cur];
    {
        LaunchScope ls(c, FD_K_PACK);
        dim3 grid((g.nx + 127) / 128, g.ny, g.nz * 4);
        k_pack<T><<<grid, 128, 0, c->stream>>>(src[0], src[1], src[2], src[3], F, g);
    }
    FD_CUDA(cudaGetLastError());
    return launch_halo<T>(c, F, 4);
}

// padded (or, with the dense geometry of the w arrays, dense) values -> dense caller-layout arrays
template <class T>
static int do_unpack(fd_ctx* c, const T* F, const Geom& g, typename Scalar<T>::type* const dst[4]) {
    LaunchScope ls(c, FD_K_UNPACK);
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz * 4);
    k_unpack<T><<<grid, 128, 0, c->stream>>>(F, dst[0], dst[1], dst[2], dst[3], g);
    FD_CUDA(cudaGetLastError());
    return FD_OK;
}

static Geom dense_geom(const Geom& g) {  // the w arrays seen as "padded" arrays without ghosts
    Geom d = g;
    d.px = g.nx;
    d.py = g.ny;
    d.pz = g.nz;
    d.gx = d.gy = d.gz = 0;
    d.fs = g.n;
    return d;
}

template <class T>
static int do_load(fd_ctx* c, const void* const in[4], int where) {
    typedef typename Scalar<T>::type S;
    const size_t nscal = (size_t)c->nx * c->ny * c->nz;
    const size_t nb = nscal * sizeof(S);
    const S* src[4];
    for (int q = 0; q < 4; ++q) {
        if (where == FD_HOST) {
            S* stage = (S*)c->W + (size_t)q * nscal;  // w is scratch between steps (alpha_1 = 0)
            FD_CUDA(cudaMemcpyAsync(stage, in[q], nb, cudaMemcpyHostToDevice, c->stream));
            src[q] = stage;
        } else {
            src[q] = (const S*)in[q];
        }
    }
    int rc = do_pack<T>(c, src);
    if (rc) return rc;
    c->loaded = true;
    if (where == FD_HOST) FD_CUDA(cudaStreamSynchronize(c->stream));
    return FD_OK;
}

// four dense caller-layout arrays at `dense` (device) -> the caller's host arrays
template <class S>
static int copy_out(fd_ctx* c, const S* dense, void* const out[4]) {
    const size_t nscal = (size_t)c->nx * c->ny * c->nz;
    for (int q = 0; q < 4; ++q)
        FD_CUDA(cudaMemcpyAsync(out[q], dense + (size_t)q * nscal, nscal * sizeof(S), cudaMemcpyDeviceToHost, c->stream));
    FD_CUDA(cudaStreamSynchronize(c->stream));
    return FD_OK;
}

template <class T>
static int do_store(fd_ctx* c, void* const out[4], int where) {
    typedef typename Scalar<T>::type S;
    const size_t nscal = (size_t)c->nx * c->ny * c->nz;
    S* dst[4];
    for (int q = 0; q < 4; ++q) dst[q] = where == FD_HOST ? (S*)c->W + (size_t)q * nscal : (S*)out[q];
    int rc = do_unpack<T>(c, (const T*)c->F[c->cur], c->g, dst);
    if (rc) return rc;
    return where == FD_HOST ? copy_out<S>(c, (const S*)c->W, out) : FD_OK;
}

template <class T>
static int do_rhs(fd_ctx* c, void* const out[4], int where) {
    typedef typename Scalar<T>::type S;
    SubD sub;
    sub.alpha = 0;
    sub.beta = 0;
    sub.dt = 1;
    sub.read_w = 0;
    sub.write_w = 1;
    sub.write_f = 0;  // w <- rhs, state untouched
    int rc = launch_substep<T>(c, sub);
    if (rc) return rc;
    const size_t nscal = (size_t)c->nx * c->ny * c->nz;
    if constexpr (Scalar<T>::lanes == 1) {  // the w arrays already are in the caller's layout
        for (int q = 0; q < 4; ++q)
            FD_CUDA(cudaMemcpyAsync(out[q], (const S*)c->W + (size_t)q * nscal, nscal * sizeof(S),
                                    where == FD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->stream));
        if (where == FD_HOST) FD_CUDA(cudaStreamSynchronize(c->stream));
        return FD_OK;
    } else {
        // paired layout: un-pair w; the write copy of the fields is free scratch for the host staging
        S* dst[4];
        for (int q = 0; q < 4; ++q) dst[q] = where == FD_HOST ? (S*)c->F[1 - c->cur] + (size_t)q * nscal : (S*)out[q];
        rc = do_unpack<T>(c, (const T*)c->W, dense_geom(c->g), dst);
        if (rc) return rc;
        return where == FD_HOST ? copy_out<S>(c, (const S*)c->F[1 - c->cur], out) : FD_OK;
    }
}

// Switch between the plain and the paired layout, carrying a loaded state across through the w scratch.
static int set_layout(fd_ctx* c, bool paired) {
    if (paired == c->paired) return FD_OK;
    const size_t nscal = (size_t)c->nx * c->ny * c->nz;
    void* dense[4];
    for (int q = 0; q < 4; ++q) dense[q] = (char*)c->W + (size_t)q * nscal * 4;  // fp32 only
    int rc = FD_OK;
    if (c->loaded) {
        rc = FD_DISPATCH(c, do_store<T>(c, dense, FD_DEVICE));
        if (rc) return rc;
    }
    c->paired = paired;
    c->esize = paired ? 8 : 4;
    c->g = make_geom(c->nx, c->ny, c->nz, c->esize, paired);
    // ghost cells of the other layout are interior cells of this one: start both copies from zero again
    FD_CUDA(cudaMemsetAsync(c->F[1 - c->cur], 0, c->f_bytes, c->stream));
    if (c->Div) FD_CUDA(cudaMemsetAsync(c->Div, 0, c->div_bytes, c->stream));
    if (c->loaded) {
        FD_CUDA(cudaMemsetAsync(c->F[c->cur], 0, c->f_bytes, c->stream));
        rc = FD_DISPATCH(c, do_load<T>(c, (const void* const*)dense, FD_DEVICE));
    }
    return rc;
}

// Pick the kernel variant and bring layout, tensor maps and work list in line with it.  Nothing is changed
// unless the whole switch succeeds: an unsupported target is refused before the layout is touched, and if the
// tensor-map setup fails afterwards the previous layout and variant are restored (c->variant, c->paired and
// c->tiled always describe the same kernels).
static int resolve_variant(fd_ctx* c) {
    // Whatever happens below (also on the failure paths, which may have converted the layout or re-made the tensor maps
    // before giving up), a step captured earlier no longer describes what a step launches.
    c->epoch++;
    int want = c->variant_req;
    const bool is_auto = want == FD_VARIANT_AUTO;
    if (is_auto) {
        // Grids of a few ten thousand cells per SM-wave are bound by the fixed cost of a tiled launch (tensor-memory
        // allocation, six warm-up planes per z chunk): below ~50^3 (fp64) / ~69^3 (fp32) cells the one-thread-per-cell
        // kernels are faster (measured on B200); above, the staged kernels win by up to 4x.
        const long long cells = (long long)c->nx * c->ny * c->nz;
        const bool tiny = cells <= (c->dtype == FD_F64 ? 131072LL : 327680LL);
        want = tiny ? FD_VARIANT_DIRECT : pair_ok(c) ? FD_VARIANT_PAIRED : FD_VARIANT_TILED;
        if (tiny)
            snprintf(c->tiled.err, sizeof(c->tiled.err), "automatic variant: grids of at most %lld cells run the one-thread-per-cell kernels",
                     c->dtype == FD_F64 ? 131072LL : 327680LL);
    }
    if (want == FD_VARIANT_PAIRED && !pair_ok(c))
        return fail(FD_EUNSUPPORTED, "paired variant needs fp32 and an even nz >= 8 (got dtype %d, nz %d)", c->dtype, c->nz);
    if (want == FD_VARIANT_TILED || want == FD_VARIANT_PAIRED) {
        const bool tp = want == FD_VARIANT_PAIRED;
        const Geom tg = make_geom(c->nx, c->ny, c->nz, tp ? 8 : (c->dtype == FD_F32 ? 4 : 8), tp);
        if (!tiled_supported(tg)) {  // checked on the TARGET layout, before anything is converted
            if (!is_auto)
                return fail(FD_EUNSUPPORTED,
                            "tiled variant cannot run this grid in the %s layout: it needs >= 4 values per axis and "
                            "4 * padded field size < 2^32 values (the kernels use 32-bit store offsets)", tp ? "paired" : "plain");
            snprintf(c->tiled.err, sizeof(c->tiled.err), "automatic variant: the staged kernels need >= 4 values per axis and 4 * padded field size < 2^32 values");
            want = FD_VARIANT_DIRECT;
        }
    }
    if (want == FD_VARIANT_TILED || want == FD_VARIANT_PAIRED) {
        const bool was_paired = c->paired;
        const int was_variant = c->variant;
        int rc = set_layout(c, want == FD_VARIANT_PAIRED);
        if (rc) return rc;
        rc = FD_DISPATCH(c, tiled_prepare<T>(c->tiled, c->g, c->F[0], c->F[1], c->W));
        if (rc != FD_OK) {
            char why[256];
            snprintf(why, sizeof(why), "%s", tiled_error_of(c->tiled));
            if (is_auto) {
                want = FD_VARIANT_DIRECT;  // runs on either layout
            } else {
                int rb = set_layout(c, was_paired);
                if (rb == FD_OK && (was_variant == FD_VARIANT_TILED || was_variant == FD_VARIANT_PAIRED))
                    rb = FD_DISPATCH(c, tiled_prepare<T>(c->tiled, c->g, c->F[0], c->F[1], c->W));
                if (rb != FD_OK) c->variant = FD_VARIANT_DIRECT;  // last resort: the direct kernels need no setup
                return fail(FD_ECUDA, "tiled variant setup failed: %s", why);
            }
        }
    }
    c->variant = want;
    return FD_OK;
}

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
#define FD_CHECK_CTX(c) \
    if (!(c)) return fail(FD_EINVAL, "%s: ctx is NULL", __func__)

extern "C" const char* fd_last_error(void) { return g_err; }

extern "C" int fd_create(fd_ctx** out, int nx, int ny, int nz, double dx, double nu, double cs, int dtype) {
    if (!out) return fail(FD_EINVAL, "fd_create: out is NULL");
    *out = nullptr;
    if (nx < 8 || ny < 8 || nz < 8) return fail(FD_EINVAL, "fd_create: every axis needs n >= 8 (got %d,%d,%d)", nx, ny, nz);
    if (!(dx > 0) || !std::isfinite(dx)) return fail(FD_EINVAL, "fd_create: dx must be finite and > 0");
    if (!(nu >= 0) || !std::isfinite(nu)) return fail(FD_EINVAL, "fd_create: nu must be finite and >= 0");
    if (!(cs >= 0) || !std::isfinite(cs)) return fail(FD_EINVAL, "fd_create: cs must be finite and >= 0");
    if (dtype != FD_F32 && dtype != FD_F64) return fail(FD_EINVAL, "fd_create: bad dtype %d", dtype);
    if (nx % 4 != 0) return fail(FD_EUNSUPPORTED, "fd_create: nx must be a multiple of 4 (got %d)", nx);
    if ((long long)nx * ny * nz > (1LL << 33)) return fail(FD_EUNSUPPORTED, "fd_create: grid too large");
    // launch grids put rows in gridDim.y and (field, plane) in gridDim.z, both limited to 65535
    if (ny > 65535 || nz > 16383)
        return fail(FD_EUNSUPPORTED, "fd_create: ny <= 65535 and nz <= 16383 (CUDA launch-grid limits; got ny %d, nz %d)", ny, nz);
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(FD_ECUDA, "fd_create: no CUDA device (%s); libfd6 has no CPU fallback", cudaGetErrorString(e));
    }
    fd_ctx* c = new (std::nothrow) fd_ctx();
    if (!c) return fail(FD_ENOMEM, "fd_create: host allocation failed");
    c->dtype = dtype;
    c->nx = nx;
    c->ny = ny;
    c->nz = nz;
    c->dx = dx;
    c->nu = nu;
    c->cs = cs;
    c->alloc = g_alloc;
    c->release = g_free;
    c->alloc_user = g_alloc_user;
    // The context starts in the plain layout; resolve_variant switches fp32 grids with an even nz to the paired
    // one.  The buffers are sized for whichever of the two layouts is larger.
    c->paired = false;
    c->esize = dtype == FD_F32 ? 4 : 8;
    c->g = make_geom(nx, ny, nz, c->esize, false);
    c->f_bytes = (size_t)c->g.fs * 4 * c->esize;
    c->div_bytes = (size_t)c->g.fs * c->esize;
    if (pair_ok(c)) {
        const Geom gp = make_geom(nx, ny, nz, 8, true);
        if ((size_t)gp.fs * 4 * 8 > c->f_bytes) c->f_bytes = (size_t)gp.fs * 4 * 8;
        if ((size_t)gp.fs * 8 > c->div_bytes) c->div_bytes = (size_t)gp.fs * 8;
    }
    const size_t w_bytes = (size_t)nx * ny * nz * 4 * (dtype == FD_F32 ? 4 : 8);
    int rc = FD_OK;
    for (int b = 0; b < 2 && rc == FD_OK; ++b) {
        rc = ctx_alloc(c, &c->F[b], c->f_bytes);
        if (rc == FD_OK && cudaMemsetAsync(c->F[b], 0, c->f_bytes, c->stream) != cudaSuccess)
            rc = fail(FD_ECUDA, "fd_create: memset failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    if (rc == FD_OK) rc = ctx_alloc(c, &c->W, w_bytes);
    if (rc == FD_OK && cudaMemsetAsync(c->W, 0, w_bytes, c->stream) != cudaSuccess)
        rc = fail(FD_ECUDA, "fd_create: memset failed: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc == FD_OK) rc = resolve_variant(c);
    if (rc != FD_OK) {
        char keep[sizeof(g_err)];
        strncpy(keep, g_err, sizeof(keep));
        fd_destroy(c);
        strncpy(g_err, keep, sizeof(g_err));
        return rc;
    }
    *out = c;
    return FD_OK;
}

extern "C" int fd_destroy(fd_ctx* c) {
    if (!c) return FD_OK;
    cudaStreamSynchronize(c->stream);
    for (auto& r : c->pending) {
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    for (auto& ev : c->pool) cudaEventDestroy(ev);
    drop_graphs(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    tiled_release(c->tiled);
    ctx_free(c, c->F[0]);
    ctx_free(c, c->F[1]);
    ctx_free(c, c->W);
    ctx_free(c, c->Div);
    ctx_free(c, c->ftab);
    cudaGetLastError();
    delete c;
    return FD_OK;
}

extern "C" int fd_set_path(fd_ctx* c, int path) {
    FD_CHECK_CTX(c);
    if (path != FD_PATH_55 && path != FD_PATH_19) return fail(FD_EINVAL, "fd_set_path: bad path %d", path);
    if (path == FD_PATH_19 && !c->Div) {
        int rc = ctx_alloc(c, &c->Div, c->div_bytes);
        if (rc) return rc;
        FD_CUDA(cudaMemsetAsync(c->Div, 0, c->div_bytes, c->stream));
    }
    c->path = path;
    c->epoch++;
    return FD_OK;
}

extern "C" int fd_set_variant(fd_ctx* c, int variant) {
    FD_CHECK_CTX(c);
    if (variant < FD_VARIANT_AUTO || variant > FD_VARIANT_PAIRED) return fail(FD_EINVAL, "fd_set_variant: bad variant %d", variant);
    int old = c->variant_req;
    c->variant_req = variant;
    int rc = resolve_variant(c);
    if (rc) c->variant_req = old;
    return rc;
}

extern "C" int fd_set_tile_shape(fd_ctx* c, int shape) {
    FD_CHECK_CTX(c);
    if (shape < -1 || shape > 1) return fail(FD_EINVAL, "fd_set_tile_shape: shape must be -1 (automatic), 0 (wide) or 1 (tall)");
    const int old = c->tiled.shape_req;
    c->tiled.shape_req = shape;
    const int rc = resolve_variant(c);  // re-prepares the tensor maps and the work list of the current variant
    if (rc) {
        // the rollback inside resolve_variant still saw the rejected request: put the old one back, then prepare again,
        // so that shape_req and the prepared launches agree (the message of the refusal is kept)
        char keep[sizeof(g_err)];
        memcpy(keep, g_err, sizeof(keep));
        c->tiled.shape_req = old;
        resolve_variant(c);
        memcpy(g_err, keep, sizeof(keep));
    }
    return rc;
}

extern "C" int fd_set_forcing(fd_ctx* c, const double* k, const double* e, double phi, double f0, double dt_ref) {
    FD_CHECK_CTX(c);
    if (!std::isfinite(f0) || f0 < 0) return fail(FD_EINVAL, "fd_set_forcing: f0 must be finite and >= 0");
    c->epoch++;  // whatever happens below, captured steps are stale
    if (f0 == 0) {
        c->force_on = false;
        return FD_OK;
    }
    if (!k || !e) return fail(FD_EINVAL, "fd_set_forcing: NULL vector");
    for (int a = 0; a < 3; ++a)
        if (!std::isfinite(k[a]) || !std::isfinite(e[a])) return fail(FD_EINVAL, "fd_set_forcing: non-finite vector");
    if (!std::isfinite(phi) || !(dt_ref > 0) || !std::isfinite(dt_ref)) return fail(FD_EINVAL, "fd_set_forcing: bad phi or dt_ref");
    const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2], ke = k[0] * e[0] + k[1] * e[1] + k[2] * e[2];
    const double den2 = k2 - ke * ke;
    if (!(den2 > 0)) return fail(FD_EINVAL, "fd_set_forcing: k must not be parallel to e (|k|^2 - (k.e)^2 > 0)");
    // Eq. 25:  N = f0 cs sqrt(|k| cs / dt),  f_k = (k x e) / sqrt(|k|^2 - (k.e)^2)
    const double N = f0 * c->cs * std::sqrt(std::sqrt(k2) * c->cs / dt_ref), den = std::sqrt(den2);
    c->famp[0] = N * (k[1] * e[2] - k[2] * e[1]) / den;
    c->famp[1] = N * (k[2] * e[0] - k[0] * e[2]) / den;
    c->famp[2] = N * (k[0] * e[1] - k[1] * e[0]) / den;
    // separable phase tables, formed in double and rounded once: cx sx (with phi) | cy sy | cz sz
    const int n[3] = {c->nx, c->ny, c->nz};
    const size_t count = 2 * ((size_t)n[0] + n[1] + n[2]), ssize = c->dtype == FD_F64 ? 8 : 4;
    if (!c->ftab) {
        int rc = ctx_alloc(c, &c->ftab, count * ssize);
        if (rc) return rc;
    }
    std::vector<double> tab(count);
    size_t off = 0;
    for (int a = 0; a < 3; ++a) {
        for (int i = 0; i < n[a]; ++i) {
            const double th = k[a] * (i * c->dx) + (a == 0 ? phi : 0.0);
            tab[off + i] = std::cos(th);
            tab[off + n[a] + i] = std::sin(th);
        }
        off += 2 * (size_t)n[a];
    }
    if (c->dtype == FD_F64) {
        FD_CUDA(cudaMemcpyAsync(c->ftab, tab.data(), count * 8, cudaMemcpyHostToDevice, c->stream));
    } else {
        std::vector<float> tf(tab.begin(), tab.end());
        FD_CUDA(cudaMemcpyAsync(c->ftab, tf.data(), count * 4, cudaMemcpyHostToDevice, c->stream));
    }
    FD_CUDA(cudaStreamSynchronize(c->stream));  // the host tables go out of scope
    c->force_on = true;
    return FD_OK;
}

extern "C" int fd_set_stream(fd_ctx* c, void* s) {
    FD_CHECK_CTX(c);
    if ((cudaStream_t)s != c->stream) {
        int rc = drain_profile(c);
        if (rc) return rc;
        FD_CUDA(cudaStreamSynchronize(c->stream));  // keep ordering across a stream change
    }
    c->stream = (cudaStream_t)s;
    return FD_OK;
}

static int check_ptrs(const char* fn, const void* a, const void* b, const void* c_, const void* d, int where) {
    if (!a || !b || !c_ || !d) return fail(FD_EINVAL, "%s: NULL field pointer", fn);
    if (where != FD_HOST && where != FD_DEVICE) return fail(FD_EINVAL, "%s: bad `where` %d", fn, where);
    return FD_OK;
}

extern "C" int fd_load(fd_ctx* c, const void* lnrho, const void* ux, const void* uy, const void* uz, int where) {
    FD_CHECK_CTX(c);
    int rc = check_ptrs("fd_load", lnrho, ux, uy, uz, where);
    if (rc) return rc;
    const void* in[4] = {lnrho, ux, uy, uz};
    return FD_DISPATCH(c, do_load<T>(c, in, where));
}

extern "C" int fd_store(fd_ctx* c, void* lnrho, void* ux, void* uy, void* uz, int where) {
    FD_CHECK_CTX(c);
    int rc = check_ptrs("fd_store", lnrho, ux, uy, uz, where);
    if (rc) return rc;
    void* out[4] = {lnrho, ux, uy, uz};
    return FD_DISPATCH(c, do_store<T>(c, out, where));
}

extern "C" int fd_rhs(fd_ctx* c, void* r0, void* r1, void* r2, void* r3, int where) {
    FD_CHECK_CTX(c);
    int rc = check_ptrs("fd_rhs", r0, r1, r2, r3, where);
    if (rc) return rc;
    void* out[4] = {r0, r1, r2, r3};
    return FD_DISPATCH(c, do_rhs<T>(c, out, where));
}

extern "C" int fd_rk3_step(fd_ctx* c, double dt, int nsteps) {
    FD_CHECK_CTX(c);
    if (nsteps < 0) return fail(FD_EINVAL, "fd_rk3_step: nsteps < 0");
    if (!std::isfinite(dt)) return fail(FD_EINVAL, "fd_rk3_step: dt is not finite");
    return FD_DISPATCH(c, do_rk3<T>(c, dt, nsteps));
}

extern "C" int fd_set_graphs(fd_ctx* c, int on) {
    FD_CHECK_CTX(c);
    c->graphs_on = on != 0;
    if (!c->graphs_on) drop_graphs(c);
    return FD_OK;
}

extern "C" int fd_sync(fd_ctx* c) {
    FD_CHECK_CTX(c);
    FD_CUDA(cudaStreamSynchronize(c->stream));
    FD_CUDA(cudaGetLastError());
    return FD_OK;
}

extern "C" int fd_get_info(const fd_ctx* c, fd_info* o) {
    FD_CHECK_CTX(c);
    if (!o) return fail(FD_EINVAL, "fd_get_info: out is NULL");
    const Geom& g = c->g;
    o->nx = c->nx;
    o->ny = c->ny;
    o->nz = c->nz;
    o->dtype = c->dtype;
    o->path = c->path;
    o->variant = c->variant;
    o->pitch_x = g.px;
    o->pitch_y = g.py;
    o->pitch_z = g.pz;
    o->ghost_x = g.gx;
    o->ghost_y = g.gy;
    o->ghost_z = g.gz;
    o->field_stride = (size_t)g.fs;
    o->device_bytes = c->bytes;
    const bool staged = c->variant == FD_VARIANT_TILED || c->variant == FD_VARIANT_PAIRED;
    o->tile_shape = staged ? c->tiled.shape : -1;
    o->tile_x = o->tile_y = o->work_items = 0;
    if (staged) {
        if (c->dtype == FD_F64)
            shape_dims<double>(c->tiled.shape, &o->tile_x, &o->tile_y);
        else if (c->paired)
            shape_dims<V2>(c->tiled.shape, &o->tile_x, &o->tile_y);
        else
            shape_dims<float>(c->tiled.shape, &o->tile_x, &o->tile_y);
        o->work_items = c->tiled.items;
    }
    o->graph_state = !c->graphs_on ? FD_GRAPH_OFF
                     : c->graph_failed ? FD_GRAPH_FAILED
                     : c->profiling ? FD_GRAPH_WAITING
                     : (c->graph_epoch == c->epoch && (c->graph[0].exec || c->graph[1].exec)) ? FD_GRAPH_CAPTURED
                                                                                              : FD_GRAPH_WAITING;
    snprintf(o->graph_note, sizeof(o->graph_note), "%s", c->graph_note);
    return FD_OK;
}

extern "C" unsigned long long fd_kernel_launches(const fd_ctx* c) { return c ? c->launches : 0ULL; }

extern "C" int fd_set_profiling(fd_ctx* c, int on) {
    FD_CHECK_CTX(c);
    if (!on) {
        int rc = drain_profile(c);
        if (rc) return rc;
    }
    c->profiling = on != 0;
    return FD_OK;
}

extern "C" int fd_get_profile(fd_ctx* c, int id, double* ms, unsigned long long* n) {
    FD_CHECK_CTX(c);
    if (id < 0 || id >= FD_K_COUNT) return fail(FD_EINVAL, "fd_get_profile: bad kernel id %d", id);
    int rc = drain_profile(c);
    if (rc) return rc;
    if (ms) *ms = c->prof_ms[id];
    if (n) *n = c->prof_n[id];
    return FD_OK;
}

extern "C" int fd_reset_profile(fd_ctx* c) {
    FD_CHECK_CTX(c);
    int rc = drain_profile(c);
    if (rc) return rc;
    for (int i = 0; i < FD_K_COUNT; ++i) {
        c->prof_ms[i] = 0;
        c->prof_n[i] = 0;
    }
    return FD_OK;
}

// Host-only: the work list the tiled kernels would run for a grid (no CUDA call, usable without a device).
extern "C" int fd_plan_work_list(int nx, int ny, int nz, int dtype, int sm_count, fd_work_list* o) {
    if (!o) return fail(FD_EINVAL, "fd_plan_work_list: out is NULL");
    if (nx < 8 || ny < 8 || nz < 8 || sm_count < 1) return fail(FD_EINVAL, "fd_plan_work_list: bad grid or SM count");
    if (dtype != FD_F32 && dtype != FD_F64) return fail(FD_EINVAL, "fd_plan_work_list: bad dtype %d", dtype);
    const bool paired = dtype == FD_F32 && nz % 2 == 0 && nz / 2 >= 4;  // the layout the staged kernels would use
    int tx, ty;  // the tile shape tiled_prepare would pick for this grid
    if (dtype == FD_F64)
        shape_dims<double>(pick_shape<double>(nx, ny, sm_count, -1), &tx, &ty);
    else if (paired)
        shape_dims<V2>(pick_shape<V2>(nx, ny, sm_count, -1), &tx, &ty);
    else
        shape_dims<float>(0, &tx, &ty);
    const int planes = paired ? nz / 2 : nz;
    int items = 0;
    const Sched sc = plan_work_list((nx + tx - 1) / tx, (ny + ty - 1) / ty, planes, sm_count, &items);
    o->tile_x = tx;
    o->tile_y = ty;
    o->tiles_x = sc.ntx;
    o->tiles_y = (ny + ty - 1) / ty;
    o->planes = planes;
    o->full_tiles = sc.n_full;
    o->chunks = sc.k;
    o->chunk_planes = sc.zc;
    o->split_plane = sc.za;
    o->items = items;
    return FD_OK;
}

template <class T>
static int do_poison(fd_ctx* c, bool ghosts) {
    const T nan = T(typename Scalar<T>::type(NAN));
    if (ghosts) {
        c->loaded = true;  // the zero state is gone: a layout switch must carry the fields across
        long long n = (long long)c->g.px * c->g.py * c->g.pz * 4;
        for (int b = 0; b < 2; ++b) {
            c->launches++;
            k_poison_ghosts<T><<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>((T*)c->F[b], c->g, nan);
        }
    } else {
        long long n = c->g.n * 4;
        c->launches++;
        k_fill<T><<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>((T*)c->W, n, nan);
    }
    FD_CUDA(cudaGetLastError());
    return FD_OK;
}

// ---- include/fd6_testing.h: test hooks, not part of the product ABI ----
extern "C" int fd_debug_poison_w(fd_ctx* c) {
    FD_CHECK_CTX(c);
    return FD_DISPATCH(c, do_poison<T>(c, false));
}

extern "C" int fd_debug_set_tile_overlap(fd_ctx* c, int overlap) {
    FD_CHECK_CTX(c);
    if (overlap < 0) return fail(FD_EINVAL, "fd_debug_set_tile_overlap: overlap < 0");
    const int old = c->tiled.overlap;
    c->tiled.overlap = overlap;
    int rc = resolve_variant(c);
    // under AUTO a refused overlap would silently fall back to the direct kernels: report it instead
    if (rc == FD_OK && overlap > 0 && c->variant != FD_VARIANT_TILED && c->variant != FD_VARIANT_PAIRED)
        rc = fail(FD_EUNSUPPORTED, "fd_debug_set_tile_overlap: the staged kernels do not run this grid with overlap %d (%s)", overlap,
                  tiled_error_of(c->tiled));
    if (rc) {
        char keep[sizeof(g_err)];
        memcpy(keep, g_err, sizeof(keep));
        c->tiled.overlap = old;
        resolve_variant(c);
        memcpy(g_err, keep, sizeof(keep));
    }
    return rc;
}

extern "C" int fd_debug_poison_ghosts(fd_ctx* c) {
    FD_CHECK_CTX(c);
    return FD_DISPATCH(c, do_poison<T>(c, true));
}

// ------------------------------------------------------------------------------------------------
// fd_rhs_static (include/fd6.h): fd_rhs on FD_PATH_55 for callers that cannot allocate device memory.
//
// The stencil kernel needs one thing beyond its inputs and outputs: the ghost-padded copy of the four fields it reads
// (DESIGN.md "HBM layout").  A context gets that from cudaMalloc or the allocator hook; here it is a fixed array in the
// library image, so the call allocates nothing.  Every GPU that loads libfd6.so holds these bytes until the process ends.
//
// `g_static_scratch` below is a device symbol.  In HOST code that name is only a handle the CUDA runtime uses to find the
// symbol — it is not a device address and must never be handed to a kernel.  The address that kernels can use comes
// from cudaGetSymbolAddress, asked for once per device with that device current (static_scratch_of_current_device),
// and it is that pointer which the launches below receive.  All of this has to live in this one .cu file: the array has
// internal linkage, another translation unit would be looking at a different symbol.
// ------------------------------------------------------------------------------------------------
#include <mutex>

static __device__ __align__(256) unsigned char g_static_scratch[FD_RHS_STATIC_MAX_BYTES];

static const int kStaticMaxDevices = 64;
static std::mutex g_static_mutex;
static void* g_static_addr[kStaticMaxDevices] = {};  // device address of g_static_scratch on device d; NULL: not asked yet

static int static_scratch_of_current_device(void** out) {
    int dev = -1;
    FD_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(FD_EUNSUPPORTED, "fd_rhs_static: device ordinal %d is outside 0..%d", dev, kStaticMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        void* p = nullptr;
        FD_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return fail(FD_ECUDA, "fd_rhs_static: cudaGetSymbolAddress gave a NULL address on device %d", dev);
        g_static_addr[dev] = p;
    }
    *out = g_static_addr[dev];
    return FD_OK;
}

// k_direct_main<T, true> with the update of Eq. 10 taken out: the right-hand side of one cell goes straight to the
// caller's four dense result arrays (a context's fd_rhs writes it to w first and copies).  Fin is the padded scratch.
// block (64,4,1), grid (ceil(nx/64), ceil(ny/4), nz), T = float or double (plain layout).
template <class T>
__global__ void __launch_bounds__(256) k_rhs55_static(const T* __restrict__ Fin, T* __restrict__ r0, T* __restrict__ r1,
                                                      T* __restrict__ r2, T* __restrict__ r3, Geom g, Coef<T> c) {
    const int i = blockIdx.x * 64 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k = blockIdx.z;
    if (i >= g.nx || j >= g.ny) return;
    const long long sx = 1, sy = g.px, sz = (long long)g.px * g.py;
    const long long p = (i + g.gx) + sy * (j + g.gy) + sz * (k + g.gz);
    const T* l = Fin + p;
    const T* uu[3] = {Fin + g.fs + p, Fin + 2 * g.fs + p, Fin + 3 * g.fs + p};
    const long long st[3] = {sx, sy, sz};
    T u[3], gl[3], G[3][3], L[3], Q[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) gl[a] = d1(l, st[a], c);
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        u[q] = uu[q][0];
        T dd[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            G[q][a] = d1(uu[q], st[a], c);
            dd[a] = d2(uu[q], st[a], c);
        }
        L[q] = dd[0] + dd[1] + dd[2];
        Q[q] = dd[q];
    }
    Q[0] += dmix(uu[1], sx, sy, c) + dmix(uu[2], sx, sz, c);
    Q[1] += dmix(uu[0], sy, sx, c) + dmix(uu[2], sy, sz, c);
    Q[2] += dmix(uu[0], sz, sx, c) + dmix(uu[1], sz, sy, c);
    T Rv[4];
    assemble<T, true>(u, gl, G, L, Q, c, Rv);
    const long long pw = i + (long long)g.nx * (j + (long long)g.ny * k);
    r0[pw] = Rv[0];
    r1[pw] = Rv[1];
    r2[pw] = Rv[2];
    r3[pw] = Rv[3];
}

template <class T>
static int do_rhs_static(fd_ctx* rec, void* scratch, const void* const in[4], void* const out[4]) {
    // copy-in + periodic halo fill into the scratch: the helpers a context uses, pointed at the built-in array
    rec->F[0] = scratch;
    rec->cur = 0;
    const T* src[4] = {(const T*)in[0], (const T*)in[1], (const T*)in[2], (const T*)in[3]};
    int rc = do_pack<T>(rec, src);
    if (rc) return rc;
    const Geom& g = rec->g;
    dim3 block(64, 4, 1), grid((g.nx + 63) / 64, (g.ny + 3) / 4, g.nz);
    k_rhs55_static<T><<<grid, block, 0, rec->stream>>>((const T*)scratch, (T*)out[0], (T*)out[1], (T*)out[2], (T*)out[3], g,
                                                       make_coef<T>(rec));
    FD_CUDA(cudaGetLastError());
    return FD_OK;
}

extern "C" int fd_rhs_static(int nx, int ny, int nz, double dx, double nu, double cs, int dtype, const void* lnrho, const void* ux,
                             const void* uy, const void* uz, void* d_lnrho, void* d_ux, void* d_uy, void* d_uz, void* cuda_stream) {
    if (!lnrho || !ux || !uy || !uz || !d_lnrho || !d_ux || !d_uy || !d_uz) return fail(FD_EINVAL, "fd_rhs_static: NULL field pointer");
    if (nx < 8 || ny < 8 || nz < 8) return fail(FD_EINVAL, "fd_rhs_static: every axis needs n >= 8 (got %d,%d,%d)", nx, ny, nz);
    if (!(dx > 0) || !std::isfinite(dx)) return fail(FD_EINVAL, "fd_rhs_static: dx must be finite and > 0");
    if (!(nu >= 0) || !std::isfinite(nu)) return fail(FD_EINVAL, "fd_rhs_static: nu must be finite and >= 0");
    if (!(cs >= 0) || !std::isfinite(cs)) return fail(FD_EINVAL, "fd_rhs_static: cs must be finite and >= 0");
    if (dtype != FD_F32 && dtype != FD_F64) return fail(FD_EINVAL, "fd_rhs_static: bad dtype %d", dtype);
    if (nx % 4 != 0) return fail(FD_EUNSUPPORTED, "fd_rhs_static: nx must be a multiple of 4 (got %d)", nx);
    const size_t esize = dtype == FD_F32 ? 4 : 8;
    // 64-bit size check before make_geom: three axes of >= 8 values each bound every axis by the array size
    const unsigned long long rough = (unsigned long long)(nx + 8) * (unsigned long long)(ny + 6) * (unsigned long long)(nz + 6) * 4ULL * esize;
    if (rough > FD_RHS_STATIC_MAX_BYTES)
        return fail(FD_EUNSUPPORTED,
                    "fd_rhs_static: the ghost-padded state of a %dx%dx%d %s grid needs at least %llu bytes, the built-in scratch "
                    "array holds %u (e.g. 64^3 fp32, 48^3 fp64); use fd_create + fd_rhs for larger grids",
                    nx, ny, nz, dtype == FD_F32 ? "fp32" : "fp64", rough, (unsigned)FD_RHS_STATIC_MAX_BYTES);
    // A context record on the host stack: only the argument block of the launch helpers (geometry, constants, stream).
    // It owns no device memory and nothing is allocated for it.
    fd_ctx rec;
    rec.nx = nx;
    rec.ny = ny;
    rec.nz = nz;
    rec.dx = dx;
    rec.nu = nu;
    rec.cs = cs;
    rec.dtype = dtype;
    rec.esize = esize;
    rec.paired = false;
    rec.stream = (cudaStream_t)cuda_stream;
    rec.g = make_geom(nx, ny, nz, esize, false);
    const unsigned long long need = (unsigned long long)rec.g.fs * 4ULL * esize;
    if (need > FD_RHS_STATIC_MAX_BYTES)
        return fail(FD_EUNSUPPORTED,
                    "fd_rhs_static: the ghost-padded state of a %dx%dx%d %s grid needs %llu bytes, the built-in scratch array "
                    "holds %u (e.g. 64^3 fp32, 48^3 fp64); use fd_create + fd_rhs for larger grids",
                    nx, ny, nz, dtype == FD_F32 ? "fp32" : "fp64", need, (unsigned)FD_RHS_STATIC_MAX_BYTES);
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(FD_ECUDA, "fd_rhs_static: no CUDA device (%s); libfd6 has no CPU fallback", cudaGetErrorString(e));
    }
    void* scratch = nullptr;
    int rc = static_scratch_of_current_device(&scratch);
    if (rc) return rc;
    const void* in[4] = {lnrho, ux, uy, uz};
    void* out[4] = {d_lnrho, d_ux, d_uy, d_uz};
    return dtype == FD_F64 ? do_rhs_static<double>(&rec, scratch, in, out) : do_rhs_static<float>(&rec, scratch, in, out);
}
