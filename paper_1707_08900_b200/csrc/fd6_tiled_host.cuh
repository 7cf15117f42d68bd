// fd6_tiled_host.cuh — host side of FD_VARIANT_TILED / FD_VARIANT_PAIRED: launch parameters, tile shapes, tensor maps,
// the work-list planner and the launch wrappers.  The kernels themselves are in fd6_kernels_tiled.cuh and are compiled
// in translation units of their own (fd6_tiled_inst.cu); fd6.cu sees only this file.
#pragma once
#include <cuda.h>

#include <algorithm>
#include <cstdio>
#include <functional>
#include <queue>
#include <type_traits>
#include <vector>

#include "fd6_common.cuh"

namespace fd6 {

// Coefficients with the physics constants, dt and the RK substep folded in (formed in double on the host,
// rounded once to the scalar type; V2 holds the same number in both halves).
template <class T>
struct KC {
    T ar[3];   // Eq. 6:  a_m / (60 dx)                     first derivatives of ln rho
    T au[3];   // dt a_m / (60 dx)                          first derivatives of u (carry dt)
    T lo[4];   // dt nu b_m / (180 dx^2), m = 0..3          second derivative along an axis other than i
    T lq[4];   // PATH55: dt (4 nu / 3) b_m (d_ii u_i enters lap u_i and d_i div u);  PATH19: same as lo
    T cxy[3];  // centre coefficient of the in-plane second derivatives of u_x, u_y, u_z
    T mq[3];   // dt (nu / 3) c_m / (720 dx^2)              Eq. 8
    T nu, nu2, nu23, cs2dt, dt;
    T alpha, beta;
    T fa[3];   // FORCE: dt N f_k (Eq. 24-25), the amplitude of the forcing term in dt*rhs_i
    int read_w, write_f, write_w;
};

// Work list of one launch (1-D grid, one CTA per item, launched in this order).  The first n_full tiles (a
// multiple of the SM count) are marched through all of z by one CTA each; the remaining tiles, which would
// fill only part of a last wave, are cut into k z-chunks of zc planes so that their items fill whole waves
// again (each chunk re-stages 6 warm-up planes, which is why only the remainder is cut).
struct Sched {
    int ntx;     // tiles along x; tile index = bx + ntx * by
    int n_full;  // tiles with a single item
    int k, zc;   // chunks per remaining tile, planes per chunk
    int nty;     // tiles along y
    int za;      // 0, or the "split" list for grids with about as many tiles as SMs: EVERY tile is cut at stored plane za;
                 // item b < tiles is tile b over planes [0, za), item tiles + b is tile b over [za, nz).  The long items
                 // are dispatched first, the short ones fill the SMs that would otherwise idle (n_full, k, zc unused).
    int ov;      // 0, or (include/fd6_testing.h, fd_debug_set_tile_overlap) the number of values by which neighbouring tiles
                 // overlap in x and y: every tile is still computed in full, a value is stored by the tile that holds it
                 // furthest from its edge.  Emulates the redundant halo-ring evaluation of temporal blocking (DESIGN 7).
};

// The tensor maps of one launch (each 128 bytes, passed by value as a __grid_constant__ parameter).
struct Maps {
    CUtensorMap f_in;  // padded fields, read copy: box (TX+8, TY+6, 1, 4)
    CUtensorMap w_ld;  // dense w:                  box (TX, TY, 1, 4)
};

// Arithmetic type of the kernels of storage type T.  fp64 and the paired layout compute on their stored value; PLAIN
// fp32 computes on V2 = the two cells (i, j, k), (i, j+1, k) of one thread ("y pairs"): the pair shares the eight
// values of its x column and its own-row x differences, every shared-memory access is a conflict-free 4-byte load
// with consecutive lanes on consecutive words, and all arithmetic except the odd y offsets is packed (FFMA2).
template <class T> struct Arith { typedef T type; static constexpr int CY = 1; };
template <> struct Arith<float> { typedef V2 type; static constexpr int CY = 2; };

// Tile shapes (registers and tensor memory per thread bound the CTA size).  TX x TY threads; a
// thread owns RY columns of values, a value of the arithmetic type holds CY vertically adjacent cells, so the tile is
// TX x TH cells with TH = TY * RY * CY.  Two shapes, picked per grid by pick_shape():
//   S = 0 "wide"  12 warps, one value per thread (32 x 12 values): 76 shared-memory loads per value
//   S = 1 "tall"   8 warps, two vertically adjacent values per thread (32 x 16 values): the thread's x column is loaded
//                 once for both (64 loads per value, bit-identical results); the state of two columns fills the tensor
//                 memory of 2 warps per lane quadrant and ~230 registers.  Faster once a grid has enough tiles to fill
//                 the SMs (C4: fused kernel -1.4 %, sustained +1.5 %, 20 % fewer shared-memory wavefronts); slower on
//                 small grids, where fewer and larger tiles mean fewer work items (C2: +30 %).
// Plain fp32 (y pairs) has the wide shape only.
template <class T, int S>
struct TileShape;
template <>
struct TileShape<float, 0> {
    static constexpr int TX = 32, TY = 12, NS = 4, RY = 1, TH = TY * RY * Arith<float>::CY;
};
template <>
struct TileShape<double, 0> {
    static constexpr int TX = 32, TY = 12, NS = 4, RY = 1, TH = TY * RY;
};
template <>
struct TileShape<double, 1> {
    static constexpr int TX = 32, TY = 8, NS = 4, RY = 2, TH = TY * RY;
};
template <>
struct TileShape<V2, 0> {
    static constexpr int TX = 32, TY = 12, NS = 4, RY = 1, TH = TY * RY;
};
template <>
struct TileShape<V2, 1> {
    static constexpr int TX = 32, TY = 8, NS = 4, RY = 2, TH = TY * RY;
};
template <class T> struct Shapes { static constexpr int count = 2; };
template <> struct Shapes<float> { static constexpr int count = 1; };

// Shape for a grid: the tall one when its tiles give at least two thirds of an SM wave (measured: C3 with 128 tall
// tiles on 148 SMs gains, C2 with 32 loses).  tile_h receives the tile height in stored values.
template <class T>
inline int pick_shape(int nx, int ny, int sm_count, int request) {
    if (Shapes<T>::count < 2) return 0;
    if (request >= 0) return request > 0 ? 1 : 0;
    const long long tall = (long long)((nx + 31) / 32) * ((ny + 15) / 16);
    return 3 * tall >= 2LL * sm_count ? 1 : 0;
}
template <class T>
inline void shape_dims(int s, int* tx, int* th) {
    if constexpr (Shapes<T>::count > 1) {
        if (s == 1) {
            *tx = TileShape<T, 1>::TX;
            *th = TileShape<T, 1>::TH;
            return;
        }
    }
    *tx = TileShape<T, 0>::TX;
    *th = TileShape<T, 0>::TH;
}

// ---- host side -------------------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TiledState {
    bool ready = false;
    Maps maps[2];      // maps[cur]: read copy F[cur]
    bool force_fits = true;  // the forcing's z table fits in shared memory beside the rings
    Sched sched{};     // work list
    int items = 0;     // grid size
    int shape = 0;     // tile shape of the prepared launches (TileShape<T, shape>)
    int shape_req = -1;  // -1: pick_shape decides; 0 / 1: forced (fd_set_tile_shape)
    int overlap = 0;     // tile overlap of the temporal-blocking emulation (include/fd6_testing.h); 0 in every product launch
    int sm_count = 0;
    char err[256] = "";
};

inline bool tiled_supported(const Geom& g) {  // the kernels address F_out and w with 32-bit element offsets
    return g.nx >= 4 && g.ny >= 4 && g.nz >= 4 && 4 * g.fs < (1LL << 32) && 4 * g.n < (1LL << 32);
}

inline PFN_encodeTiled tiled_encode_fn() {
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (PFN_encodeTiled)p;
        else
            cudaGetLastError();
    }
    return fn;
}

// 4-D tensor map over `nf` arrays of (ex, ey, ez) values with pitches (px, py) and array stride fs (all in
// values); the x extent and the box are given in values and converted to scalars here.
template <class T>
inline int tiled_make_map(TiledState& ts, CUtensorMap* tm, void* base, long long ex, long long ey, long long ez, int nf, long long px,
                          long long py, long long fs, int box_x, int box_y, int box_f) {
    typedef typename Scalar<T>::type S;
    constexpr int L = Scalar<T>::lanes;
    PFN_encodeTiled enc = tiled_encode_fn();
    if (!enc) {
        snprintf(ts.err, sizeof(ts.err), "cuTensorMapEncodeTiled is not available from this driver");
        return 3;
    }
    const cuuint64_t dims[4] = {(cuuint64_t)ex * L, (cuuint64_t)ey, (cuuint64_t)ez, (cuuint64_t)nf};
    const cuuint64_t strides[3] = {(cuuint64_t)px * sizeof(T), (cuuint64_t)px * py * sizeof(T), (cuuint64_t)fs * sizeof(T)};
    const cuuint32_t box[4] = {(cuuint32_t)(box_x * L), (cuuint32_t)box_y, 1, (cuuint32_t)box_f};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(tm, sizeof(S) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box,
                     estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(ts.err, sizeof(ts.err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return 3;
    }
    return 0;
}

// Work list (see Sched; pure host arithmetic, also reachable through fd_plan_work_list for the CPU tests): one CTA
// per SM is resident, so whole waves of S tiles run as full columns and the remaining tiles are cut into the
// number of z-chunks that minimises (waves x planes staged per item).
// Time (in planes) at which a launch ends when its items, `count[i]` items of `cost[i]` planes each in this order, are
// dispatched in index order, each to the SM that becomes free first (one resident CTA per SM): what the hardware does.
inline long long list_makespan(const int* count, const int* cost, int classes, int S) {
    std::priority_queue<long long, std::vector<long long>, std::greater<long long>> free_at;
    for (int s = 0; s < S; ++s) free_at.push(0);
    long long end = 0;
    for (int c = 0; c < classes; ++c)
        for (int i = 0; i < count[c]; ++i) {
            const long long t = free_at.top() + cost[c];
            free_at.pop();
            free_at.push(t);
            end = std::max(end, t);
        }
    return end;
}

inline Sched plan_work_list(int ntx, int nty, int nz, int S, int* items) {
    const int tiles = ntx * nty;
    const int n_full = (tiles / S) * S, rem = tiles - n_full;
    const int warm = 2 * R + 4;  // planes an item stages before its first output (+ fill latency)
    int best_k = 1;
    double best_cost = 1e300;
    for (int k = 1; rem > 0 && k <= (nz + 1) / 2 && k <= 64; ++k) {  // chunks of >= 2 planes
        const int zc = (nz + k - 1) / k;
        const int real = (nz + zc - 1) / zc;
        const long long waves = ((long long)rem * real + S - 1) / S;
        const double cost = (double)waves * (zc + warm);  // time ~ waves x planes staged per item
        if (cost < best_cost) {
            best_cost = cost;
            best_k = k;
        }
    }
    Sched sc;
    sc.ntx = ntx;
    sc.nty = nty;
    sc.ov = 0;
    sc.za = 0;
    sc.n_full = n_full;
    sc.zc = (nz + best_k - 1) / best_k;
    sc.k = (nz + sc.zc - 1) / sc.zc;
    *items = n_full + rem * sc.k;
    // Grids with about as many tiles as SMs (C3: 128 tall tiles on 148 SMs) leave SMs idle for a whole column, and cutting
    // only a remainder cannot help while any item is a full column.  Cut EVERY tile at one plane za instead: the long
    // parts go out first, the short parts are packed onto the SMs left over (C3: 128 x 232 planes + 128 x 24 planes,
    // the launch ends after 242 plane-times instead of 266 by this model).  Taken when the model beats the two-tier list by
    // more than 3 %.  Measured at C3 in one session (profiles/r03_alt_split_C3_*.json.txt): first repetition 13092 ->
    // 13626 Mcell/s (+4 %, less than the model's 9 %: a short item costs more than its planes + warm-up), median of five
    // under the rising power cap 12203 / 12585 -> 12648; a cut 8 planes lower (224) is 4 % SLOWER than no split, so the
    // plane comes from the model's minimum, never from a round number.
    if (tiles < 4 * S && nz >= 16) {
        const int cnt2[2] = {n_full, rem * sc.k}, cost2[2] = {nz + warm, sc.zc + warm};
        const long long cur = list_makespan(cnt2, cost2, 2, S);
        long long best = cur;
        int best_za = 0;
        const int step = std::max(1, nz / 256);
        for (int za = (nz + 1) / 2; za <= nz - 2; za += step) {
            const int cnt[2] = {tiles, tiles}, cost[2] = {za + warm, nz - za + warm};
            const long long m = list_makespan(cnt, cost, 2, S);
            if (m < best) {
                best = m;
                best_za = za;
            }
        }
        if (best_za > 0 && 100 * best < 97 * cur) {
            sc.za = best_za;
            sc.n_full = 0;
            sc.k = 2;
            sc.zc = best_za;
            *items = 2 * tiles;
        }
    }
    return sc;
}

// The kernel instantiations of one (value type, FORCE, tile shape) live in a translation unit of their own
// (fd6_tiled_inst.cu; compiled in parallel by build.py): this is the whole interface between them and fd6.cu.
template <class T, bool FORCE, int S>
struct TiledTU {
    static size_t smem_bytes(int planes);                 // dynamic shared memory of a launch over `planes` stored planes
    static cudaError_t set_smem(size_t bytes);            // opt every instantiation of this unit in to `bytes`
    static int max_ctas_per_sm(size_t bytes);             // occupancy of the fused kernel (the design assumes 1)
    // launches the instantiation for (path55, mode); false if there is none
    static bool launch(bool path55, int mode, int items, size_t smem, cudaStream_t stream, const Maps& m, const Geom& g, const KC<typename Arith<T>::type>& c,
                       const Sched& sc, T* Fout, T* W, T* Div, const ForceTab<T>& ft);
};

template <class T, int S>
inline int tiled_prepare_shape(TiledState& ts, const Geom& g, void* F0, void* F1, void* W) {
    constexpr int TX = TileShape<T, S>::TX, TH = TileShape<T, S>::TH;
    void* F[2] = {F0, F1};
    int rc = 0;
    for (int cur = 0; cur < 2 && rc == 0; ++cur) {
        Maps& m = ts.maps[cur];
        rc = tiled_make_map<T>(ts, &m.f_in, F[cur], g.px, g.py, g.pz, 4, g.px, g.py, g.fs, TX + 8, TH + 2 * R, 4);
        if (rc == 0) rc = tiled_make_map<T>(ts, &m.w_ld, W, g.nx, g.ny, g.nz, 4, g.nx, g.ny, g.n, TX, TH, 4);
    }
    if (rc) return rc;
    const size_t smem = TiledTU<T, false, S>::smem_bytes(0);
    const size_t smem_f = TiledTU<T, true, S>::smem_bytes(g.nz);  // + the forcing's z table
    ts.force_fits = smem_f <= 227 * 1024;
    cudaError_t e = TiledTU<T, false, S>::set_smem(smem);
    if (e == cudaSuccess && ts.force_fits) e = TiledTU<T, true, S>::set_smem(smem_f);
    if (e != cudaSuccess) {
        snprintf(ts.err, sizeof(ts.err), "cudaFuncSetAttribute(smem): %s", cudaGetErrorString(e));
        cudaGetLastError();
        return 3;
    }
    // the kernels take all of tensor memory and the work list counts waves of one CTA per SM
    if (TiledTU<T, false, S>::max_ctas_per_sm(smem) != 1) {
        snprintf(ts.err, sizeof(ts.err), "the tiled kernels are designed for exactly one resident CTA per SM");
        return 3;
    }
    const int ov = ts.overlap;
    if (ov > 0 && (Arith<T>::CY != 1 || ov % 2 != 0 || ov >= TX || ov >= TH)) {
        snprintf(ts.err, sizeof(ts.err), "tile overlap: even, smaller than the tile, 8-byte value types only");
        return 3;
    }
    // tiles step by (TX - ov, TH - ov); the last tile of a row / column may hang over the grid (clipped as usual)
    const int ntx = ov ? (std::max(g.nx - ov, 1) + (TX - ov) - 1) / (TX - ov) : (g.nx + TX - 1) / TX;
    const int nty = ov ? (std::max(g.ny - ov, 1) + (TH - ov) - 1) / (TH - ov) : (g.ny + TH - 1) / TH;
    ts.sched = plan_work_list(ntx, nty, g.nz, ts.sm_count, &ts.items);
    ts.sched.ov = ov;
    ts.shape = S;
    ts.ready = true;
    return 0;
}

// F[0], F[1]: the two padded copies; W: the dense w arrays.
template <class T>
inline int tiled_prepare(TiledState& ts, const Geom& g, void* F0, void* F1, void* W) {
    ts.ready = false;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&ts.sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (ts.sm_count <= 0) ts.sm_count = 148;
    if constexpr (Shapes<T>::count > 1) {
        if (pick_shape<T>(g.nx, g.ny, ts.sm_count, ts.shape_req) == 1) return tiled_prepare_shape<T, 1>(ts, g, F0, F1, W);
    }
    return tiled_prepare_shape<T, 0>(ts, g, F0, F1, W);
}

inline const char* tiled_error_of(const TiledState& ts) { return ts.err; }
inline void tiled_release(TiledState& ts) { ts.ready = false; }

template <class T>
inline KC<T> make_kc(double dx, double nu, double cs, bool path55, double dt, double alpha, double beta, int read_w, int write_f,
                     int write_w, const double famp[3]) {
    typedef typename Scalar<T>::type S;
    const double dx2 = dx * dx;
    const double b[4] = {-490.0 / (180.0 * dx2), 270.0 / (180.0 * dx2), -27.0 / (180.0 * dx2), 2.0 / (180.0 * dx2)};
    const double cm[3] = {270.0 / (720.0 * dx2), -27.0 / (720.0 * dx2), 2.0 / (720.0 * dx2)};
    const double a[3] = {45.0 / (60.0 * dx), -9.0 / (60.0 * dx), 1.0 / (60.0 * dx)};
    const double own = path55 ? 4.0 * nu / 3.0 : nu;
    KC<T> k;
    for (int m = 0; m < 3; ++m) {
        k.ar[m] = T(S(a[m]));
        k.au[m] = T(S(dt * a[m]));
        k.mq[m] = T(S(dt * nu / 3.0 * cm[m]));
    }
    for (int m = 0; m < 4; ++m) {
        k.lo[m] = T(S(dt * nu * b[m]));
        k.lq[m] = T(S(dt * own * b[m]));
    }
    k.cxy[0] = T(S(dt * (own + nu) * b[0]));
    k.cxy[1] = T(S(dt * (own + nu) * b[0]));
    k.cxy[2] = T(S(dt * 2.0 * nu * b[0]));
    k.nu = T(S(nu));
    k.nu2 = T(S(2.0 * nu));
    k.nu23 = T(S(2.0 * nu / 3.0));
    k.cs2dt = T(S(cs * cs * dt));
    k.dt = T(S(dt));
    k.alpha = T(S(alpha));
    k.beta = T(S(beta));
    for (int i = 0; i < 3; ++i) k.fa[i] = T(S(dt * famp[i]));
    k.read_w = read_w;
    k.write_f = write_f;
    k.write_w = write_w;
    return k;
}

// Launch of the main kernel of one substep (fused 55-point kernel, or pass 1 of the 19-point path, which
// leaves dt * div u in Div): reads copy `cur`, writes copy 1 - cur and w.
template <class T>
inline int tiled_launch_main(TiledState& ts, int path55, int cur, T* Fout, T* W, T* Div, const Geom& g, const KC<typename Arith<T>::type>& c,
                             const ForceTab<T>& ft, cudaStream_t stream) {
    const bool force = ft.tab != nullptr;
    if (force && !ts.force_fits) return 4;
    const int mode = (c.read_w ? 1 : 0) | (c.write_w ? 2 : 0) | (c.write_f ? 4 : 0);
    bool launched = false;
    auto go = [&](auto shape_tag) {
        constexpr int S = decltype(shape_tag)::value;
        launched = force ? TiledTU<T, true, S>::launch(path55 != 0, mode, ts.items, TiledTU<T, true, S>::smem_bytes(g.nz), stream, ts.maps[cur], g,
                                                       c, ts.sched, Fout, W, Div, ft)
                         : TiledTU<T, false, S>::launch(path55 != 0, mode, ts.items, TiledTU<T, false, S>::smem_bytes(0), stream, ts.maps[cur], g,
                                                        c, ts.sched, Fout, W, Div, ft);
    };
    if constexpr (Shapes<T>::count > 1) {
        if (ts.shape == 1)
            go(std::integral_constant<int, 1>());
        else
            go(std::integral_constant<int, 0>());
    } else {
        go(std::integral_constant<int, 0>());
    }
    if (!launched) {
        snprintf(ts.err, sizeof(ts.err), "no tiled kernel for update mode %d", mode);
        return 3;
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) snprintf(ts.err, sizeof(ts.err), "%s", cudaGetErrorString(e));
    return e == cudaSuccess ? 0 : 3;
}

}  // namespace fd6
