// fd6_kernels_tiled.cuh — FD_VARIANT_TILED: the fast derivative/update kernel.
//
// One CTA owns a TX x TY column of cells and marches along z through a chunk of planes.  A plane of all four
// fields plus its radius-3 halo is staged into shared memory by ONE 4-D TMA box copy (cp.async.bulk.tensor,
// mbarrier complete_tx), four stages deep, so a plane is read from L2/HBM once per CTA.  Each thread owns one
// cell column and keeps everything that couples planes in registers:
//   win[f][8]   sliding window of its own cell's values along z           -> D1z, D2z             (Eq. 6, 7)
//   dl[q][4]    the in-plane first derivatives of the last planes, delayed until the plane is the centre
//   lin[i][8]   accumulator ring of the part of the right-hand side that is LINEAR in second derivatives,
//               nu (lap u_i + 1/3 d_i div u): in-plane D2x, D2y, Dxy are added when the plane is staged, and the
//               mixed derivatives that involve z (Eq. 8) are formed from the in-plane differences
//               f(x+m) - f(x-m) that D1x / D1y need anyway:  Dxz f(z) = sum_m c_m [dx_m f(z+m) - dx_m f(z-m)],
//               so plane t scatters +-c_m dx_m into the ring slots of outputs t-m and t+m (no extra loads).
// Output plane z = t-3 is assembled (Eq. 1-3) and updated (Eq. 10) when plane t = z+3 has been consumed.
// The accumulation order of every output depends only on relative plane index, never on the position in a
// tile or chunk, so periodic-shift equivariance stays bitwise.
// PATH55 = false is pass 1 of the 19-point path (no mixed derivatives, div u written, Eq. 14-16).
#pragma once
#include <cuda.h>

#include "fd6_common.cuh"

namespace fd6 {

// Coefficients with the physics constants folded in (formed in double on the host, rounded once to T).
template <class T>
struct TCoef {
    T a[3];    // Eq. 6:  a_m / (60 dx)
    T lo[4];   // nu * b_m / (180 dx^2), m = 0..3          second derivative along an axis other than i
    T lq[4];   // PATH55: (4 nu / 3) * b_m (d_ii u_i enters lap u_i and d_i div u);  PATH19: same as lo
    T cxy[3];  // centre coefficient of the in-plane part for u_x, u_y, u_z
    T mq[3];   // (nu / 3) * c_m / (720 dx^2)              Eq. 8
    T nu, cs2, nu23;
};

// ---- mbarrier / TMA primitives (PTX ISA: mbarrier, cp.async.bulk.tensor) --------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(b)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

template <class T, bool PATH55, int TX, int TY>
struct Tiled {
    static constexpr int PXS = TX + 8;  // staged row: 4 cells left of the tile (3 used; keeps rows 16-byte aligned) + TX + 4
    static constexpr int PYS = TY + 2 * R;
    static constexpr int FIELD = PXS * PYS;
    static constexpr int STAGE = 4 * FIELD;  // elements per stage: four fields of one plane
    static constexpr int S = 4;              // stages (divides the unroll factor 8: stage offsets are immediates)
    static constexpr int THREADS = TX * TY;
    static constexpr size_t SMEM = (size_t)S * STAGE * sizeof(T) + S * sizeof(uint64_t);

    struct State {
        T win[4][8];
        T lin[3][8];
        T dl[8][4];
    };

    template <int PH>
    static __device__ __forceinline__ void step(State& st, const T* __restrict__ sp0, const TCoef<T>& c, const Sub<T>& s, int p,
                                                bool store_ok, const T* __restrict__ wp, T* __restrict__ wq, T* __restrict__ fo,
                                                T* __restrict__ dv, long long fs, long long n) {
        constexpr int n8 = PH & 7, n4 = PH & 3;
        const T* sp = sp0 + n4 * STAGE;
        const bool out = p >= 2 * R;  // planes 0..5 of a chunk only warm the window and the rings up
        T wold[4];
        if (out && s.read_w) {
#pragma unroll
            for (int f = 0; f < 4; ++f) wold[f] = store_ok ? wp[f * n] : T(0);
        }
        T inpl[3];                      // in-plane part of nu (lap u_i + 1/3 d_i div u) at the staged plane
        T dgx = T(0), dgy = T(0);       // nu/3 d_xy u_y -> component x, nu/3 d_xy u_x -> component y
        T ex[3], ey[3], ez[3];          // the differences that feed Dxz u_z, Dyz u_z, Dzx u_x + Dzy u_y
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            const T* q = sp + f * FIELD;
            const T ctr = q[0];
            st.win[f][n8] = ctr;
            const T xp1 = q[1], xm1 = q[-1], xp2 = q[2], xm2 = q[-2], xp3 = q[3], xm3 = q[-3];
            const T yp1 = q[PXS], ym1 = q[-PXS], yp2 = q[2 * PXS], ym2 = q[-2 * PXS], yp3 = q[3 * PXS], ym3 = q[-3 * PXS];
            const T dx1 = xp1 - xm1, dx2 = xp2 - xm2, dx3 = xp3 - xm3;
            const T dy1 = yp1 - ym1, dy2 = yp2 - ym2, dy3 = yp3 - ym3;
            st.dl[2 * f][n4] = c.a[0] * dx1 + c.a[1] * dx2 + c.a[2] * dx3;
            st.dl[2 * f + 1][n4] = c.a[0] * dy1 + c.a[1] * dy2 + c.a[2] * dy3;
            if (f > 0) {
                const T sx1 = xp1 + xm1, sx2 = xp2 + xm2, sx3 = xp3 + xm3;
                const T sy1 = yp1 + ym1, sy2 = yp2 + ym2, sy3 = yp3 + ym3;
                const T* bx = f == 1 ? c.lq : c.lo;  // d_xx u_x and d_yy u_y carry 4nu/3 on the 55-point path
                const T* by = f == 2 ? c.lq : c.lo;
                inpl[f - 1] = c.cxy[f - 1] * ctr + bx[1] * sx1 + bx[2] * sx2 + bx[3] * sx3 + by[1] * sy1 + by[2] * sy2 + by[3] * sy3;
            }
            if (PATH55) {
                if (f == 1) { ez[0] = dx1; ez[1] = dx2; ez[2] = dx3; }
                if (f == 2) { ez[0] += dy1; ez[1] += dy2; ez[2] += dy3; }
                if (f == 3) { ex[0] = dx1; ex[1] = dx2; ex[2] = dx3; ey[0] = dy1; ey[1] = dy2; ey[2] = dy3; }
                if (f == 1 || f == 2) {  // Eq. 8 in the xy plane: d_xy u_x -> (grad div)_y, d_xy u_y -> (grad div)_x
                    const T q1 = (q[PXS + 1] - q[PXS - 1]) + (q[-PXS - 1] - q[-PXS + 1]);
                    const T q2 = (q[2 * PXS + 2] - q[2 * PXS - 2]) + (q[-2 * PXS - 2] - q[-2 * PXS + 2]);
                    const T q3 = (q[3 * PXS + 3] - q[3 * PXS - 3]) + (q[-3 * PXS - 3] - q[-3 * PXS + 3]);
                    const T dq = c.mq[0] * q1 + c.mq[1] * q2 + c.mq[2] * q3;
                    if (f == 1) dgy = dq; else dgx = dq;
                }
            }
        }
        if (PATH55) {
            inpl[0] += dgx;
            inpl[1] += dgy;
            const T* e[3] = {ex, ey, ez};
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                st.lin[i][(n8 + 3) & 7] = -(c.mq[2] * e[i][2]);  // first contribution to output t+3
                st.lin[i][(n8 + 2) & 7] -= c.mq[1] * e[i][1];
                st.lin[i][(n8 + 1) & 7] -= c.mq[0] * e[i][0];
                st.lin[i][n8] += inpl[i];
                st.lin[i][(n8 + 7) & 7] += c.mq[0] * e[i][0];
                st.lin[i][(n8 + 6) & 7] += c.mq[1] * e[i][1];
                st.lin[i][(n8 + 5) & 7] += c.mq[2] * e[i][2];  // output t-3 is complete
            }
        } else {
#pragma unroll
            for (int i = 0; i < 3; ++i) st.lin[i][n8] = inpl[i];
        }
        if (!out) return;
        // ---- output plane z = t - 3: z derivatives from the window, Eq. 1-3, Eq. 10
        constexpr int cz = (n8 + 5) & 7, r4 = (n4 + 1) & 3;
        T d1z[4], fc[4];
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            fc[f] = st.win[f][cz];
            d1z[f] = c.a[0] * (st.win[f][(cz + 1) & 7] - st.win[f][(cz + 7) & 7]) + c.a[1] * (st.win[f][(cz + 2) & 7] - st.win[f][(cz + 6) & 7]) +
                     c.a[2] * (st.win[f][(cz + 3) & 7] - st.win[f][(cz + 5) & 7]);
        }
        T lin[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const T* bz = i == 2 ? c.lq : c.lo;
            const int f = i + 1;
            lin[i] = st.lin[i][cz] + (bz[0] * fc[f] + bz[1] * (st.win[f][(cz + 1) & 7] + st.win[f][(cz + 7) & 7]) +
                                      bz[2] * (st.win[f][(cz + 2) & 7] + st.win[f][(cz + 6) & 7]) +
                                      bz[3] * (st.win[f][(cz + 3) & 7] + st.win[f][(cz + 5) & 7]));
        }
        const T g[3] = {st.dl[0][r4], st.dl[1][r4], d1z[0]};
        const T u[3] = {fc[1], fc[2], fc[3]};
        T G[3][3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            G[i][0] = st.dl[2 * (i + 1)][r4];
            G[i][1] = st.dl[2 * (i + 1) + 1][r4];
            G[i][2] = d1z[i + 1];
        }
        const T div = G[0][0] + G[1][1] + G[2][2];
        T Rv[4];
        Rv[0] = -(u[0] * g[0] + u[1] * g[1] + u[2] * g[2]) - div;
        const T tdiv = c.nu23 * div;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const T adv = u[0] * G[i][0] + u[1] * G[i][1] + u[2] * G[i][2];
            const T sg = (G[i][0] + G[0][i]) * g[0] + (G[i][1] + G[1][i]) * g[1] + (G[i][2] + G[2][i]) * g[2];
            Rv[1 + i] = (c.nu * sg - tdiv * g[i]) - adv - c.cs2 * g[i] + lin[i];
        }
        if (store_ok) {
            if (!PATH55) *dv = div;
#pragma unroll
            for (int f = 0; f < 4; ++f) {
                const T wn = s.read_w ? s.alpha * wold[f] + s.dt * Rv[f] : s.dt * Rv[f];
                if (s.write_w) wq[f * n] = wn;
                if (s.write_f) fo[f * fs] = fc[f] + s.beta * wn;
            }
        }
    }

    static __device__ __forceinline__ void run(const CUtensorMap* tm, T* __restrict__ Fout, T* __restrict__ W, T* __restrict__ Div,
                                               const Geom& g, const TCoef<T>& c, const Sub<T>& s, int zc) {
        extern __shared__ __align__(128) unsigned char smem_raw[];
        T* sm = reinterpret_cast<T*>(smem_raw);
        uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)S * STAGE * sizeof(T));
        const int tx = threadIdx.x, ty = threadIdx.y;
        const int tid = ty * TX + tx;
        const int X0 = blockIdx.x * TX, Y0 = blockIdx.y * TY;
        const int zs = blockIdx.z * zc, ze = min(zs + zc, g.nz);
        const int np = ze - zs + 2 * R;  // staged planes t = zs-3 .. ze+2
        const int bx = g.gx + X0 - 4, by = g.gy + Y0 - R, bz = g.gz + zs - R;
        constexpr uint32_t kStageBytes = (uint32_t)(STAGE * sizeof(T));
        if (tid == 0) {
#pragma unroll
            for (int i = 0; i < S; ++i) mbar_init(&full[i], 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
        if (tid == 0) {
            for (int i = 0; i < S && i < np; ++i) {
                mbar_expect_tx(&full[i], kStageBytes);
                tma_load_4d(sm + i * STAGE, tm, &full[i], bx, by, bz + i, 0);
            }
        }
        const int i = X0 + tx, j = Y0 + ty;
        const bool store_ok = i < g.nx && j < g.ny;
        const long long plane_w = (long long)g.nx * g.ny, plane_f = (long long)g.px * g.py;
        // pointers of output plane zs; advanced by one plane per produced output
        long long ow = i + (long long)g.nx * (j + (long long)g.ny * zs);
        long long of = (i + g.gx) + (long long)g.px * ((j + g.gy) + (long long)g.py * (zs + g.gz));
        if (!store_ok) { ow = 0; of = 0; }
        const T* sp0 = sm + (ty + R) * PXS + (tx + 4);
        State st;
#pragma unroll
        for (int a = 0; a < 8; ++a) {
#pragma unroll
            for (int f = 0; f < 4; ++f) st.win[f][a] = T(0);
#pragma unroll
            for (int q = 0; q < 3; ++q) st.lin[q][a] = T(0);
        }
#pragma unroll
        for (int q = 0; q < 8; ++q)
#pragma unroll
            for (int a = 0; a < 4; ++a) st.dl[q][a] = T(0);

        for (int pb = 0; pb < np; pb += 8) {
#pragma unroll
            for (int ph = 0; ph < 8; ++ph) {
                const int p = pb + ph;
                if (p < np) {
                    mbar_wait(&full[ph & 3], (uint32_t)((p >> 2) & 1));
                    switch (ph) {  // ph is a compile-time constant after unrolling
                        case 0: step<0>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                        case 1: step<1>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                        case 2: step<2>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                        case 3: step<3>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                        case 4: step<4>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                        case 5: step<5>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                        case 6: step<6>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                        default: step<7>(st, sp0, c, s, p, store_ok, W + ow, W + ow, Fout + of, Div + of, g.fs, g.n); break;
                    }
                    if (p >= 2 * R && store_ok) {
                        ow += plane_w;
                        of += plane_f;
                    }
                    __syncthreads();  // every thread is done reading stage ph&3
                    if (tid == 0 && p + S < np) {
                        mbar_expect_tx(&full[ph & 3], kStageBytes);
                        tma_load_4d(sm + (ph & 3) * STAGE, tm, &full[ph & 3], bx, by, bz + p + S, 0);
                    }
                }
            }
        }
    }
};

template <class T, bool PATH55, int TX, int TY>
__global__ void __launch_bounds__(TX* TY, 1)
    k_tiled_main(const __grid_constant__ CUtensorMap tm, T* __restrict__ Fout, T* __restrict__ W, T* __restrict__ Div, const Geom g,
                 const TCoef<T> c, const Sub<T> s, int zc) {
    Tiled<T, PATH55, TX, TY>::run(&tm, Fout, W, Div, g, c, s, zc);
}

// Tile shape per element type (registers per thread bound the CTA size).
template <class T>
struct TileShape;
template <>
struct TileShape<float> {
    static constexpr int TX = 64, TY = 8;
};
template <>
struct TileShape<double> {
    static constexpr int TX = 32, TY = 8;
};

// ---- host side -------------------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TiledState {
    bool ready = false;
    CUtensorMap tmF[2];
    int zc = 0;        // planes per z chunk
    int sm_count = 0;
    char err[256] = "";
};

inline bool tiled_supported(const Geom& g, int /*dtype*/) { return g.nx >= 8 && g.ny >= 8 && g.nz >= 8; }

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

template <class T>
static int tiled_make_map(TiledState& ts, CUtensorMap* tm, void* base, const Geom& g) {
    PFN_encodeTiled enc = tiled_encode_fn();
    if (!enc) {
        snprintf(ts.err, sizeof(ts.err), "cuTensorMapEncodeTiled is not available from this driver");
        return 3;
    }
    constexpr int TX = TileShape<T>::TX, TY = TileShape<T>::TY;
    const cuuint64_t dims[4] = {(cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz, 4};
    const cuuint64_t strides[3] = {(cuuint64_t)g.px * sizeof(T), (cuuint64_t)g.px * g.py * sizeof(T), (cuuint64_t)g.fs * sizeof(T)};
    const cuuint32_t box[4] = {(cuuint32_t)(TX + 8), (cuuint32_t)(TY + 2 * R), 1, 4};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(tm, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box,
                     estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(ts.err, sizeof(ts.err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return 3;
    }
    return 0;
}

template <class T>
static int tiled_prepare_t(TiledState& ts, const Geom& g, void* F0, void* F1) {
    int rc = tiled_make_map<T>(ts, &ts.tmF[0], F0, g);
    if (rc == 0) rc = tiled_make_map<T>(ts, &ts.tmF[1], F1, g);
    if (rc) return rc;
    constexpr int TX = TileShape<T>::TX, TY = TileShape<T>::TY;
    cudaError_t e = cudaFuncSetAttribute(k_tiled_main<T, true, TX, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)Tiled<T, true, TX, TY>::SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_tiled_main<T, false, TX, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)Tiled<T, false, TX, TY>::SMEM);
    if (e != cudaSuccess) {
        snprintf(ts.err, sizeof(ts.err), "cudaFuncSetAttribute(smem): %s", cudaGetErrorString(e));
        cudaGetLastError();
        return 3;
    }
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&ts.sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (ts.sm_count <= 0) ts.sm_count = 148;
    // z chunking: one CTA per SM is resident; pick the number of chunks that fills whole waves of SMs best while
    // keeping the 6-plane warm-up of every chunk below ~5 %.
    const long long tiles = (long long)((g.nx + TX - 1) / TX) * ((g.ny + TY - 1) / TY);
    int best_c = 1;
    double best_cost = 1e300;
    for (int cks = 1; cks <= g.nz / 8 && cks <= 64; ++cks) {
        const int zc = (g.nz + cks - 1) / cks;
        const int real = (g.nz + zc - 1) / zc;
        const long long ctas = tiles * real;
        const long long waves = (ctas + ts.sm_count - 1) / ts.sm_count;
        const double cost = (double)waves * (zc + 2 * R + 4);  // time ~ waves x planes staged per CTA (+ fill latency)
        if (cost < best_cost) {
            best_cost = cost;
            best_c = cks;
        }
    }
    ts.zc = (g.nz + best_c - 1) / best_c;
    ts.ready = true;
    return 0;
}

inline const char* tiled_error_of(const TiledState& ts) { return ts.err; }

inline int tiled_prepare(TiledState& ts, const Geom& g, int dtype, void* F0, void* F1, void* /*Div*/) {
    ts.ready = false;
    return dtype == 0 ? tiled_prepare_t<float>(ts, g, F0, F1) : tiled_prepare_t<double>(ts, g, F0, F1);
}
inline void tiled_release(TiledState& ts) { ts.ready = false; }

template <class T>
static TCoef<T> make_tcoef(double dx, double nu, double cs, bool path55) {
    const double dx2 = dx * dx;
    const double b[4] = {-490.0 / (180.0 * dx2), 270.0 / (180.0 * dx2), -27.0 / (180.0 * dx2), 2.0 / (180.0 * dx2)};
    const double cm[3] = {270.0 / (720.0 * dx2), -27.0 / (720.0 * dx2), 2.0 / (720.0 * dx2)};
    const double own = path55 ? 4.0 * nu / 3.0 : nu;
    TCoef<T> k;
    k.a[0] = T(45.0 / (60.0 * dx));
    k.a[1] = T(-9.0 / (60.0 * dx));
    k.a[2] = T(1.0 / (60.0 * dx));
    for (int m = 0; m < 4; ++m) {
        k.lo[m] = T(nu * b[m]);
        k.lq[m] = T(own * b[m]);
    }
    k.cxy[0] = T((own + nu) * b[0]);
    k.cxy[1] = T((own + nu) * b[0]);
    k.cxy[2] = T(2.0 * nu * b[0]);
    for (int m = 0; m < 3; ++m) k.mq[m] = T(nu / 3.0 * cm[m]);
    k.nu = T(nu);
    k.cs2 = T(cs * cs);
    k.nu23 = T(2.0 * nu / 3.0);
    return k;
}

// Launch of the main kernel of one substep (fused 55-point kernel, or pass 1 of the 19-point path).
template <class T>
static int tiled_launch_main(TiledState& ts, int path55, int cur, T* Fout, T* W, T* Div, const Geom& g, double dx, double nu, double cs,
                             const Sub<T>& s, cudaStream_t stream) {
    constexpr int TX = TileShape<T>::TX, TY = TileShape<T>::TY;
    dim3 block(TX, TY, 1), grid((g.nx + TX - 1) / TX, (g.ny + TY - 1) / TY, (g.nz + ts.zc - 1) / ts.zc);
    const TCoef<T> c = make_tcoef<T>(dx, nu, cs, path55 != 0);
    if (path55)
        k_tiled_main<T, true, TX, TY><<<grid, block, Tiled<T, true, TX, TY>::SMEM, stream>>>(ts.tmF[cur], Fout, W, Div, g, c, s, ts.zc);
    else
        k_tiled_main<T, false, TX, TY><<<grid, block, Tiled<T, false, TX, TY>::SMEM, stream>>>(ts.tmF[cur], Fout, W, Div, g, c, s, ts.zc);
    return cudaGetLastError() == cudaSuccess ? 0 : 3;
}

}  // namespace fd6
