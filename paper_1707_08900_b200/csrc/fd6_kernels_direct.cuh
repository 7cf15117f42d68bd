// fd6_kernels_direct.cuh — layout kernels (pack/unpack, periodic halo fill) and the FD_VARIANT_DIRECT
// derivative/update kernels: one thread per cell, neighbours straight from the ghost-padded arrays through
// L1/L2.  Simple and size-agnostic; the tiled TMA kernels in fd6_kernels_tiled.cuh are the fast path.
#pragma once
#include "fd6_common.cuh"

namespace fd6 {

// ------------------------------------------------------------------------------------------------
// a0  pack / unpack: caller's dense arrays <-> interior of the padded arrays.
// grid (ceil(nx/128), ny, nz) x 4 fields through blockIdx.z = k + nz*q.
// ------------------------------------------------------------------------------------------------
// Dense caller arrays hold scalars; in the paired layout value (i,j,k) gathers cells k and k + g.nz.
template <class T>
__device__ __forceinline__ T dense_get(const typename Scalar<T>::type* __restrict__ a, long long idx, long long half) {
    return a[idx];
}
template <>
__device__ __forceinline__ V2 dense_get<V2>(const float* __restrict__ a, long long idx, long long half) {
    return V2(a[idx], a[idx + half]);
}
template <class T>
__device__ __forceinline__ void dense_put(typename Scalar<T>::type* __restrict__ a, long long idx, long long half, T v) {
    a[idx] = v;
}
template <>
__device__ __forceinline__ void dense_put<V2>(float* __restrict__ a, long long idx, long long half, V2 v) {
    a[idx] = v.v.x;
    a[idx + half] = v.v.y;
}

template <class T>
__global__ void __launch_bounds__(128)
    k_pack(const typename Scalar<T>::type* __restrict__ d0, const typename Scalar<T>::type* __restrict__ d1_,
           const typename Scalar<T>::type* __restrict__ d2_, const typename Scalar<T>::type* __restrict__ d3, T* __restrict__ F, Geom g) {
    int i = blockIdx.x * 128 + threadIdx.x, j = blockIdx.y, k = blockIdx.z % g.nz, q = blockIdx.z / g.nz;
    if (i >= g.nx) return;
    const typename Scalar<T>::type* src = q == 0 ? d0 : (q == 1 ? d1_ : (q == 2 ? d2_ : d3));
    F[q * g.fs + (i + g.gx) + (long long)g.px * ((j + g.gy) + (long long)g.py * (k + g.gz))] =
        dense_get<T>(src, i + (long long)g.nx * (j + (long long)g.ny * k), g.n);
}

template <class T>
__global__ void __launch_bounds__(128)
    k_unpack(const T* __restrict__ F, typename Scalar<T>::type* __restrict__ d0, typename Scalar<T>::type* __restrict__ d1_,
             typename Scalar<T>::type* __restrict__ d2_, typename Scalar<T>::type* __restrict__ d3, Geom g) {
    int i = blockIdx.x * 128 + threadIdx.x, j = blockIdx.y, k = blockIdx.z % g.nz, q = blockIdx.z / g.nz;
    if (i >= g.nx) return;
    typename Scalar<T>::type* dst = q == 0 ? d0 : (q == 1 ? d1_ : (q == 2 ? d2_ : d3));
    dense_put<T>(dst, i + (long long)g.nx * (j + (long long)g.ny * k), g.n,
                 F[q * g.fs + (i + g.gx) + (long long)g.px * ((j + g.gy) + (long long)g.py * (k + g.gz))]);
}

// ------------------------------------------------------------------------------------------------
// a1 / a7  periodic halo fill, radius 3 (Alg. 2/3 "Compute boundary conditions").
//   (T = V2: the stored grid has nz/2 planes and z-periodicity swaps the halves of a pair, see zwrap.)
//   One kernel, every ghost value read straight from the interior (no ordering between faces):
//   blocks [0, row_blocks): `rpb` ghost ROWS each (rpb > 1 on narrow grids, where a row has fewer sectors than the block has
//       threads; row index in [0, nfields * yz_rows)); a ghost row (j or k outside the domain) = the x-extended copy of the
//       interior row it wraps to, its own 2R x ghosts taken from the far end of that row; this also fills the
//       edge ghosts (two coordinates outside) the Eq. 8 diagonals read, and the corners (never read);
//   remaining blocks: the x ghosts of the interior rows, one thread per (row, side): the x ghost pad is exactly one
//       32-byte sector (gx values) and rows are 32-byte aligned, so a side is one aligned sector copy — the low pad
//       [0, gx) takes the last gx interior values, the high pad the first gx (only R of them are ever read).
// ------------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(128) k_halo(T* __restrict__ F, Geom g, int nfields, int yz_rows, int rpb, int row_blocks) {
    if ((int)blockIdx.x < row_blocks) {
        // ghost rows: first the 2R ghost z-planes (py rows each), then for every interior plane its 2R ghost y-rows
        const int tpr = 128 / rpb;  // threads per row
        const int row = blockIdx.x * rpb + threadIdx.x / tpr, lane = threadIdx.x - (threadIdx.x / tpr) * tpr;
        if (row >= nfields * yz_rows) return;
        const int q = row / yz_rows;
        int b = row - q * yz_rows, jj, kk;
        const int zrows = 2 * R * g.py;
        if (b < zrows) {
            int zp = b / g.py;
            jj = b - zp * g.py;
            kk = zp < R ? zp + (g.gz - R) : g.gz + g.nz + (zp - R);
        } else {
            b -= zrows;
            int k = b / (2 * R), yr = b - k * (2 * R);
            kk = k + g.gz;
            jj = yr < R ? yr + (g.gy - R) : g.gy + g.ny + (yr - R);
        }
        int js = jj - g.gy, ks = kk - g.gz;  // wrap to the interior row (n >= R: one correction suffices)
        js += js < 0 ? g.ny : 0;
        js -= js >= g.ny ? g.ny : 0;
        const bool zw = ks < 0 || ks >= g.nz;  // paired layout: crossing the z boundary swaps the two halves
        ks += ks < 0 ? g.nz : 0;
        ks -= ks >= g.nz ? g.nz : 0;
        T* base = F + q * g.fs;
        T* drow = base + (long long)g.px * (jj + (long long)g.py * kk);
        const T* srow = base + (long long)g.px * ((js + g.gy) + (long long)g.py * (ks + g.gz));
        if (g.nx % g.gx == 0) {
            // whole 32-byte sectors (gx values): sector 0 is the low pad, the last one the high pad
            constexpr int VPS = (int)(32 / sizeof(T));  // == g.gx
            const int nsec = g.nx / VPS + 2;
            for (int sct = lane; sct < nsec; sct += tpr) {
                const int ssrc = sct == 0 ? nsec - 2 : (sct == nsec - 1 ? 1 : sct);
                union { uint4 u[2]; T v[VPS]; } buf;
                const uint4* sp = reinterpret_cast<const uint4*>(srow + ssrc * VPS);
                buf.u[0] = sp[0];
                buf.u[1] = sp[1];
                if (zw) {
#pragma unroll
                    for (int e = 0; e < VPS; ++e) buf.v[e] = zwrap<T>(buf.v[e]);
                }
                uint4* dp = reinterpret_cast<uint4*>(drow + sct * VPS);
                dp[0] = buf.u[0];
                dp[1] = buf.u[1];
            }
        } else {
            T* dst = drow + (g.gx - R);
            const T* src = srow + (g.gx - R);
            for (int x = lane; x < g.nx + 2 * R; x += tpr) {
                const int xs = x < R ? x + g.nx : (x >= g.nx + R ? x - g.nx : x);
                const T v = src[xs];
                dst[x] = zw ? zwrap<T>(v) : v;
            }
        }
        return;
    }
    long long t = (long long)(blockIdx.x - row_blocks) * 128 + threadIdx.x;
    const int side = (int)(t & 1);
    t >>= 1;
    long long rows = (long long)g.ny * g.nz;
    if (t >= rows * nfields) return;
    int q = (int)(t / rows);
    long long r = t - q * rows;
    int j = (int)(r % g.ny), k = (int)(r / g.ny);
    T* row = F + q * g.fs + (long long)g.px * ((j + g.gy) + (long long)g.py * (k + g.gz));
    const uint4* src = reinterpret_cast<const uint4*>(side ? row + g.gx : row + g.nx);
    uint4* dst = reinterpret_cast<uint4*>(side ? row + g.gx + g.nx : row);
    const uint4 a = src[0], b = src[1];
    dst[0] = a;
    dst[1] = b;
}

// ------------------------------------------------------------------------------------------------
// a2-a4 (PATH55 = true) fused 55-point kernel:  27 derivatives, Eq. 1-3, Eq. 10           (Alg. 2)
// a6    (PATH55 = false) 19-point pass 1: div u to global, partial update without nu/3 grad div (Eq. 14-16)
// block (64,4,1), grid (ceil(nx/64), ceil(ny/4), nz): one thread per cell.
// ------------------------------------------------------------------------------------------------
template <class T, bool PATH55>
__global__ void __launch_bounds__(256) k_direct_main(const T* __restrict__ Fin, T* __restrict__ Fout, T* __restrict__ W,
                                                     T* __restrict__ Div, Geom g, Coef<T> c, Sub<T> s, ForceTab<T> ft) {
    int i = blockIdx.x * 64 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k = blockIdx.z;
    if (i >= g.nx || j >= g.ny) return;
    const long long sx = 1, sy = g.px, sz = (long long)g.px * g.py;
    const long long p = (i + g.gx) + sy * (j + g.gy) + sz * (k + g.gz);
    const long long pw = i + (long long)g.nx * (j + (long long)g.ny * k);
    const T* l = Fin + p;
    const T* uu[3] = {Fin + g.fs + p, Fin + 2 * g.fs + p, Fin + 3 * g.fs + p};
    const long long st[3] = {sx, sy, sz};

    T u[3], gl[3], G[3][3], L[3], Q[3] = {T(0), T(0), T(0)};
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
        if (PATH55) Q[q] = dd[q];  // d_qq u_q is shared between the Laplacian and grad div
    }
    if (PATH55) {
        Q[0] += dmix(uu[1], sx, sy, c) + dmix(uu[2], sx, sz, c);
        Q[1] += dmix(uu[0], sy, sx, c) + dmix(uu[2], sy, sz, c);
        Q[2] += dmix(uu[0], sz, sx, c) + dmix(uu[1], sz, sy, c);
    }
    T Rv[4];
    assemble<T, PATH55>(u, gl, G, L, Q, c, Rv);
    if (ft.tab) {  // + f = N f_k cos(k.x + phi) (Eq. 2, Eq. 24-25)
        T cxy, sxy, cz, sz;
        ft.xy(i, j, cxy, sxy);
        ft.z(k, cz, sz);
        const T cth = cxy * cz - sxy * sz;
#pragma unroll
        for (int a = 0; a < 3; ++a) Rv[1 + a] += c.fa[a] * cth;
    }
    if (!PATH55) Div[p] = G[0][0] + G[1][1] + G[2][2];
    const T fc[4] = {l[0], u[0], u[1], u[2]};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        T* wp = W + q * g.n + pw;
        T wn = rk_w(s, Rv[q], wp);
        if (s.write_w) *wp = wn;
        if (s.write_f) Fout[q * g.fs + p] = fc[q] + s.beta * wn;
    }
}

// a8  19-point pass 2:  w_i += dt nu/3 D1_i(div) (Eq. 17);  F_out,i += beta dt nu/3 D1_i(div) (Eq. 18).
// Launch order: blocks run x fastest, then the gridDim.y block rows of a y band, then z, then the next band.  With
// one band (gridDim.y = all block rows) that is plane after plane, the best order for DRAM as long as the seven div
// planes a block reads stay in L2; at 1024^3 they do not (7 x 8.5 MB next to the streamed w and u), and bands of 16
// block rows keep them there (pass 2 at C5: 11.4 -> 10.2 ms; at C4 the banded order is 10 % slower).
// grid = (ceil(nx/64), band rows, bands * nz).
template <class T>
__global__ void __launch_bounds__(256) k_direct_pass2(const T* __restrict__ Div, T* __restrict__ Fout, T* __restrict__ W,
                                                      Geom g, Coef<T> c, Sub<T> s) {
    const int band = (int)gridDim.z == g.nz ? 0 : blockIdx.z / g.nz, k = blockIdx.z - band * g.nz;
    int i = blockIdx.x * 64 + threadIdx.x, j = (band * gridDim.y + blockIdx.y) * 4 + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const long long sy = g.px, sz = (long long)g.px * g.py;
    const long long p = (i + g.gx) + sy * (j + g.gy) + sz * (k + g.gz);
    const long long pw = i + (long long)g.nx * (j + (long long)g.ny * k);
    const long long st[3] = {1, sy, sz};
    const T scale = s.dt * c.nu3;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T add = scale * d1(Div + p, st[a], c);
        T* wp = W + (1 + a) * g.n + pw;
        if (s.write_w) *wp += add;
        if (s.write_f) Fout[(1 + a) * g.fs + p] += s.beta * add;
    }
}

// The same pass for the PLAIN fp32 layout with two x-adjacent cells per thread (8-byte accesses: as many bytes per load
// instruction as the paired layout has; one cell per thread is bound by the load/store unit: 1.6 against 1.17 ms at C4).
// nx is even (fd_create: nx % 4 == 0) and every row starts 32-byte aligned, so the pairs (2i, 2i+1) are aligned.
// grid = (ceil(nx/128), band rows, bands * nz), block (64, 4).
__global__ void __launch_bounds__(256) k_direct_pass2_x2(const float* __restrict__ Div, float* __restrict__ Fout, float* __restrict__ W,
                                                         Geom g, Coef<float> c, Sub<float> s) {
    const int band = (int)gridDim.z == g.nz ? 0 : blockIdx.z / g.nz, k = blockIdx.z - band * g.nz;
    const int i = 2 * (blockIdx.x * 64 + threadIdx.x), j = (band * gridDim.y + blockIdx.y) * 4 + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const long long sy = g.px, sz = (long long)g.px * g.py;
    const long long p = (i + g.gx) + sy * (j + g.gy) + sz * (k + g.gz);
    const long long pw = i + (long long)g.nx * (j + (long long)g.ny * k);
    const float scale = s.dt * c.nu3;
    auto ld2 = [&](long long off) { return *reinterpret_cast<const float2*>(Div + p + off); };
    float2 add[3];
    {   // Eq. 6 along x for cells i and i + 1 from the five aligned pairs that cover i-3 .. i+4
        const float2 a = ld2(-4), b = ld2(-2), m = ld2(0), d = ld2(2), e = ld2(4);
        add[0].x = scale * (c.a1 * (m.y - b.y) + c.a2 * (d.x - b.x) + c.a3 * (d.y - a.y));
        add[0].y = scale * (c.a1 * (d.x - m.x) + c.a2 * (d.y - b.y) + c.a3 * (e.x - b.x));
    }
#pragma unroll
    for (int ax = 1; ax < 3; ++ax) {
        const long long st = ax == 1 ? sy : sz;
        const float2 p1 = ld2(st), m1 = ld2(-st), p2 = ld2(2 * st), m2 = ld2(-2 * st), p3 = ld2(3 * st), m3 = ld2(-3 * st);
        add[ax].x = scale * (c.a1 * (p1.x - m1.x) + c.a2 * (p2.x - m2.x) + c.a3 * (p3.x - m3.x));
        add[ax].y = scale * (c.a1 * (p1.y - m1.y) + c.a2 * (p2.y - m2.y) + c.a3 * (p3.y - m3.y));
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (s.write_w) {
            float2* wp = reinterpret_cast<float2*>(W + (1 + a) * g.n + pw);
            float2 w = *wp;
            w.x += add[a].x;
            w.y += add[a].y;
            *wp = w;
        }
        if (s.write_f) {
            float2* fp = reinterpret_cast<float2*>(Fout + (1 + a) * g.fs + p);
            float2 f = *fp;
            f.x += s.beta * add[a].x;
            f.y += s.beta * add[a].y;
            *fp = f;
        }
    }
}

// a8 for the staged variants (8-byte value types: fp64 and the paired fp32 layout): two x-adjacent values per thread with
// 16-byte accesses, marching along z with the seven div planes of the z derivative in a register window, so a value costs
// 5.5 div loads of 16 bytes instead of 18 of 8 (4 for x beside the window's centre, 6 for y, 1 new plane for z, per pair)
// and every load of an iteration is issued before the first use.  nx is even (fd_create: nx % 4 == 0), rows of the padded
// and of the dense arrays start 32-byte aligned, so the pairs (2i, 2i+1) are 16-byte aligned; the x ghost pad holds 4
// values, which covers the aligned pair at i - 4 (its low half is never used).  Arithmetic per value is the expression of
// d1() on the same operands: results equal k_direct_pass2 bitwise.  Measured on B200 (profiles/r03_bench_C*_19.json.txt):
// C4 pass 2 1.19 -> 1.05 ms per launch, C5 +7.5 % per step; chunks of 8, 16 and 32 planes are within 0.3 %, 64 is 1.6 %
// slower; evict-first (ld/st.global.cs) accesses for w and F_out were 3 % SLOWER per step and are not used.
// grid = (ceil(nx/128), ceil(ny/4), ceil(nz/zc)), block (64, 4); a thread updates planes [blockIdx.z * zc, + zc).
template <class T>
struct __align__(16) Pair2 {
    T x, y;
};
template <class T>
__device__ __forceinline__ T d1v(T p1, T m1, T p2, T m2, T p3, T m3, const Coef<T>& c) {
    return c.a1 * (p1 - m1) + c.a2 * (p2 - m2) + c.a3 * (p3 - m3);
}
// WW = s.write_w at compile time: the last substep of a step does not touch w (Sub<T>), needs 12 registers fewer and runs
// three blocks per SM instead of two, which it needs to keep enough bytes in flight with half the streams.
template <class T, bool WW>
__global__ void __launch_bounds__(256, WW ? 2 : 3) k_pass2_march(const T* __restrict__ Div, T* __restrict__ Fout, T* __restrict__ W, Geom g,
                                                                 Coef<T> c, Sub<T> s, int zc) {
    static_assert(sizeof(T) == 8, "two 8-byte values per 16-byte access");
    typedef Pair2<T> P;
    const int i = 2 * (blockIdx.x * 64 + threadIdx.x), j = blockIdx.y * 4 + threadIdx.y, k0 = blockIdx.z * zc;
    if (i >= g.nx || j >= g.ny) return;
    const int k1 = min(k0 + zc, g.nz);
    const long long sy = g.px, sz = (long long)g.px * g.py;
    const T* d = Div + (i + g.gx) + sy * (j + g.gy) + sz * (k0 + g.gz);
    T* f = Fout + g.fs + (i + g.gx) + sy * (j + g.gy) + sz * (k0 + g.gz);
    T* w = W + g.n + i + (long long)g.nx * (j + (long long)g.ny * k0);
    const long long wz = (long long)g.nx * g.ny;
    auto ld = [](const T* p) { return *reinterpret_cast<const P*>(p); };
    auto st = [](T* p, P v) { *reinterpret_cast<P*>(p) = v; };
    const T scale = s.dt * c.nu3;
    P zm3 = ld(d - 3 * sz), zm2 = ld(d - 2 * sz), zm1 = ld(d - sz), z0 = ld(d), zp1 = ld(d + sz), zp2 = ld(d + 2 * sz);
    for (int k = k0; k < k1; ++k) {
        const P zp3 = ld(d + 3 * sz);
        const P xa = ld(d - 4), xb = ld(d - 2), xd = ld(d + 2), xe = ld(d + 4);
        const P yp1 = ld(d + sy), ym1 = ld(d - sy), yp2 = ld(d + 2 * sy), ym2 = ld(d - 2 * sy), yp3 = ld(d + 3 * sy), ym3 = ld(d - 3 * sy);
        P wv[3], fv[3];
        if (WW) {
#pragma unroll
            for (int a = 0; a < 3; ++a) wv[a] = ld(w + a * g.n);
        }
        if (s.write_f) {
#pragma unroll
            for (int a = 0; a < 3; ++a) fv[a] = ld(f + a * g.fs);
        }
        P add[3];
        // Eq. 6 along x for values i and i + 1 from the aligned pairs that cover i-3 .. i+4 (z0 is the pair itself)
        add[0].x = scale * d1v(z0.y, xb.y, xd.x, xb.x, xd.y, xa.y, c);
        add[0].y = scale * d1v(xd.x, z0.x, xd.y, xb.y, xe.x, xb.x, c);
        add[1].x = scale * d1v(yp1.x, ym1.x, yp2.x, ym2.x, yp3.x, ym3.x, c);
        add[1].y = scale * d1v(yp1.y, ym1.y, yp2.y, ym2.y, yp3.y, ym3.y, c);
        add[2].x = scale * d1v(zp1.x, zm1.x, zp2.x, zm2.x, zp3.x, zm3.x, c);
        add[2].y = scale * d1v(zp1.y, zm1.y, zp2.y, zm2.y, zp3.y, zm3.y, c);
        if (WW) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                wv[a].x += add[a].x;
                wv[a].y += add[a].y;
                st(w + a * g.n, wv[a]);
            }
        }
        if (s.write_f) {
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                fv[a].x += s.beta * add[a].x;
                fv[a].y += s.beta * add[a].y;
                st(f + a * g.fs, fv[a]);
            }
        }
        zm3 = zm2;
        zm2 = zm1;
        zm1 = z0;
        z0 = zp1;
        zp1 = zp2;
        zp2 = zp3;
        d += sz;
        f += sz;
        w += wz;
    }
}

// Test hooks: poison w / all ghost cells with NaN.
template <class T>
__global__ void k_fill(T* __restrict__ a, long long n, T v) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) a[t] = v;
}
template <class T>
__global__ void k_poison_ghosts(T* __restrict__ F, Geom g, T v) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    long long per = (long long)g.px * g.py * g.pz;
    if (t >= per * 4) return;
    int q = (int)(t / per);
    long long r = t - q * per;
    int x = (int)(r % g.px), y = (int)((r / g.px) % g.py), z = (int)(r / ((long long)g.px * g.py));
    bool interior = x >= g.gx && x < g.gx + g.nx && y >= g.gy && y < g.gy + g.ny && z >= g.gz && z < g.gz + g.nz;
    if (!interior) F[q * g.fs + r] = v;
}

}  // namespace fd6
