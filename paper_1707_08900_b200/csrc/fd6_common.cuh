// fd6_common.cuh — shared device-side definitions of libfd6 (product code; shares nothing with oracle/).
//
// Notation follows the paper: F = (ln rho, u_x, u_y, u_z), w = the 2N-RK intermediate
// arrays, R = stencil radius 3.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fd6 {

constexpr int R = 3;  // stencil radius, "For both stencils, R = 3"

// ------------------------------------------------------------------------------------------------
// V2 — two fp32 cells in one 64-bit value.  In the paired layout cell
// (i,j,k) and cell (i,j,k+nz/2) are stored side by side, so every kernel sees a grid of nz/2 planes whose
// elements are V2, and the arithmetic on both cells is ONE packed instruction (Blackwell FFMA2 / FADD2 /
// FMUL2: fma.rn.f32x2 etc., PTX ISA 8.6, sm_100) with both halves rounded exactly like the scalar op.
// ------------------------------------------------------------------------------------------------
struct __align__(8) V2 {
    float2 v;
    V2() = default;
    __host__ __device__ explicit V2(float s) : v{s, s} {}
    __host__ __device__ explicit V2(double s) : v{(float)s, (float)s} {}
    __host__ __device__ explicit V2(int s) : v{(float)s, (float)s} {}
    __host__ __device__ V2(float lo, float hi) : v{lo, hi} {}
};
__device__ __forceinline__ V2 mk(float2 f) {
    V2 r;
    r.v = f;
    return r;
}
__device__ __forceinline__ V2 operator+(V2 a, V2 b) { return mk(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ V2 operator-(V2 a) { return V2(-a.v.x, -a.v.y); }
__device__ __forceinline__ V2 operator-(V2 a, V2 b) { return mk(__fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y))); }
__device__ __forceinline__ V2 operator*(V2 a, V2 b) { return mk(__fmul2_rn(a.v, b.v)); }
__device__ __forceinline__ V2& operator+=(V2& a, V2 b) { return a = a + b; }
__device__ __forceinline__ V2& operator-=(V2& a, V2 b) { return a = a - b; }

// fma_(a, b, c) = a*b + c with one rounding, for every value type the kernels are instantiated on.
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ V2 fma_(V2 a, V2 b, V2 c) { return mk(__ffma2_rn(a.v, b.v, c.v)); }

// Periodic wrap across the z boundary of the stored grid: in the paired layout the plane below plane 0 is
// plane nz/2-1 of the OTHER half, so the two halves of every value trade places; scalars are unchanged.
template <class T>
__device__ __forceinline__ T zwrap(T v) { return v; }
template <>
__device__ __forceinline__ V2 zwrap<V2>(V2 v) { return V2(v.v.y, v.v.x); }

// Scalar type behind a value type, and cells per value.
template <class T> struct Scalar { typedef T type; static constexpr int lanes = 1; };
template <> struct Scalar<V2> { typedef float type; static constexpr int lanes = 2; };

// make_value<T>(lo, hi): a value from the scalars of its cell(s): lo for a plain type, (lo, hi) for a V2 pair.
template <class T> __host__ __device__ __forceinline__ T make_value(typename Scalar<T>::type lo, typename Scalar<T>::type) { return T(lo); }
template <> __host__ __device__ __forceinline__ V2 make_value<V2>(float lo, float hi) { return V2(lo, hi); }

// Forcing term of Eq. 2 (Eq. 24-25):  f = N f_k cos(k.x + phi), x = (i, j, k) dx.  The phase is
// separable, so the host tabulates (in double, rounded once) cos and sin of k_x x_i + phi, of k_y y_j and of k_z z_k;
// `tab` holds them back to back as scalars: cx[nx] sx[nx] cy[ny] sy[ny] cz[nzc] sz[nzc], nzc = the CALLER's nz.
// A kernel forms cos(theta) = cxy cz - sxy sz with cxy = cx cy - sx sy, sxy = sx cy + cx sy.
template <class T>
struct ForceTab {
    const typename Scalar<T>::type* tab;  // NULL: forcing off
    int nx, ny, nzc;
    __device__ __forceinline__ void xy(int i, int j, T& cxy, T& sxy) const {
        typedef typename Scalar<T>::type S;
        const S cx = tab[i], sx = tab[nx + i], cy = tab[2 * nx + j], sy = tab[2 * nx + ny + j];
        cxy = T(cx * cy - sx * sy);
        sxy = T(sx * cy + cx * sy);
    }
    // stored plane z holds cells z (and z + nzc/2 in the paired layout)
    __device__ __forceinline__ void z(int zz, T& cz, T& sz) const {
        const typename Scalar<T>::type* c = tab + 2 * nx + 2 * ny;
        const int hi = Scalar<T>::lanes == 2 ? zz + nzc / 2 : zz;
        cz = make_value<T>(c[zz], c[hi]);
        sz = make_value<T>(c[nzc + zz], c[nzc + hi]);
    }
};

// Ghost-padded array geometry, in units of the value type T of the kernels (one cell,
// or a V2 pair of cells: then nz is HALF the caller's nz).  Value (i,j,k) of a padded field lives at
//   (i + gx) + px * ((j + gy) + py * (k + gz));  the four fields of one copy are fs values apart.
struct Geom {
    int nx, ny, nz;
    int px, py, pz;
    int gx, gy, gz;
    long long fs;  // padded field stride (elements)
    long long n;   // nx*ny*nz, the dense (w) field stride
};

// Stencil coefficients of Eq. 6-8 pre-divided by their denominators, and the physics constants.
template <class T>
struct Coef {
    T a1, a2, a3;      // Eq. 6:  45, -9, 1   over 60 dx
    T b0, b1, b2, b3;  // Eq. 7: -490, 270, -27, 2 over 180 dx^2
    T m1, m2, m3;      // Eq. 8:  270, -27, 2 over 720 dx^2
    T nu, nu3, cs2;    // nu, nu/3, cs^2
    T fa[3];           // N f_k of the forcing term (Eq. 24-25); used only when a ForceTab is given
};

// One RK substep (Eq. 10):  w <- alpha w + dt rhs ; F_out <- F + beta w.
//   read_w == 0  : alpha is 0 and w is NOT read (alpha^(1) = 0; stale/NaN w cannot leak)
//   write_f == 0 : only w is written (fd_rhs uses alpha = 0, dt = 1 to obtain the plain right-hand side)
//   write_w == 0 : w is not written (last substep of a step: the next substep has alpha = 0 and never reads it)
template <class T>
struct Sub {
    T alpha, beta, dt;
    int read_w, write_f, write_w;
};

// Eq. 6 / 7 / 8 around pointer f with element strides s (one axis) or sa, sb (a plane).
template <class T>
__device__ __forceinline__ T d1(const T* __restrict__ f, long long s, const Coef<T>& c) {
    return c.a1 * (f[s] - f[-s]) + c.a2 * (f[2 * s] - f[-2 * s]) + c.a3 * (f[3 * s] - f[-3 * s]);
}
template <class T>
__device__ __forceinline__ T d2(const T* __restrict__ f, long long s, const Coef<T>& c) {
    return c.b0 * f[0] + c.b1 * (f[s] + f[-s]) + c.b2 * (f[2 * s] + f[-2 * s]) + c.b3 * (f[3 * s] + f[-3 * s]);
}
template <class T>
__device__ __forceinline__ T dmix(const T* __restrict__ f, long long sa, long long sb, const Coef<T>& c) {
    T q1 = (f[sa + sb] - f[-sa + sb]) + (f[-sa - sb] - f[sa - sb]);
    T q2 = (f[2 * sa + 2 * sb] - f[-2 * sa + 2 * sb]) + (f[-2 * sa - 2 * sb] - f[2 * sa - 2 * sb]);
    T q3 = (f[3 * sa + 3 * sb] - f[-3 * sa + 3 * sb]) + (f[-3 * sa - 3 * sb] - f[3 * sa - 3 * sb]);
    return c.m1 * q1 + c.m2 * q2 + c.m3 * q3;
}

// Eq. 1-3 assembled from the derivative values at one cell.
//   u[i]; g[j] = d_j ln rho; G[i][j] = d_j u_i; L[i] = sum_j d_jj u_i; Q[i] = (grad div u)_i (ignored if !withQ).
// R[0] = -u.g - div u;  R[1+i] = -u.grad u_i - cs^2 g_i + nu (L_i + Q_i/3 + 2 S_ij g_j),
// S_ij = (G_ij + G_ji)/2 - delta_ij div/3  =>  2 S_ij g_j = sum_j (G_ij + G_ji) g_j - (2/3) div g_i.
template <class T, bool withQ>
__device__ __forceinline__ void assemble(const T u[3], const T g[3], const T G[3][3], const T L[3], const T Q[3],
                                         const Coef<T>& c, T Rout[4]) {
    const T div = G[0][0] + G[1][1] + G[2][2];
    Rout[0] = -(u[0] * g[0] + u[1] * g[1] + u[2] * g[2]) - div;
    const T twothirds_div = T(2.0 / 3.0) * div;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        T adv = u[0] * G[i][0] + u[1] * G[i][1] + u[2] * G[i][2];
        T sg = (G[i][0] + G[0][i]) * g[0] + (G[i][1] + G[1][i]) * g[1] + (G[i][2] + G[2][i]) * g[2] - twothirds_div * g[i];
        T visc = L[i] + sg;
        T r = c.nu * visc - adv - c.cs2 * g[i];
        if (withQ) r += c.nu3 * Q[i];
        Rout[1 + i] = r;
    }
}

// Eq. 10 on one value.
template <class T>
__device__ __forceinline__ T rk_w(const Sub<T>& s, T rhs, const T* __restrict__ w_ptr) {
    return s.read_w ? s.alpha * (*w_ptr) + s.dt * rhs : s.dt * rhs;
}

}  // namespace fd6
