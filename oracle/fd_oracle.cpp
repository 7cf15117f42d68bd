// fd_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU oracle for the hot path of arXiv 1707.08900
// (Pekkilä et al.): one 2N-storage RK3 step of isothermal compressible hydrodynamics
// on a periodic 3-D grid with sixth-order central differences.  Written from
// /root/reference/PAPER.md only; every function cites the passage it follows.
//
// Rules this file keeps:
//   * no ghost zones, no tiling, no fusion, no SIMD intrinsics: periodic access by
//     modular indexing, one cell at a time, paper's order of terms;
//   * shares no code, header, table or helper with the CUDA path; nothing under
//     paper_1707_08900_b200/ includes or links this file;
//   * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
//     reference legs may load the library built from it.
//
// Parity status: every function below is pinned by tests/test_oracle_pins.py
// (P0..P13 of DESIGN.md; the forcing term O11 by P13) EXCEPT the nonlinear multi-step evolution of general
// fields beyond one substep, which is "parity unpinned beyond the oracle itself"
// (it is pinned only through the per-substep closed form P3, the linear closed
// form P6 and the 19-vs-55 O(dx^6) agreement).
//
// Not reentrant: fdo_set_forcing stores the forcing term in a file-static that every later fdo_rhs_* / fdo_rk3_step_*
// call of the PROCESS reads, so two threads (or two interleaved users) with different forcings would see each other's;
// oracle/oracle.py sets and clears it around each call (`with forcing(...)`).  Fine for a test oracle; do not call the
// fdo_* functions concurrently.
//
// Build: oracle/build.py  (g++ -O2 -ffp-contract=off -fopenmp, no -ffast-math).
// The only parallelism is one `#pragma omp parallel for` over k-planes; every cell
// is independent inside a sweep, so threading does not change any result bit.

#include <cmath>
#include <cstddef>
#include <cstdint>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------
// O2..O4  The three stencils, on values already gathered around a point.
// v[0..6] = f(-3), f(-2), f(-1), f(0), f(+1), f(+2), f(+3) along one axis.
// ---------------------------------------------------------------------------------

// Eq. 6:  d/dx f_i = (-f_{i-3} + 9 f_{i-2} - 45 f_{i-1} + 45 f_{i+1} - 9 f_{i+2} + f_{i+3}) / (60 dx),
// written as antisymmetric differences so that a constant gives exactly 0 (pin P5).
template <class T>
T stencil_d1(const T v[7], T dx) {
    return (T(45) * (v[4] - v[2]) - T(9) * (v[5] - v[1]) + (v[6] - v[0])) / (T(60) * dx);
}

// Eq. 7: d2/dx2 f_i = (2 f_{i-3} - 27 f_{i-2} + 270 f_{i-1} - 490 f_i + 270 f_{i+1} - 27 f_{i+2} + 2 f_{i+3}) / (180 dx^2).
// The paper prints 1/(180 dx): reading G1 of DESIGN.md takes dx^2 (dimensional analysis; pin P1 fails otherwise).
template <class T>
T stencil_d2(const T v[7], T dx) {
    return (T(-490) * v[3] + T(270) * (v[4] + v[2]) - T(27) * (v[5] + v[1]) + T(2) * (v[6] + v[0])) /
           (T(180) * dx * dx);
}

// Eq. 8, bidiagonal mixed derivative in the (a,b) plane:
//   [270 q1 - 27 q2 + 2 q3] / (720 dx dy),  q_m = f(+m,+m) - f(-m,+m) + f(-m,-m) - f(+m,-m).
// pp[m-1] = f(+m,+m), mp[m-1] = f(-m,+m), mm[m-1] = f(-m,-m), pm[m-1] = f(+m,-m); first sign is axis a.
template <class T>
T stencil_dmix(const T pp[3], const T mp[3], const T mm[3], const T pm[3], T dx) {
    T q1 = pp[0] - mp[0] + mm[0] - pm[0];
    T q2 = pp[1] - mp[1] + mm[1] - pm[1];
    T q3 = pp[2] - mp[2] + mm[2] - pm[2];
    return (T(270) * q1 - T(27) * q2 + T(2) * q3) / (T(720) * dx * dx);
}

// ---------------------------------------------------------------------------------
// O1  Periodic grid: dense arrays, index i + nx*(j + ny*k); neighbours by modular
// indexing (PAPER.md:95 grid; PAPER.md:187 periodic boundary conditions).
// ---------------------------------------------------------------------------------
struct Dims {
    int n[3];  // nx, ny, nz
};

inline int wrap(int i, int n) {
    int r = i % n;
    return r < 0 ? r + n : r;
}

template <class T>
inline T at(const T* f, const Dims& d, int i, int j, int k) {
    return f[(size_t)wrap(i, d.n[0]) + (size_t)d.n[0] * ((size_t)wrap(j, d.n[1]) + (size_t)d.n[1] * (size_t)wrap(k, d.n[2]))];
}

// Gather f(-3..3) along `axis` around (i,j,k).
template <class T>
inline void gather_line(const T* f, const Dims& d, int i, int j, int k, int axis, T v[7]) {
    for (int m = -3; m <= 3; ++m) {
        int o[3] = {0, 0, 0};
        o[axis] = m;
        v[m + 3] = at(f, d, i + o[0], j + o[1], k + o[2]);
    }
}

template <class T>
inline T d1_at(const T* f, const Dims& d, int i, int j, int k, int axis, T dx) {
    T v[7];
    gather_line(f, d, i, j, k, axis, v);
    return stencil_d1(v, dx);
}

template <class T>
inline T d2_at(const T* f, const Dims& d, int i, int j, int k, int axis, T dx) {
    T v[7];
    gather_line(f, d, i, j, k, axis, v);
    return stencil_d2(v, dx);
}

template <class T>
inline T dmix_at(const T* f, const Dims& d, int i, int j, int k, int a, int b, T dx) {
    T pp[3], mp[3], mm[3], pm[3];
    for (int m = 1; m <= 3; ++m) {
        int oa[3] = {0, 0, 0}, ob[3] = {0, 0, 0};
        oa[a] = m;
        ob[b] = m;
        pp[m - 1] = at(f, d, i + oa[0] + ob[0], j + oa[1] + ob[1], k + oa[2] + ob[2]);
        mp[m - 1] = at(f, d, i - oa[0] + ob[0], j - oa[1] + ob[1], k - oa[2] + ob[2]);
        mm[m - 1] = at(f, d, i - oa[0] - ob[0], j - oa[1] - ob[1], k - oa[2] - ob[2]);
        pm[m - 1] = at(f, d, i + oa[0] - ob[0], j + oa[1] - ob[1], k + oa[2] - ob[2]);
    }
    return stencil_dmix(pp, mp, mm, pm, dx);
}

// ---------------------------------------------------------------------------------
// O5..O7  Right-hand side of Eq. 1-3 at one cell.
//   F[0] = ln rho, F[1..3] = u_x, u_y, u_z   (G9: ln rho is stored).
//   path 55: Q_i = d_ii u_i + sum_{j!=i} d_ij u_j         (Eq. 7 + Eq. 8)
//   path 19: Q_i = D1_i(divA), divA = precomputed div u    (Eq. 14, Eq. 9, Alg. 3)
//   include_Q = false gives the "partial" RHS of Eq. 15 (no nu/3 grad div term).
// ---------------------------------------------------------------------------------
enum { PATH_55 = 0, PATH_19 = 1 };

template <class T>
struct CellDerivs {
    T g[3];     // g_i   = d_i ln rho
    T G[3][3];  // G_ij  = d_j u_i
    T L[3];     // L_i   = sum_j d_jj u_i   (Eq. 7 on every axis; G6: never composite)
    T div;      // G_00 + G_11 + G_22        (Eq. 14)
};

template <class T>
inline void cell_derivs(const T* const F[4], const Dims& d, int i, int j, int k, T dx, CellDerivs<T>& c) {
    for (int a = 0; a < 3; ++a) c.g[a] = d1_at(F[0], d, i, j, k, a, dx);
    for (int c_i = 0; c_i < 3; ++c_i)
        for (int a = 0; a < 3; ++a) c.G[c_i][a] = d1_at(F[1 + c_i], d, i, j, k, a, dx);
    for (int c_i = 0; c_i < 3; ++c_i) {
        T s = T(0);
        for (int a = 0; a < 3; ++a) s += d2_at(F[1 + c_i], d, i, j, k, a, dx);
        c.L[c_i] = s;
    }
    c.div = c.G[0][0] + c.G[1][1] + c.G[2][2];
}

// Q on the 55-point path: grad(div u)_i by direct second and bidiagonal mixed derivatives.
template <class T>
inline void grad_div_55(const T* const F[4], const Dims& d, int i, int j, int k, T dx, T Q[3]) {
    for (int a = 0; a < 3; ++a) {
        T s = d2_at(F[1 + a], d, i, j, k, a, dx);
        for (int b = 0; b < 3; ++b)
            if (b != a) s += dmix_at(F[1 + b], d, i, j, k, a, b, dx);
        Q[a] = s;
    }
}

// ---------------------------------------------------------------------------------
// O11  Forcing term of Eq. 2:  f(x) = Re{ N f_k exp(i k.x + i phi) }            (Eq. 24)
//   N = f0 cs sqrt(|k| cs / dt),   f_k = (k x e) / sqrt(|k|^2 - (k.e)^2)                            (Eq. 25)
// f_k is real, so f = N f_k cos(k.x + phi).  One (k, e, phi) is frozen over a step ("picked randomly at
// every timestep"); x = (i, j, k) dx, the origin is cell 0 shifted by `origin` cells (windowed runs).  f0 = 0: off,
// the paper's performance runs (G8).  Evaluated in double whatever T is.
// ---------------------------------------------------------------------------------
struct Forcing {
    double k[3] = {0, 0, 0}, e[3] = {0, 0, 0}, phi = 0, f0 = 0, dt = 1, origin[3] = {0, 0, 0};
};
static Forcing g_forcing;

inline void forcing_at(const Forcing& fo, double cs, double dx, int i, int j, int k, double f[3]) {
    const double* kv = fo.k;
    const double k2 = kv[0] * kv[0] + kv[1] * kv[1] + kv[2] * kv[2];
    const double ke = kv[0] * fo.e[0] + kv[1] * fo.e[1] + kv[2] * fo.e[2];
    const double N = fo.f0 * cs * std::sqrt(std::sqrt(k2) * cs / fo.dt);
    const double den = std::sqrt(k2 - ke * ke);
    const double cr[3] = {kv[1] * fo.e[2] - kv[2] * fo.e[1], kv[2] * fo.e[0] - kv[0] * fo.e[2], kv[0] * fo.e[1] - kv[1] * fo.e[0]};
    const double x[3] = {(i + fo.origin[0]) * dx, (j + fo.origin[1]) * dx, (k + fo.origin[2]) * dx};
    const double c = std::cos(kv[0] * x[0] + kv[1] * x[1] + kv[2] * x[2] + fo.phi);
    for (int a = 0; a < 3; ++a) f[a] = N * (cr[a] / den) * c;
}

// Eq. 1-3 assembled (O7).  R[0] continuity, R[1..3] momentum; the forcing f of Eq. 2 is added by the callers (O11).
template <class T>
inline void assemble_rhs(const T u[3], const CellDerivs<T>& c, const T Q[3], bool include_Q, T nu, T cs, T R[4]) {
    // Eq. 1:  d_t ln rho = -u . grad ln rho - div u
    R[0] = -(u[0] * c.g[0] + u[1] * c.g[1] + u[2] * c.g[2]) - c.div;
    for (int a = 0; a < 3; ++a) {
        // Eq. 3:  S_ab = 1/2 (d_b u_a + d_a u_b) - 1/3 delta_ab div u
        T Sg = T(0);
        for (int b = 0; b < 3; ++b) {
            T S = T(0.5) * (c.G[a][b] + c.G[b][a]);
            if (a == b) S -= c.div / T(3);
            Sg += S * c.g[b];
        }
        T adv = u[0] * c.G[a][0] + u[1] * c.G[a][1] + u[2] * c.G[a][2];
        T visc = c.L[a] + T(2) * Sg;
        if (include_Q) visc += Q[a] / T(3);
        // Eq. 2:  d_t u = -(u.grad)u - cs^2 grad ln rho + nu (lap u + 1/3 grad div u + 2 S.grad ln rho)
        R[1 + a] = -adv - cs * cs * c.g[a] + nu * visc;
    }
}

template <class T>
void fill_div(const T* const F[4], const Dims& d, T dx, T* divA) {
    const int nx = d.n[0], ny = d.n[1], nz = d.n[2];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                divA[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k)] =
                    d1_at(F[1], d, i, j, k, 0, dx) + d1_at(F[2], d, i, j, k, 1, dx) + d1_at(F[3], d, i, j, k, 2, dx);
}

// O10: full RHS (including nu Q / 3) of the current state, for fd_rhs parity.
template <class T>
void rhs_full(int path, const Dims& d, T dx, T nu, T cs, const T* const F[4], T* const R[4]) {
    const int nx = d.n[0], ny = d.n[1], nz = d.n[2];
    std::vector<T> divA;
    if (path == PATH_19) {
        divA.resize((size_t)nx * ny * nz);
        fill_div(F, d, dx, divA.data());
    }
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t p = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                CellDerivs<T> c;
                cell_derivs(F, d, i, j, k, dx, c);
                T Q[3];
                if (path == PATH_55)
                    grad_div_55(F, d, i, j, k, dx, Q);
                else
                    for (int a = 0; a < 3; ++a) Q[a] = d1_at(divA.data(), d, i, j, k, a, dx);
                T u[3] = {F[1][p], F[2][p], F[3][p]};
                T r[4];
                assemble_rhs(u, c, Q, true, nu, cs, r);
                if (g_forcing.f0 != 0) {  // + f (Eq. 2, Eq. 24)
                    double f[3];
                    forcing_at(g_forcing, (double)cs, (double)dx, i, j, k, f);
                    for (int a = 0; a < 3; ++a) r[1 + a] += T(f[a]);
                }
                for (int q = 0; q < 4; ++q) R[q][p] = r[q];
            }
}

// ---------------------------------------------------------------------------------
// O9  2N-storage RK3 coefficients.  The paper does not print them (PAPER.md:122-124,
// "[1, p. 9]"); reading G2 takes Williamson's (1980) set that the Pencil Code uses.
// alpha^(1) = 0.
// ---------------------------------------------------------------------------------
template <class T>
inline T rk_alpha(int s) {
    return s == 0 ? T(0) : (s == 1 ? T(-5) / T(9) : T(-153) / T(128));
}
template <class T>
inline T rk_beta(int s) {
    return s == 0 ? T(1) / T(3) : (s == 1 ? T(15) / T(16) : T(8) / T(15));
}

// Eq. 10 on one value:  w <- alpha w + dt * rhs ;  u <- u + beta w.
// At s = 1 alpha = 0 and w is NOT read (G4: stale/NaN w must not leak in).
template <class T>
inline void rk_update(int s, T dt, T rhs, T f_old, T& w, T& f_new) {
    T wn = (s == 0) ? dt * rhs : rk_alpha<T>(s) * w + dt * rhs;
    w = wn;
    f_new = f_old + rk_beta<T>(s) * wn;
}

// O8 (55): Alg. 2. Separate read/write arrays, swap after each substep.
// O8 (19): Alg. 3 reconstructed from Eq. 14-18 and App. A (G5):
//   sweep 1: div u for all cells; partial w and partial F_out without the nu/3 grad div term (Eq. 15-16);
//   sweep 2: w_i += dt nu/3 D1_i(div) (Eq. 17);  F_out,i += beta dt nu/3 D1_i(div) (Eq. 18), i = 1..3.
template <class T>
void rk3_steps(int path, const Dims& d, T dx, T nu, T cs, T dt, int nsteps, T* const Fio[4], T* const W[4]) {
    const int nx = d.n[0], ny = d.n[1], nz = d.n[2];
    const size_t N = (size_t)nx * ny * nz;
    std::vector<T> outbuf(4 * N), divA;
    if (path == PATH_19) divA.resize(N);
    T* cur[4] = {Fio[0], Fio[1], Fio[2], Fio[3]};
    T* out[4] = {outbuf.data(), outbuf.data() + N, outbuf.data() + 2 * N, outbuf.data() + 3 * N};

    for (int step = 0; step < nsteps; ++step) {
        for (int s = 0; s < 3; ++s) {
            const T* const Fc[4] = {cur[0], cur[1], cur[2], cur[3]};
            if (path == PATH_19) fill_div(Fc, d, dx, divA.data());
#pragma omp parallel for schedule(static)
            for (int k = 0; k < nz; ++k)
                for (int j = 0; j < ny; ++j)
                    for (int i = 0; i < nx; ++i) {
                        size_t p = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                        CellDerivs<T> c;
                        cell_derivs(Fc, d, i, j, k, dx, c);
                        T Q[3] = {T(0), T(0), T(0)};
                        if (path == PATH_55) grad_div_55(Fc, d, i, j, k, dx, Q);
                        T u[3] = {Fc[1][p], Fc[2][p], Fc[3][p]};
                        T r[4];
                        assemble_rhs(u, c, Q, path == PATH_55, nu, cs, r);
                        if (g_forcing.f0 != 0) {  // + f (Eq. 2, Eq. 24): the same frozen f on all three substeps
                            double f[3];
                            forcing_at(g_forcing, (double)cs, (double)dx, i, j, k, f);
                            for (int a = 0; a < 3; ++a) r[1 + a] += T(f[a]);
                        }
                        for (int q = 0; q < 4; ++q) rk_update(s, dt, r[q], Fc[q][p], W[q][p], out[q][p]);
                    }
            if (path == PATH_19) {
#pragma omp parallel for schedule(static)
                for (int k = 0; k < nz; ++k)
                    for (int j = 0; j < ny; ++j)
                        for (int i = 0; i < nx; ++i) {
                            size_t p = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                            for (int a = 0; a < 3; ++a) {
                                T gd = d1_at(divA.data(), d, i, j, k, a, dx);
                                T add = dt * (nu / T(3)) * gd;
                                W[1 + a][p] = W[1 + a][p] + add;                             // Eq. 17
                                out[1 + a][p] = out[1 + a][p] + rk_beta<T>(s) * add;         // Eq. 18
                            }
                        }
            }
            for (int q = 0; q < 4; ++q) {  // "swapped efficiently using pointers"
                T* t = cur[q];
                cur[q] = out[q];
                out[q] = t;
            }
        }
    }
    if (cur[0] != Fio[0])
        for (int q = 0; q < 4; ++q)
            for (size_t p = 0; p < N; ++p) Fio[q][p] = cur[q][p];
}

// The same Eq. 10 update applied to the scalar test ODE y' = lambda y (complex lambda
// as a real 2-vector).  Uses rk_update, i.e. the very coefficients and order of the
// PDE integrator, so pin P7 (closed form 1 + z + z^2/2 + z^3/6) pins O9.
void rk3_linear(double lre, double lim, double dt, int nsteps, double y[2]) {
    double w[2] = {0.0, 0.0};
    for (int step = 0; step < nsteps; ++step)
        for (int s = 0; s < 3; ++s) {
            double r[2] = {lre * y[0] - lim * y[1], lre * y[1] + lim * y[0]};
            double yn[2];
            rk_update<double>(s, dt, r[0], y[0], w[0], yn[0]);
            rk_update<double>(s, dt, r[1], y[1], w[1], yn[1]);
            y[0] = yn[0];
            y[1] = yn[1];
        }
}

template <class T>
void deriv_field(int kind, int a, int b, const Dims& d, T dx, const T* f, T* out) {
    const int nx = d.n[0], ny = d.n[1], nz = d.n[2];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t p = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                out[p] = kind == 1 ? d1_at(f, d, i, j, k, a, dx)
                                   : (kind == 2 ? d2_at(f, d, i, j, k, a, dx) : dmix_at(f, d, i, j, k, a, b, dx));
            }
}

bool bad_dims(int nx, int ny, int nz) { return nx < 1 || ny < 1 || nz < 1; }

}  // namespace

// ---------------------------------------------------------------------------------
// C entry points (loaded with ctypes by oracle/oracle.py).  All arrays are dense,
// x fastest: idx = i + nx*(j + ny*k).  Return 0 on success, 1 on bad arguments.
// ---------------------------------------------------------------------------------
extern "C" {

int fdo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void fdo_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

// Forcing of every later fdo_rhs_* / fdo_rk3_step_* call (O11); f0 = 0 switches it off.  dt is the step size N is
// formed with (Eq. 25); origin = cell offset of array index 0 (windowed runs).  1: bad arguments (k parallel to e, dt <= 0).
int fdo_set_forcing(const double k[3], const double e[3], double phi, double f0, double dt, const double origin[3]) {
    Forcing fo;
    if (f0 != 0) {
        const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2], ke = k[0] * e[0] + k[1] * e[1] + k[2] * e[2];
        if (!(dt > 0) || !(k2 - ke * ke > 0)) return 1;
        for (int a = 0; a < 3; ++a) {
            fo.k[a] = k[a];
            fo.e[a] = e[a];
            fo.origin[a] = origin ? origin[a] : 0.0;
        }
        fo.phi = phi;
        fo.f0 = f0;
        fo.dt = dt;
    }
    g_forcing = fo;
    return 0;
}

// Stencils on caller-gathered values (non-periodic use: polynomial exactness, pin P1).
double fdo_stencil_d1(const double v[7], double dx) { return stencil_d1<double>(v, dx); }
double fdo_stencil_d2(const double v[7], double dx) { return stencil_d2<double>(v, dx); }
double fdo_stencil_dmix(const double pp[3], const double mp[3], const double mm[3], const double pm[3], double dx) {
    return stencil_dmix<double>(pp, mp, mm, pm, dx);
}

// One derivative of one periodic field. kind: 1 = Eq. 6 along a; 2 = Eq. 7 along a; 3 = Eq. 8 in plane (a,b).
int fdo_deriv_f64(int kind, int a, int b, int nx, int ny, int nz, double dx, const double* f, double* out) {
    if (bad_dims(nx, ny, nz) || kind < 1 || kind > 3 || a < 0 || a > 2 || (kind == 3 && (b < 0 || b > 2 || b == a))) return 1;
    Dims d{{nx, ny, nz}};
    deriv_field<double>(kind, a, b, d, dx, f, out);
    return 0;
}

int fdo_rhs_f64(int path, int nx, int ny, int nz, double dx, double nu, double cs, const double* lnrho, const double* ux,
                const double* uy, const double* uz, double* r0, double* r1, double* r2, double* r3) {
    if (bad_dims(nx, ny, nz) || (path != PATH_55 && path != PATH_19)) return 1;
    Dims d{{nx, ny, nz}};
    const double* F[4] = {lnrho, ux, uy, uz};
    double* R[4] = {r0, r1, r2, r3};
    rhs_full<double>(path, d, dx, nu, cs, F, R);
    return 0;
}

int fdo_rhs_f32(int path, int nx, int ny, int nz, double dx, double nu, double cs, const float* lnrho, const float* ux,
                const float* uy, const float* uz, float* r0, float* r1, float* r2, float* r3) {
    if (bad_dims(nx, ny, nz) || (path != PATH_55 && path != PATH_19)) return 1;
    Dims d{{nx, ny, nz}};
    const float* F[4] = {lnrho, ux, uy, uz};
    float* R[4] = {r0, r1, r2, r3};
    rhs_full<float>(path, d, (float)dx, (float)nu, (float)cs, F, R);
    return 0;
}

// nsteps full RK3 steps in place. w0..w3 are the 2N intermediate arrays (in/out; never read at s = 1).
int fdo_rk3_step_f64(int path, int nx, int ny, int nz, double dx, double nu, double cs, double dt, int nsteps,
                     double* lnrho, double* ux, double* uy, double* uz, double* w0, double* w1, double* w2, double* w3) {
    if (bad_dims(nx, ny, nz) || (path != PATH_55 && path != PATH_19) || nsteps < 0) return 1;
    Dims d{{nx, ny, nz}};
    double* F[4] = {lnrho, ux, uy, uz};
    double* W[4] = {w0, w1, w2, w3};
    rk3_steps<double>(path, d, dx, nu, cs, dt, nsteps, F, W);
    return 0;
}

int fdo_rk3_step_f32(int path, int nx, int ny, int nz, double dx, double nu, double cs, double dt, int nsteps,
                     float* lnrho, float* ux, float* uy, float* uz, float* w0, float* w1, float* w2, float* w3) {
    if (bad_dims(nx, ny, nz) || (path != PATH_55 && path != PATH_19) || nsteps < 0) return 1;
    Dims d{{nx, ny, nz}};
    float* F[4] = {lnrho, ux, uy, uz};
    float* W[4] = {w0, w1, w2, w3};
    rk3_steps<float>(path, d, (float)dx, (float)nu, (float)cs, (float)dt, nsteps, F, W);
    return 0;
}

// y' = lambda y integrated with the same Eq. 10 update and coefficients (pin P7).
int fdo_rk3_linear(double lambda_re, double lambda_im, double dt, int nsteps, double* y_re, double* y_im) {
    if (nsteps < 0 || !y_re || !y_im) return 1;
    double y[2] = {*y_re, *y_im};
    rk3_linear(lambda_re, lambda_im, dt, nsteps, y);
    *y_re = y[0];
    *y_im = y[1];
    return 0;
}

}  // extern "C"
