"""Pins of the CPU oracle (oracle/fd_oracle.cpp) against things OTHER than itself:
what the paper prints, closed forms, the continuum equations, invariants and brute force.
DESIGN.md "Oracle pins" lists them as P0..P12; a plausible mistake anywhere in the oracle
(dropped term, wrong sign/index, transposed axis) fails at least one of them.

No GPU, no CUDA library: only oracle/ and the input generators are imported.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_1707_08900_b200 import inputs as I

P55, P19 = O.PATH_55, O.PATH_19
TWO_PI = 2.0 * math.pi


# ------------------------------------------------------------------------------- helpers
def s1(a):  # Fourier symbol of Eq. 6 (P2): D1 cos(theta) = -(s1/dx) sin(theta)
    return (45 * np.sin(a) - 9 * np.sin(2 * a) + np.sin(3 * a)) / 30


def s2(a):  # Eq. 7: D2 cos(theta) = -(s2/dx^2) cos(theta)
    return (490 - 540 * np.cos(a) + 54 * np.cos(2 * a) - 4 * np.cos(3 * a)) / 180


def sm(a, b):  # Eq. 8: Dmix cos(theta) = -(sm/dx^2) cos(theta)
    return (270 * np.sin(a) * np.sin(b) - 27 * np.sin(2 * a) * np.sin(2 * b) + 2 * np.sin(3 * a) * np.sin(3 * b)) / 180


def grid_phase(shape_xyz, kvec, phi):
    """theta(i,j,k) = 2 pi (kx i/nx + ky j/ny + kz k/nz) + phi as an (nz,ny,nx) array."""
    nx, ny, nz = shape_xyz
    i = np.arange(nx)[None, None, :]
    j = np.arange(ny)[None, :, None]
    k = np.arange(nz)[:, None, None]
    return TWO_PI * (kvec[0] * i / nx + kvec[1] * j / ny + kvec[2] * k / nz) + phi


def relinf(A, B):
    """max over components of max|A-B| / max|B| (reading G14)."""
    worst = 0.0
    for a, b in zip(A, B):
        den = np.abs(b).max()
        err = np.abs(a - b).max()
        worst = max(worst, err / den if den > 0 else err)
    return worst


def read_golden_coeffs(golden_dir):
    out = {}
    with open(os.path.join(golden_dir, "stencil_coefficients.txt")) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            left, right = line.split(":")
            toks = left.split()
            out[toks[0]] = (int(toks[1]), [int(t) for t in toks[2:]], [int(t) for t in right.split()])
    return out


# --------------------------------------------------- P0: the coefficients the paper prints
def test_p0_impulse_response_reproduces_printed_coefficients(golden_dir):
    g = read_golden_coeffs(golden_dir)
    dx = 0.37
    den, offs, cs = g["eq6"]
    for o, c in zip(offs, cs):
        v = np.zeros(7)
        v[o + 3] = 1.0
        assert O.stencil_d1(v, dx) == pytest.approx(c / (den * dx), rel=1e-15, abs=1e-300)
    den, offs, cs = g["eq7"]
    for o, c in zip(offs, cs):
        v = np.zeros(7)
        v[o + 3] = 1.0
        assert O.stencil_d2(v, dx) == pytest.approx(c / (den * dx * dx), rel=1e-15)
    den, ms, cs = g["eq8"]
    signs = {"pp": +1, "mp": -1, "mm": +1, "pm": -1}  # Eq. 8 as printed
    for m, c in zip(ms, cs):
        for name, sg in signs.items():
            arrs = {n: np.zeros(3) for n in signs}
            arrs[name][m - 1] = 1.0
            got = O.stencil_dmix(arrs["pp"], arrs["mp"], arrs["mm"], arrs["pm"], dx)
            assert got == pytest.approx(sg * c / (den * dx * dx), rel=1e-15)


def test_p0_periodic_impulse_places_taps_on_the_right_axis_and_side(golden_dir):
    """A unit impulse on a non-cubic periodic grid: the response of the field operators must be the printed
    coefficients, mirrored (out[p] uses f[p+m]), on the requested axis only, with wrap-around."""
    g = read_golden_coeffs(golden_dir)
    nx, ny, nz, dx = 8, 9, 10, 0.5
    f = np.zeros((nz, ny, nx))
    p = (1, 7, 2)  # (k, j, i) close to the seams
    f[p] = 1.0
    for a in range(3):
        for kind, key, scale in ((1, "eq6", dx), (2, "eq7", dx * dx)):
            den, offs, cs = g[key]
            out = O.deriv(f, kind, a, dx=dx)
            exp = np.zeros_like(f)
            for o, c in zip(offs, cs):
                q = list(p)
                q[2 - a] = (q[2 - a] - o) % f.shape[2 - a]  # out[q] sees the impulse at q+o
                exp[tuple(q)] += c / (den * scale)
            np.testing.assert_allclose(out, exp, rtol=1e-15, atol=1e-300)
    den, ms, cs = g["eq8"]
    for a in range(3):
        for b in range(3):
            if a == b:
                continue
            out = O.deriv(f, 3, a, b, dx=dx)
            exp = np.zeros_like(f)
            for m, c in zip(ms, cs):
                for sa, sb, sg in ((1, 1, 1), (-1, 1, -1), (-1, -1, 1), (1, -1, -1)):
                    q = list(p)
                    q[2 - a] = (q[2 - a] - sa * m) % f.shape[2 - a]
                    q[2 - b] = (q[2 - b] - sb * m) % f.shape[2 - b]
                    exp[tuple(q)] += sg * c / (den * dx * dx)
            np.testing.assert_allclose(out, exp, rtol=1e-15, atol=1e-300)


# ------------------------------------------------------------ P1: polynomial exactness
def test_p1_d1_d2_exact_on_polynomials_up_to_degree_6():
    h, x0 = 0.25, 0.3
    xs = x0 + h * np.arange(-3, 4)
    for p in range(0, 7):
        d1_exact = p * x0 ** (p - 1) if p > 0 else 0.0
        d2_exact = p * (p - 1) * x0 ** (p - 2) if p > 1 else 0.0
        assert O.stencil_d1(xs ** p, h) == pytest.approx(d1_exact, abs=2e-13)
        assert O.stencil_d2(xs ** p, h) == pytest.approx(d2_exact, abs=2e-12)
    # first failures have the textbook leading error D - exact = +h^6 f^(7)/140 and +h^6 f^(8)/560
    # (from the symbols: s1(a)/a = 1 - a^6/140 + ..., s2(a)/a^2 = 1 - a^6/560 + ...)
    assert O.stencil_d1(xs ** 7, h) - 7 * x0 ** 6 == pytest.approx(math.factorial(7) / 140 * h ** 6, rel=1e-6)
    assert O.stencil_d2(xs ** 7, h) == pytest.approx(42 * x0 ** 5, abs=2e-12)  # D2 is exact to degree 7
    assert O.stencil_d2(xs ** 8, h) - 56 * x0 ** 6 == pytest.approx(math.factorial(8) / 560 * h ** 6, rel=1e-6)


def test_p1_eq7_needs_dx_squared_reading_g1():
    # x^2 has second derivative 2 for every dx only with the 1/(180 dx^2) prefactor
    for h in (0.1, 0.5, 2.0):
        xs = h * np.arange(-3, 4)
        assert O.stencil_d2(xs ** 2, h) == pytest.approx(2.0, rel=1e-13)


def test_p1_dmix_exact_on_bivariate_monomials():
    h, x0, y0 = 0.25, 0.3, -0.2

    def mix(fn):
        m = np.arange(1, 4) * h
        return O.stencil_dmix(fn(x0 + m, y0 + m), fn(x0 - m, y0 + m), fn(x0 - m, y0 - m), fn(x0 + m, y0 - m), h)

    for a in range(0, 8):
        for b in range(0, 8 - a):
            exact = (a * x0 ** (a - 1) if a else 0.0) * (b * y0 ** (b - 1) if b else 0.0)
            assert mix(lambda x, y: x ** a * y ** b) == pytest.approx(exact, abs=5e-12), (a, b)
    for a, b in ((1, 7), (3, 5), (5, 3), (7, 1)):  # first monomials it must NOT be exact on
        exact = a * x0 ** (a - 1) * b * y0 ** (b - 1)
        assert abs(mix(lambda x, y: x ** a * y ** b) - exact) > 1e-6, (a, b)


# --------------------------------------------------------------- P2: Fourier symbols
@pytest.mark.parametrize("shape,kvec", [((12, 16, 20), (2, -3, 1)), ((16, 12, 8), (-1, 2, 3))])
def test_p2_fourier_symbols(shape, kvec):
    nx, ny, nz = shape
    dx = 0.4
    th = grid_phase(shape, kvec, 0.7)
    f = np.cos(th)
    ang = [TWO_PI * kvec[0] / nx, TWO_PI * kvec[1] / ny, TWO_PI * kvec[2] / nz]
    for a in range(3):
        np.testing.assert_allclose(O.deriv(f, 1, a, dx=dx), -s1(ang[a]) / dx * np.sin(th), atol=1e-13)
        np.testing.assert_allclose(O.deriv(f, 2, a, dx=dx), -s2(ang[a]) / dx ** 2 * np.cos(th), atol=1e-12)
        for b in range(3):
            if b != a:
                np.testing.assert_allclose(O.deriv(f, 3, a, b, dx=dx), -sm(ang[a], ang[b]) / dx ** 2 * np.cos(th),
                                           atol=1e-12)


# ------------------------------------------- P3: whole nonlinear RHS from symbols only
def _closed_form_rhs(shape, dx, nu, cs, kv, ph, amp, path):
    """RHS of Eq. 1-3 for fields that are sums of cosines, every discrete derivative taken from the
    Fourier symbols (no neighbour access, no stencil code).  kv (4,M,3), ph (4,M), amp (4,M)."""
    nx, ny, nz = shape
    nn = (nx, ny, nz)
    val = [0.0] * 4
    d1 = [[0.0] * 3 for _ in range(4)]
    d2 = [[0.0] * 3 for _ in range(4)]
    dm = [[[0.0] * 3 for _ in range(3)] for _ in range(4)]
    d11 = [[[0.0] * 3 for _ in range(3)] for _ in range(4)]  # D1_a D1_b (composite, Eq. 9)
    for q in range(4):
        for m in range(kv.shape[1]):
            th = grid_phase(shape, kv[q, m], ph[q, m])
            c, s = amp[q, m] * np.cos(th), amp[q, m] * np.sin(th)
            ang = [TWO_PI * kv[q, m, a] / nn[a] for a in range(3)]
            val[q] = val[q] + c
            for a in range(3):
                d1[q][a] = d1[q][a] - s1(ang[a]) / dx * s
                d2[q][a] = d2[q][a] - s2(ang[a]) / dx ** 2 * c
                for b in range(3):
                    dm[q][a][b] = dm[q][a][b] - sm(ang[a], ang[b]) / dx ** 2 * c
                    d11[q][a][b] = d11[q][a][b] - s1(ang[a]) * s1(ang[b]) / dx ** 2 * c
    u = val[1:]
    gl = d1[0]
    gu = d1[1:]
    div = gu[0][0] + gu[1][1] + gu[2][2]
    R = [-(u[0] * gl[0] + u[1] * gl[1] + u[2] * gl[2]) - div]
    for i in range(3):
        lap = d2[1 + i][0] + d2[1 + i][1] + d2[1 + i][2]
        if path == P55:
            gd = sum(d2[1 + j][i] if j == i else dm[1 + j][i][j] for j in range(3))
        else:
            gd = sum(d11[1 + j][i][j] for j in range(3))
        Sg = sum((0.5 * (gu[i][j] + gu[j][i]) - (div / 3 if i == j else 0.0)) * gl[j] for j in range(3))
        adv = sum(u[j] * gu[i][j] for j in range(3))
        R.append(-adv - cs ** 2 * gl[i] + nu * (lap + gd / 3 + 2 * Sg))
    return np.stack(R)


@pytest.mark.parametrize("path", [P55, P19])
def test_p3_rhs_equals_symbol_closed_form(path):
    shape = (16, 12, 20)
    rng = np.random.default_rng(7)
    M = 5
    kv = rng.integers(-3, 4, (4, M, 3))
    ph = rng.uniform(0, TWO_PI, (4, M))
    amp = rng.uniform(0.05, 0.3, (4, M))
    dx, nu, cs = 0.37, 0.08, 1.3
    F = np.stack([sum(amp[q, m] * np.cos(grid_phase(shape, kv[q, m], ph[q, m])) for m in range(M)) for q in range(4)])
    ref = _closed_form_rhs(shape, dx, nu, cs, kv, ph, amp, path)
    got = O.rhs(F, dx, nu, cs, path)
    assert relinf(got, ref) < 5e-13


def test_p3_config_c1_rhs_equals_symbol_closed_form():
    cfg = I.CONFIGS["C1"]
    kv, ph = I.draw_modes(cfg.seed, 8, cfg.kmax)
    F = I.make_state(cfg)
    amp = np.full((4, 8), cfg.amp / math.sqrt(8))
    kzyx = kv  # (kx, ky, kz) order already
    for path in (P55, P19):
        ref = _closed_form_rhs((cfg.n,) * 3, cfg.dx, cfg.nu, cfg.cs, kzyx, ph, amp, path)
        assert relinf(O.rhs(F, cfg.dx, cfg.nu, cfg.cs, path), ref) < 5e-13


# -------------------------------- P4: sixth-order convergence on analytic sinusoids
def test_p4_sixth_order_convergence_of_all_three_stencils():
    errs = {1: [], 2: [], 3: []}
    for n in (16, 32, 64):
        dx = TWO_PI / n
        g = np.arange(n) * dx
        Z, Y, X = np.meshgrid(g, g, g, indexing="ij")
        f = np.sin(2 * X + 0.3) * np.cos(Y - 0.1) + np.sin(X + 2 * Y + Z)
        fx = 2 * np.cos(2 * X + 0.3) * np.cos(Y - 0.1) + np.cos(X + 2 * Y + Z)
        fxx = -4 * np.sin(2 * X + 0.3) * np.cos(Y - 0.1) - np.sin(X + 2 * Y + Z)
        fxy = -2 * np.cos(2 * X + 0.3) * np.sin(Y - 0.1) - 2 * np.sin(X + 2 * Y + Z)
        errs[1].append(np.abs(O.deriv(f, 1, 0, dx=dx) - fx).max())
        errs[2].append(np.abs(O.deriv(f, 2, 0, dx=dx) - fxx).max())
        errs[3].append(np.abs(O.deriv(f, 3, 0, 1, dx=dx) - fxy).max())
    for kind, e in errs.items():
        for coarse, fine in zip(e[:-1], e[1:]):
            order = math.log2(coarse / fine)
            assert 5.5 < order < 6.5, (kind, e)


# ------------------------------- P5: zero RHS on a uniform state at rest (exactly 0.0)
@pytest.mark.parametrize("path", [P55, P19])
def test_p5_uniform_state_at_rest_has_exactly_zero_rhs(path):
    F = np.zeros((4, 8, 9, 10))
    F[0] = 0.731
    R = O.rhs(F, 0.1, 5e-3, 1.0, path)
    assert np.all(R == 0.0)
    out = O.rk3_step(F, 0.1, 5e-3, 1.0, 0.01, 2, path)
    assert np.array_equal(out, F)


# --------------------------------- P6: fully discrete shear-mode closed form (Eq. 22 twin)
@pytest.mark.parametrize("path", [P55, P19])
@pytest.mark.parametrize("wave_axis,vel_comp", [(0, 1), (0, 2), (1, 0), (1, 2), (2, 0), (2, 1)])
def test_p6_shear_mode_decay_matches_discrete_closed_form(path, wave_axis, vel_comp):
    n, k, u0, nu, cs, nsteps = 32, 5, 1e-2, 5e-3, 1.0, 10
    dx = TWO_PI / n
    dt = 0.1 * dx / cs
    g = np.arange(n) * dx
    coords = np.meshgrid(g, g, g, indexing="ij")  # Z, Y, X
    xi = coords[2 - wave_axis]
    F = np.zeros((4, n, n, n))
    F[1 + vel_comp] = u0 * np.sin(k * xi)
    z = -nu * dt * s2(k * dx) / dx ** 2
    G = 1 + z + z * z / 2 + z ** 3 / 6
    out = O.rk3_step(F, dx, nu, cs, dt, nsteps, path)
    np.testing.assert_allclose(out[1 + vel_comp], G ** nsteps * u0 * np.sin(k * xi), atol=2e-15 * 1e2 * u0)
    for q in range(4):
        if q != 1 + vel_comp:
            assert np.abs(out[q]).max() < 1e-16
    # and the discrete decay factor tends to the paper's continuum law, Eq. 22
    assert G ** nsteps == pytest.approx(math.exp(-nu * k * k * nsteps * dt), rel=1e-4)


# ------------------------- P6b: longitudinal (sound) mode pins cs^2, div u and the 4/3 nu
@pytest.mark.parametrize("path", [P55, P19])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p6b_longitudinal_mode_linear_rhs(path, axis):
    """ln rho = e cos(k x), u_axis = e sin(k x + 0.4) with e -> 0: quadratic terms are O(e^2) and the RHS is
    R0 = -D1 u;  R_axis = -cs^2 D1 lnrho + nu (D2 u + Q/3), Q = D2 u (55) or D1 D1 u (19): the 4/3 nu law."""
    n, k, e, nu, cs = 24, 3, 1e-9, 0.05, 1.7
    dx = TWO_PI / n
    g = np.arange(n) * dx
    xi = np.meshgrid(g, g, g, indexing="ij")[2 - axis]
    a = k * dx
    F = np.zeros((4, n, n, n))
    F[0] = e * np.cos(k * xi)
    F[1 + axis] = e * np.sin(k * xi + 0.4)
    R = O.rhs(F, dx, nu, cs, path)
    d1u = e * s1(a) / dx * np.cos(k * xi + 0.4)
    d2u = -e * s2(a) / dx ** 2 * np.sin(k * xi + 0.4)
    q = d2u if path == P55 else -e * s1(a) ** 2 / dx ** 2 * np.sin(k * xi + 0.4)
    np.testing.assert_allclose(R[0], -d1u, atol=1e-6 * e)
    np.testing.assert_allclose(R[1 + axis], cs ** 2 * e * s1(a) / dx * np.sin(k * xi) + nu * (d2u + q / 3), atol=1e-6 * e)
    for c in range(3):
        if c != axis:
            assert np.abs(R[1 + c]).max() < 1e-6 * e


# ------------- P6c: sound-wave eigen-system through full RK3 steps (pins Eq. 17-18 with their beta)
@pytest.mark.parametrize("path", [P55, P19])
def test_p6c_longitudinal_mode_multi_step_matrix_closed_form(path):
    """In the linear regime (amplitude e -> 0) the pair (ln rho, u_x) = Re[(a, b) e^{ikx}] obeys y' = A y with
    A = [[0, -i s1/dx], [-i cs^2 s1/dx, -nu (s2 + q/3)/dx^2]], q = s2 (55-pt) or s1^2 (19-pt), and n RK3 steps
    give P(dt A)^n y0, P(z) = 1 + z + z^2/2 + z^3/6 — for the 19-pt path only if both sweeps (Eq. 15-18) add up."""
    n, k, e, nu, cs, nsteps = 24, 2, 1e-9, 0.3, 1.1, 4
    dx = TWO_PI / n
    dt = 0.1 * dx / cs
    g = np.arange(n) * dx
    X = np.meshgrid(g, g, g, indexing="ij")[2]
    a0, b0 = e * (1.0 + 0.0j), e * (0.3 - 0.8j)
    F = np.zeros((4, n, n, n))
    F[0] = (a0 * np.exp(1j * k * X)).real
    F[1] = (b0 * np.exp(1j * k * X)).real
    a = k * dx
    q = s2(a) if path == P55 else s1(a) ** 2
    A = np.array([[0.0, -1j * s1(a) / dx], [-1j * cs ** 2 * s1(a) / dx, -nu * (s2(a) + q / 3) / dx ** 2]])
    Zm = dt * A
    Pm = np.eye(2) + Zm + Zm @ Zm / 2 + Zm @ Zm @ Zm / 6
    y = np.linalg.matrix_power(Pm, nsteps) @ np.array([a0, b0])
    out = O.rk3_step(F, dx, nu, cs, dt, nsteps, path)
    np.testing.assert_allclose(out[0], (y[0] * np.exp(1j * k * X)).real, atol=1e-7 * e)
    np.testing.assert_allclose(out[1], (y[1] * np.exp(1j * k * X)).real, atol=1e-7 * e)
    assert abs(y[1] - b0) > 1e-3 * e  # the test moves the state by much more than its tolerance


# ------------------------------------------------------------- P7: RK3 on y' = lambda y
def test_p7_rk3_linear_closed_form_and_third_order():
    for lam in (-1.3, -0.4 + 2.1j, 0.9j):
        for dt in (0.1, 0.05):
            z = lam * dt
            got = O.rk3_linear(lam, dt, 1, 0.7 - 0.2j)
            assert got == pytest.approx((1 + z + z * z / 2 + z ** 3 / 6) * (0.7 - 0.2j), rel=1e-14)
    # global third order: error after T = 1 shrinks 8x per halving of dt; local error -> z^4/24
    errs = [abs(O.rk3_linear(-1.0, 1.0 / n, n, 1.0) - math.exp(-1.0)) for n in (20, 40, 80)]
    assert 7.0 < errs[0] / errs[1] < 9.0 and 7.0 < errs[1] / errs[2] < 9.0
    z = -0.01
    assert (O.rk3_linear(-1.0, 0.01, 1, 1.0) - math.exp(z)).real == pytest.approx(-z ** 4 / 24, rel=0.02)


def test_p7_rk3_multi_step_is_repeated_single_steps():
    cfg = I.CONFIGS["C1"]
    F = I.make_state(cfg, n_override=16)
    dx = TWO_PI / 16
    a = O.rk3_step(F, dx, cfg.nu, cfg.cs, 0.1 * dx, 3, P55)
    b = F
    for _ in range(3):
        b = O.rk3_step(b, dx, cfg.nu, cfg.cs, 0.1 * dx, 1, P55)
    assert np.array_equal(a, b)


# --------------------------------------- P8: exact periodic-shift equivariance (bitwise)
@pytest.mark.parametrize("path", [P55, P19])
def test_p8_shift_equivariance_is_bitwise(path):
    rng = np.random.default_rng(3)
    F = 0.1 * rng.standard_normal((4, 10, 12, 14))
    sh = (3, 5, 9)
    a = O.rk3_step(F, 0.3, 0.02, 1.0, 0.01, 1, path)
    b = O.rk3_step(np.roll(F, sh, (1, 2, 3)), 0.3, 0.02, 1.0, 0.01, 1, path)
    assert np.array_equal(np.roll(a, sh, (1, 2, 3)), b)


# ---------------------------- P9: axis-permutation equivariance (the symmetry of PAPER.md:414)
@pytest.mark.parametrize("path", [P55, P19])
@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (0, 2, 1), (1, 2, 0)])
def test_p9_axis_permutation_equivariance(path, perm):
    """Relabel the axes: new axis a is old axis perm[a] (axes numbered x=0,y=1,z=2), velocity components follow."""
    rng = np.random.default_rng(11)
    n = 12
    F = 0.1 * rng.standard_normal((4, n, n, n))
    R = O.rhs(F, 0.3, 0.04, 1.2, path)

    def relabel(A):
        # numpy dims of a component are (z,y,x) = oracle axes (2,1,0); new numpy dim (2-a) <- old numpy dim (2-perm[a])
        order = [0, 0, 0]
        for a in range(3):
            order[2 - a] = 2 - perm[a]
        comps = [A[0]] + [A[1 + perm[a]] for a in range(3)]
        return np.stack([np.transpose(c, order) for c in comps])

    Rp = O.rhs(relabel(F), 0.3, 0.04, 1.2, path)
    assert relinf(Rp, relabel(R)) < 1e-13


# ---------------------------------- P10: brute force with dense operator matrices (tiny grid)
@pytest.mark.parametrize("path", [P55, P19])
def test_p10_dense_operator_brute_force(path, golden_dir):
    g = read_golden_coeffs(golden_dir)
    nx, ny, nz = 8, 7, 9  # radius 3 wraps almost the whole 7-point axis
    dx, nu, cs = 0.45, 0.03, 0.9
    nn = (nx, ny, nz)

    def shift(n, m):  # (S f)[p] = f[(p+m) mod n]
        S = np.zeros((n, n))
        for p in range(n):
            S[p, (p + m) % n] = 1.0
        return S

    def on_axis(mats):  # mats[a] acts on axis a; flat index i + nx*(j + ny*k) -> kron(z, y, x)
        return np.kron(mats[2], np.kron(mats[1], mats[0]))

    eye = [np.eye(n) for n in nn]

    def op1(a, coeffs, den):
        M = sum(c * shift(nn[a], o) for o, c in zip(*coeffs)) / den
        mats = list(eye)
        mats[a] = M
        return on_axis(mats)

    D1 = [op1(a, (g["eq6"][1], g["eq6"][2]), g["eq6"][0] * dx) for a in range(3)]
    D2 = [op1(a, (g["eq7"][1], g["eq7"][2]), g["eq7"][0] * dx * dx) for a in range(3)]

    def opmix(a, b):
        tot = 0.0
        for m, c in zip(g["eq8"][1], g["eq8"][2]):
            mats_a = list(eye)
            mats_a[a] = shift(nn[a], m) - shift(nn[a], -m)
            mats_b = list(eye)
            mats_b[b] = shift(nn[b], m) - shift(nn[b], -m)
            tot = tot + c * on_axis(mats_a) @ on_axis(mats_b)
        return tot / (g["eq8"][0] * dx * dx)

    rng = np.random.default_rng(5)
    F = 0.2 * rng.standard_normal((4, nz, ny, nx))
    v = [F[q].ravel() for q in range(4)]
    gl = [D1[a] @ v[0] for a in range(3)]
    gu = [[D1[a] @ v[1 + i] for a in range(3)] for i in range(3)]
    div = gu[0][0] + gu[1][1] + gu[2][2]
    R = [-(v[1] * gl[0] + v[2] * gl[1] + v[3] * gl[2]) - div]
    for i in range(3):
        lap = sum(D2[a] @ v[1 + i] for a in range(3))
        if path == P55:
            gd = sum((D2[i] if j == i else opmix(i, j)) @ v[1 + j] for j in range(3))
        else:
            gd = D1[i] @ div
        Sg = sum((0.5 * (gu[i][j] + gu[j][i]) - (div / 3 if i == j else 0.0)) * gl[j] for j in range(3))
        R.append(-sum(v[1 + j] * gu[i][j] for j in range(3)) - cs ** 2 * gl[i] + nu * (lap + gd / 3 + 2 * Sg))
    ref = np.stack(R).reshape(4, nz, ny, nx)
    assert relinf(O.rhs(F, dx, nu, cs, path), ref) < 1e-13


# ------------------------ P11: the discrete RHS tends to the CONTINUUM Eq. 1-3 at sixth order
@pytest.mark.parametrize("path", [P55, P19])
def test_p11_rhs_converges_to_continuum_equations(path):
    """Eq. 1-3 evaluated by sympy's symbolic differentiation of analytic fields (no stencil, no oracle code)."""
    import sympy as sp

    x, y, z = sp.symbols("x y z", real=True)
    X = (x, y, z)
    nu, cs = sp.Rational(1, 20), sp.Rational(6, 5)
    lnr = sp.Rational(3, 10) * sp.cos(x + 2 * y - z + sp.Rational(1, 3))
    u = [sp.Rational(1, 5) * sp.sin(2 * x - y + z), sp.Rational(1, 4) * sp.cos(x + y + 2 * z + 1),
         sp.Rational(3, 20) * sp.sin(-x + 2 * y + z + 2)]
    divu = sum(sp.diff(u[i], X[i]) for i in range(3))
    S = [[sp.Rational(1, 2) * (sp.diff(u[i], X[j]) + sp.diff(u[j], X[i])) - (sp.Rational(1, 3) * divu if i == j else 0)
          for j in range(3)] for i in range(3)]
    rhs_sym = [-sum(u[j] * sp.diff(lnr, X[j]) for j in range(3)) - divu]
    for i in range(3):
        rhs_sym.append(-sum(u[j] * sp.diff(u[i], X[j]) for j in range(3)) - cs ** 2 * sp.diff(lnr, X[i])
                       + nu * (sum(sp.diff(u[i], X[j], 2) for j in range(3)) + sp.Rational(1, 3) * sp.diff(divu, X[i])
                               + 2 * sum(S[i][j] * sp.diff(lnr, X[j]) for j in range(3))))
    fields = sp.lambdify((x, y, z), [lnr] + u, "numpy")
    exact = sp.lambdify((x, y, z), rhs_sym, "numpy")
    errs = []
    for n in (24, 48):
        dx = TWO_PI / n
        g = np.arange(n) * dx
        Z, Y, Xg = np.meshgrid(g, g, g, indexing="ij")
        F = np.stack([np.broadcast_to(a, Xg.shape) for a in fields(Xg, Y, Z)])
        ref = np.stack([np.broadcast_to(a, Xg.shape) for a in exact(Xg, Y, Z)])
        errs.append(relinf(O.rhs(F, dx, float(nu), float(cs), path), ref))
    assert errs[1] < 5e-6  # ~ (k dx)^6/140 with k dx = 2*2pi/48
    assert 5.5 < math.log2(errs[0] / errs[1]) < 6.5, errs


# ----------------------- P12: readings G4/G7 and the window helper used for big-grid parity
def test_p12_w_buffer_contents_do_not_matter_alpha1_is_zero():
    cfg = I.CONFIGS["C1"]
    F = I.make_state(cfg, n_override=16)
    dx = TWO_PI / 16
    for path in (P55, P19):
        a = O.rk3_step(F, dx, cfg.nu, cfg.cs, 0.1 * dx, 1, path)
        b = O.rk3_step(F, dx, cfg.nu, cfg.cs, 0.1 * dx, 1, path, W=np.full_like(F, np.nan))
        assert np.array_equal(a, b)


def test_p12_19_and_55_point_paths_differ_at_sixth_order_only():
    diffs = []
    for n in (16, 32):
        cfg = I.CONFIGS["C1"]
        F = I.make_state(cfg, n_override=n)
        dx = TWO_PI / n
        a = O.rk3_step(F, dx, cfg.nu, cfg.cs, 0.1 * dx, 1, P55)
        b = O.rk3_step(F, dx, cfg.nu, cfg.cs, 0.1 * dx, 1, P19)
        diffs.append(relinf(b, a))
    assert 0 < diffs[1] < 1e-6  # two discretisations (reading G7): not equal ...
    # ... and the gap closes like dx^6 times dt ~ dx: between 2^5 and 2^8 per refinement
    assert 2 ** 5 < diffs[0] / diffs[1] < 2 ** 8, diffs


@pytest.mark.parametrize("path", [P55, P19])
def test_p12_windowed_step_equals_full_grid_step_on_the_interior(path):
    rng = np.random.default_rng(9)
    n = 48
    F = 0.05 * rng.standard_normal((4, n, n, n))
    dx = TWO_PI / n
    full = O.rk3_step(F, dx, 5e-3, 1.0, 0.1 * dx, 1, path)
    m = O.window_margin(path)
    size = 4 + 2 * m
    origin = (n - m - 2, 5 - m, 20 - m)  # straddles the periodic seam in z
    sub = I.gather_block(F, origin, size)
    got, mm = O.rk3_step_window(sub, dx, 5e-3, 1.0, 0.1 * dx, 1, path)
    assert mm == m
    exp = I.gather_block(full, tuple(o + m for o in origin), 4)
    assert np.array_equal(got, exp)
    # one cell less margin must break it (the margin is tight, not padded)
    if path == P55:
        sub2 = I.gather_block(F, tuple(o + 1 for o in origin), size - 2)
        bad = O.rk3_step(sub2, dx, 5e-3, 1.0, 0.1 * dx, 1, path)[:, m - 1:-(m - 1), m - 1:-(m - 1), m - 1:-(m - 1)]
        assert not np.array_equal(bad, exp)


def test_p12_float_instantiation_tracks_double():
    cfg = I.CONFIGS["C2"]
    F32 = I.make_state(cfg, n_override=24)
    dx = TWO_PI / 24
    a = O.rk3_step(F32.astype(np.float64), dx, cfg.nu, cfg.cs, 0.1 * dx, 1, P55)
    b = O.rk3_step(F32, dx, cfg.nu, cfg.cs, 0.1 * dx, 1, P55, dtype=np.float32)
    assert b.dtype == np.float32
    assert relinf(b.astype(np.float64), a) < 2e-6


@pytest.mark.parametrize("path", [P55, P19])
def test_p12_float_rhs_tracks_double(path):
    """fdo_rhs_f32 (the float instantiation of the pinned template) follows fdo_rhs_f64 on fp32-representable inputs."""
    cfg = I.CONFIGS["C2"]
    F32 = I.make_state(cfg, n_override=24)
    dx = TWO_PI / 24
    a = O.rhs(F32.astype(np.float64), dx, cfg.nu, cfg.cs, path)
    b = O.rhs(F32, dx, cfg.nu, cfg.cs, path, dtype=np.float32)
    assert b.dtype == np.float32
    assert relinf(b.astype(np.float64), a) < 2e-6


# ------------------------------------------------------------------------------------------------------------------
# P13  forcing term of Eq. 2 (Eq. 24-25, oracle step O11)
def _forcing_expected(spec, cs):
    """N and the unit vector f_k of Eq. 25, from vector algebra only."""
    k, e = np.asarray(spec["k"], float), np.asarray(spec["e"], float)
    N = spec["f0"] * cs * math.sqrt(np.linalg.norm(k) * cs / spec["dt"])
    fk = np.cross(k, e)
    return N, fk / np.linalg.norm(fk)  # |k x e| = sqrt(|k|^2 |e|^2 - (k.e)^2) for a unit e (Lagrange's identity)


def test_p13_forcing_field_is_one_transverse_fourier_mode_of_amplitude_n():
    n, cs = 16, 1.3
    dx = TWO_PI / n
    e = np.array([0.3, -0.5, 0.8])
    spec = dict(k=(2, -1, 3), e=tuple(e / np.linalg.norm(e)), phi=0.7, f0=0.05, dt=0.02)  # e need not be normal to k
    f = O.rhs(np.zeros((4, n, n, n)), dx, 0.01, cs, P55, force=spec)  # uniform state at rest: the RHS is f alone (P5)
    N, fk = _forcing_expected(spec, cs)
    assert abs(N - 0.05 * 1.3 * math.sqrt(math.sqrt(14.0) * 1.3 / 0.02)) < 1e-15  # Eq. 25 with the numbers put in
    assert abs(np.dot(fk, spec["k"])) < 1e-15 and abs(np.dot(fk, spec["e"])) < 1e-15  # solenoidal, normal to e
    assert np.array_equal(f[0], np.zeros((n, n, n)))  # no source in the continuity equation
    for a in range(3):
        spec_a = np.fft.fftn(f[1 + a]) / n ** 3  # array axes are (z, y, x)
        peak = spec_a[3, -1, 2]  # the +k mode
        assert abs(peak - 0.5 * N * fk[a] * np.exp(1j * 0.7)) < 1e-14
        spec_a[3, -1, 2] = spec_a[-3, 1, -2] = 0
        assert np.abs(spec_a).max() < 1e-15  # and nothing else
    # the 19-point path carries the same f
    assert np.array_equal(O.rhs(np.zeros((4, n, n, n)), dx, 0.01, cs, P19, force=spec), f)


@pytest.mark.parametrize("path", [P55, P19])
def test_p13_forcing_adds_to_the_rhs_and_leaves_it_when_switched_off(path):
    cfg = I.CONFIGS["C1"]
    F = I.make_state(cfg, n_override=12)
    dx = TWO_PI / 12
    spec = dict(k=(1, 2, 0), e=(0, 0, 1), phi=-1.1, f0=0.3, dt=0.01)
    plain = O.rhs(F, dx, cfg.nu, cfg.cs, path)
    forced = O.rhs(F, dx, cfg.nu, cfg.cs, path, force=spec)
    f = O.rhs(np.zeros_like(F), dx, cfg.nu, cfg.cs, path, force=spec)
    assert relinf(forced - plain, f) < 1e-13
    assert np.array_equal(O.rhs(F, dx, cfg.nu, cfg.cs, path), plain)  # the context manager switched it off again
    with pytest.raises(ValueError):
        O.rhs(F, dx, cfg.nu, cfg.cs, path, force=dict(k=(0, 0, 2), e=(0, 0, 1), phi=0, f0=1, dt=0.01))  # k parallel to e


@pytest.mark.parametrize("path", [P55, P19])
@pytest.mark.parametrize("axis,e", [(0, (0, 0, 1)), (1, (1, 0, 0)), (2, (0, 1, 0))])
def test_p13_forced_shear_mode_from_rest_closed_form(path, axis, e):
    """k along an axis: f is a transverse shear mode, every nonlinear term and div u vanish identically in the discrete
    system, and u = a_n f_k cos(k x + phi) with the inhomogeneous RK3 recurrence a_{n+1} = G a_n + N dt (G - 1)/z,
    G = 1 + z + z^2/2 + z^3/6, z = -nu dt s2(k dx)/dx^2 — which pins that f enters w with the weight dt of Eq. 10, on
    all three substeps, with N formed from the step's own dt."""
    n, kk, nu, nsteps = 24, 3, 0.02, 7
    dx = TWO_PI / n
    dt = 0.1 * dx
    kvec = [0, 0, 0]
    kvec[axis] = kk
    spec = dict(k=tuple(kvec), e=e, phi=0.4, f0=0.02, dt=dt)
    out = O.rk3_step(np.zeros((4, n, n, n)), dx, nu, 1.0, dt, nsteps, path, force=spec)
    N, fk = _forcing_expected(spec, 1.0)
    z = -nu * dt * s2(kk * dx) / dx ** 2
    G = 1 + z + z * z / 2 + z ** 3 / 6
    a = 0.0
    for _ in range(nsteps):
        a = G * a + N * dt * (1 + z / 2 + z * z / 6)
    idx = np.arange(n) * dx
    shape = [1, 1, 1]
    shape[2 - axis] = n
    c = np.cos(kk * idx + 0.4).reshape(shape)
    assert np.abs(out[0]).max() < 1e-16
    for comp in range(3):
        np.testing.assert_allclose(out[1 + comp], a * fk[comp] * c * np.ones((n, n, n)), atol=2e-15 * abs(a))
    assert abs(a) > 1e-3  # the test is not vacuous


def test_p13_windowed_forced_step_equals_the_full_grid_step():
    rng = np.random.default_rng(3)
    n = 40
    F = 0.05 * rng.standard_normal((4, n, n, n))
    dx = TWO_PI / n
    spec = dict(k=(2, 1, -1), e=(0, 0, 1), phi=0.2, f0=0.1, dt=0.1 * dx)
    full = O.rk3_step(F, dx, 5e-3, 1.0, 0.1 * dx, 1, P55, force=spec)
    m = O.window_margin(P55)
    origin = (n - m - 2, 5 - m, 20 - m)  # (k0, j0, i0) of the block's first cell; the oracle takes (x, y, z) order
    sub = I.gather_block(F, origin, 4 + 2 * m)
    got = O.rk3_step(sub, dx, 5e-3, 1.0, 0.1 * dx, 1, P55, force=spec, origin=origin[::-1])[:, m:-m, m:-m, m:-m]
    exp = I.gather_block(full, tuple(o + m for o in origin), 4)
    assert relinf(got, exp) < 1e-13  # the phase k.x of a shifted origin differs from the full grid's by rounding only
