"""Pins of the CPU oracle against things other than itself (no GPU needed).

Each test names the passage that fixes the expected value: a closed form, a library routine,
the hand-derived micro-example in tests/golden/, an invariant, or brute-force Monte-Carlo.
"""
import math
import os

import numpy as np
import pytest

from paper_2104_14561_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- Gauss-Hermite
def test_gh_closed_forms(oracle_mod):
    # density pi^{-1/2} e^{-xi^2}  =>  weights sum to 1 (reading R1)
    a, w = oracle_mod.gauss_hermite(1)
    assert a[0] == 0.0 and w[0] == pytest.approx(1.0, abs=1e-15)
    a, w = oracle_mod.gauss_hermite(2)
    np.testing.assert_allclose(a, [-1 / math.sqrt(2), 1 / math.sqrt(2)], rtol=0, atol=2e-16)
    np.testing.assert_allclose(w, [0.5, 0.5], rtol=0, atol=2e-16)
    a, w = oracle_mod.gauss_hermite(3)
    np.testing.assert_allclose(a, [-math.sqrt(1.5), 0.0, math.sqrt(1.5)], rtol=0, atol=3e-16)
    np.testing.assert_allclose(w, [1 / 6, 2 / 3, 1 / 6], rtol=0, atol=3e-16)


@pytest.mark.parametrize("Q", [4, 6, 8, 16, 32])
def test_gh_moments_and_library(oracle_mod, Q):
    a, w = oracle_mod.gauss_hermite(Q)
    assert np.all(np.diff(a) > 0)                       # ascending abscissae
    np.testing.assert_allclose(a, -a[::-1], atol=1e-15)
    # exact for polynomials of degree <= 2Q-1: E[xi^{2m}] = (2m-1)!!/2^m under pi^{-1/2}e^{-xi^2}
    for m in range(0, Q):
        exact = math.prod(range(1, 2 * m, 2)) / 2.0 ** m
        assert float(np.sum(w * a ** (2 * m))) == pytest.approx(exact, rel=2e-13)
    an, wn = np.polynomial.hermite.hermgauss(Q)         # library rule for weight e^{-x^2}
    np.testing.assert_allclose(a, an, rtol=0, atol=5e-14)
    np.testing.assert_allclose(w, wn / math.sqrt(math.pi), rtol=5e-12, atol=1e-300)


def test_gh_table_value(oracle_mod):
    a, _ = oracle_mod.gauss_hermite(16)
    assert a[-1] == pytest.approx(4.688738939305818, abs=2e-15)   # standard 16-point table


# ----------------------------------------------------------------------------- Eq. 15 slopes
def test_slopes_interior_match_library_on_uniform_grid(oracle_mod):
    # On a uniform grid Fritsch-Carlson's weighted mean [17] equals Eq. 15's harmonic mean
    # (reading R5), so scipy's PCHIP derivative at interior nodes is an independent pin.
    from scipy.interpolate import PchipInterpolator
    rng = np.random.default_rng(3)
    x = np.linspace(-1.0, 2.0, 41)
    u = rng.uniform(0, 1, x.size)
    u[10:14] = u[10]                                    # flat run: zero differences (R7)
    du = oracle_mod.pchip_slopes(x, u)
    ref = PchipInterpolator(x, u).derivative()(x)
    np.testing.assert_allclose(du[1:-1], ref[1:-1], rtol=0, atol=1e-13)


def test_slopes_sign_rule_and_end_nodes(oracle_mod):
    # opposite signs -> 0; same sign -> 2/(1/d1+1/d2); ends use first/last two
    x = np.array([0.0, 1.0, 3.0, 4.0, 6.0])
    u = np.array([0.0, 1.0, 5.0, 4.0, 3.0])            # deltas: 1, 2, -1, -0.5
    du = oracle_mod.pchip_slopes(x, u)
    hm = lambda p, q: 2.0 / (1.0 / p + 1.0 / q)
    np.testing.assert_allclose(du, [hm(1, 2), hm(1, 2), 0.0, hm(-1, -0.5), hm(-0.5, -1)],
                               rtol=0, atol=1e-15)
    du = oracle_mod.pchip_slopes(x, np.array([0.0, 1.0, 1.0, 2.0, 2.0]))   # zero differences
    np.testing.assert_allclose(du, [0.0, 0.0, 0.0, 0.0, 0.0], atol=0)


def test_interp_1d_matches_library_hermite_spline(oracle_mod):
    # Eq. 14 is the cubic Hermite cell formula: with the oracle's own slopes
    # scipy's CubicHermiteSpline must reproduce the interpolant at arbitrary points.
    from scipy.interpolate import CubicHermiteSpline
    rng = np.random.default_rng(5)
    x = np.sort(np.concatenate([[0.0, 1.0], rng.uniform(0, 1, 17)]))      # non-uniform grid
    wl = W.brownian_1d(nodes=x.size, lo=0.0, hi=1.0)
    wl.x = (x,)
    u = np.sort(rng.uniform(0, 1, x.size))
    o = oracle_mod.Oracle(wl)
    z = np.concatenate([rng.uniform(0, 1, 200), x])                       # incl. the nodes
    ref = CubicHermiteSpline(x, u, oracle_mod.pchip_slopes(x, u))(z)
    np.testing.assert_allclose(o.interp(u, z), ref, rtol=0, atol=3e-15)
    np.testing.assert_allclose(o.interp(u, x), u, rtol=0, atol=5e-16)


# ----------------------------------------------------------------------------- micro-example
def _read_golden():
    vals, slopes = [], []
    for line in open(os.path.join(GOLD, "micro_1d.txt")):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] == "slope":
            slopes.append((float(t[1]), float(t[2]), int(t[3])))
        else:
            vals.append((int(t[0]), float(t[1]), float(t[2]), int(t[3])))
    return vals, slopes


def test_micro_example_golden(oracle_mod):
    wl = W.brownian_1d(nodes=5, N=3, T_max=0.015, Q=2, D=0.5, lo=0.0, hi=1.0)
    o = oracle_mod.Oracle(wl)
    P = o.algorithm1()
    vals, slopes = _read_golden()
    assert len(vals) == 6 and len(slopes) == 2
    for step, xnode, v, digits in vals:
        j = int(round(xnode * 4))
        assert abs(P[step, j] - v) < 1.5 * 10.0 ** (-digits), (step, xnode)
        assert abs(P[step, 4 - j] - v) < 1.5 * 10.0 ** (-digits)         # mirror symmetry
    # step 1 by hand: 1/2 * (1+2t)(1-t)^2, t = 1-0.4/sqrt(2), (1-t)^2 = 0.08
    hand = 0.5 * (3.0 - 0.8 / math.sqrt(2.0)) * 0.08
    assert P[1, 1] == pytest.approx(hand, abs=2e-16)
    du = oracle_mod.pchip_slopes(wl.x[0], P[1])
    for xnode, v, digits in slopes:
        assert abs(du[int(round(xnode * 4))] - v) < 1.5 * 10.0 ** (-digits)


# ----------------------------------------------------------------------------- one application
def _affine_setup(d, rng, clamp=False):
    n = {1: (41,), 2: (23, 19), 3: (13, 11, 9)}[d]
    if d == 1:
        wl = W.brownian_1d(nodes=n[0], Q=5)
    elif d == 2:
        wl = W.cellular_2d(n=n, N=4, Q=(4, 5))
    else:
        wl = W.runaway_3d(n=n, N=4, Q=(3, 4, 5))
        wl.face_kind[:] = W.FACE_ABSORB
    wl.dt = 1e-3
    return wl


@pytest.mark.parametrize("d", [1, 2, 3])
def test_constant_and_affine_fields_are_reproduced(oracle_mod, d):
    # Row sums are 1 and PCHIP slopes of a linear function are exact; the GH rule is symmetric:
    # u = c0 + sum c_k x_k  |->  c0 + sum c_k (x_k + b_k dt) when every point stays inside.
    rng = np.random.default_rng(10 + d)
    wl = _affine_setup(d, rng)
    o = oracle_mod.Oracle(wl)
    J = wl.J
    X = wl.mesh()
    h = [a[1] - a[0] for a in wl.x]
    # keep all quadrature points inside: |b dt| + sigma sqrt(2dt) a_max < distance to the box
    amax = [oracle_mod.gauss_hermite(q)[0][-1] for q in wl.Q]
    b = np.stack([rng.uniform(-1, 1, J) * 0.3 * h[k] / wl.dt for k in range(d)])
    s = np.stack([rng.uniform(0, 1, J) * 0.6 * h[k] / (math.sqrt(2 * wl.dt) * amax[k])
                  for k in range(d)])
    c = rng.uniform(-1, 1, d + 1)
    u = c[0] + sum(c[k + 1] * X[k] for k in range(d))
    out = o.apply(b, s, u)
    expect = c[0] + sum(c[k + 1] * (X[k] + b[k] * wl.dt) for k in range(d))
    chi_mask = np.ones(J, bool)
    idx = np.unravel_index(np.arange(J), wl.n)
    for k in range(d):
        chi_mask &= (idx[k] > 0) & (idx[k] < wl.n[k] - 1)
    np.testing.assert_allclose(out[chi_mask], expect[chi_mask], rtol=0, atol=2e-14)
    np.testing.assert_array_equal(out[~chi_mask], u[~chi_mask])          # Dirichlet nodes kept
    ones = o.apply(b, s, np.ones(J))
    np.testing.assert_allclose(ones, 1.0, rtol=0, atol=1e-14)


def _slope_bubble(h, t):
    # sum of the two slope basis functions of Eq. 14 on a cell of width h at
    # local coordinate t: h t (1-t)^2 + h t^2 (t-1) = h t (1-t) (1-2t)
    return h * t * (1.0 - t) * (1.0 - 2.0 * t)


def test_bilinear_field_exact_value_of_reading_A_in_2d(oracle_mod):
    # Reading R4/A carries values + nodal gradient only.  For
    # u = x*y the nodal slopes are exact (y along x-lines, x along y-lines) and the 1-D Hermite
    # interpolant reproduces linear functions, so on any cell the interpolant of Eq. 13 is
    #     x*y - s_x(t_x) * s_y(t_y),      s(t) = h t (1-t) (1-2t),
    # the bilinear "bubble" a full tensor PCHIP would not have.  The value pins which corner each
    # slope term of Eq. 13 is taken from: a slope read from the wrong corner changes the product.
    wl = W.cellular_2d(n=(9, 9), N=2, Q=(1, 1))            # x in [0,2] h=1/4, y in [0,1] h=1/8
    X, Y = wl.mesh()
    o = oracle_mod.Oracle(wl)
    u = X * Y
    hx, hy = 0.25, 0.125
    for zx, zy in [(0.9, 0.43), (1.3125, 0.07), (0.06, 0.99)]:
        tx = (zx - math.floor(zx / hx) * hx) / hx
        ty = (zy - math.floor(zy / hy) * hy) / hy
        expect = zx * zy - _slope_bubble(hx, tx) * _slope_bubble(hy, ty)
        val = o.interp(u, np.array([[zx, zy]]))[0]
        assert abs(val - expect) < 2e-15, (zx, zy, val, expect)
        assert abs(val - zx * zy) > 1e-7 or abs(_slope_bubble(hx, tx) * _slope_bubble(hy, ty)) < 1e-7


def test_bilinear_fields_exact_value_of_reading_A_in_3d(oracle_mod):
    # same in 3-D: u = x*y + y*z  ->  x*y + y*z - s_x s_y - s_y s_z (each product is bilinear in two
    # coordinates and constant along the third, whose slope field is then 0)
    wl = W.runaway_3d(n=(6, 9, 5), N=2, Q=(1, 1, 1))        # p in [0,50], xi in [-1,1], r in [0,1]
    X, Y, Z = wl.mesh()
    o = oracle_mod.Oracle(wl)
    u = X * Y + Y * Z
    h = [10.0, 0.25, 0.25]
    lo = [0.0, -1.0, 0.0]
    for z in [(13.7, -0.41, 0.33), (41.0, 0.62, 0.9), (2.5, -0.93, 0.05)]:
        t = [((z[k] - lo[k]) - math.floor((z[k] - lo[k]) / h[k]) * h[k]) / h[k] for k in range(3)]
        s = [_slope_bubble(h[k], t[k]) for k in range(3)]
        expect = z[0] * z[1] + z[1] * z[2] - s[0] * s[1] - s[1] * s[2]
        val = o.interp(u, np.array([z]))[0]
        assert abs(val - expect) < 1e-14 * max(1.0, abs(expect)), (z, val, expect)


def test_sigma_zero_is_a_pure_shift_and_zero_drift_is_identity(oracle_mod):
    # sigma = 0 (or Q = 1): u_new(j) = u^J(x_j + b dt); b = 0 too => identity (SURVEY 8c pins)
    from scipy.interpolate import CubicHermiteSpline
    rng = np.random.default_rng(7)
    wl = W.brownian_1d(nodes=33, Q=7)
    x = wl.x[0]
    u = rng.uniform(0, 1, x.size)
    u[0] = u[-1] = 1.0
    o = oracle_mod.Oracle(wl)
    zero = np.zeros((1, x.size))
    np.testing.assert_allclose(o.apply(zero, zero, u), u, rtol=0, atol=1e-15)
    b = rng.uniform(-3, 3, (1, x.size))
    out = o.apply(b, zero, u)
    z = x + b[0] * wl.dt
    ref = CubicHermiteSpline(x, u, oracle_mod.pchip_slopes(x, u))(z)
    np.testing.assert_allclose(out[1:-1], ref[1:-1], rtol=0, atol=1e-14)


def test_face_rules_tie_break_and_clamp(oracle_mod):
    # Q=1 (a=0, w=1) makes a step a deterministic shift.  R8: outside an ABSORB face -> g;
    # R9: CLAMP dims are projected first, then the lowest ABSORB dimension outside decides.
    wl = W.cellular_2d(n=(5, 5), N=1, Q=(1, 1))
    wl.dt = 1.0
    wl.face_value[:] = [[0.25, 0.5], [0.75, 1.0]]
    o = oracle_mod.Oracle(wl)
    J = wl.J
    u = o.chi()
    ctr = 2 * 5 + 2                                        # node (1.0, 0.5)
    def run(bx, by):
        b = np.zeros((2, J)); b[0, ctr] = bx; b[1, ctr] = by
        return o.apply(b, np.zeros((2, J)), u)[ctr]
    assert run(+5, 0) == 0.5 and run(-5, 0) == 0.25
    assert run(0, +5) == 1.0 and run(0, -5) == 0.75
    assert run(+5, +5) == 0.5 and run(-5, +5) == 0.25      # both outside: dimension 0 wins
    wl.face_kind[0] = [W.FACE_CLAMP, W.FACE_CLAMP]
    o2 = oracle_mod.Oracle(wl)
    u2 = o2.chi()
    def run2(bx, by):
        b = np.zeros((2, J)); b[0, ctr] = bx; b[1, ctr] = by
        return o2.apply(b, np.zeros((2, J)), u2)[ctr]
    assert run2(+5, +5) == 1.0                              # dim 0 clamped, dim 1 decides
    # clamped onto x=2 (a non-Dirichlet face now): value interpolated there = chi = 0
    assert run2(+5, 0) == 0.0


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_lines_of_a_3d_problem_reproduce_the_1d_result(oracle_mod, axis):
    # Coefficients that act along one axis only, CLAMP faces on the other two: the field stays
    # constant across them (H0+H1=1, cross slopes 0), so every line equals the 1-D scheme.
    # Pins strides / index order of the tensor-product assembly (a transposed axis fails).
    n1 = 17
    ref_wl = W.ou_1d(nodes=n1, N=6, Q=5, dt=0.01)
    ref = oracle_mod.Oracle(ref_wl).algorithm1()
    n = [4, 5, 3]
    n[axis] = n1
    wl = W.runaway_3d(n=tuple(n), N=6, Q=(3, 3, 3), dt=0.01)
    Q = [3, 3, 3]; Q[axis] = 5
    wl.Q = tuple(Q)
    xs = [np.linspace(0, 1, m) for m in n]
    xs[axis] = ref_wl.x[0]
    wl.x = tuple(xs)
    wl.face_kind[:] = W.FACE_CLAMP
    wl.face_kind[axis] = W.FACE_ABSORB
    wl.face_value[:] = 0.0
    wl.face_value[axis] = 1.0
    J = wl.J
    idx = np.unravel_index(np.arange(J), n)

    def coeffs(step):
        b1, s1 = ref_wl.coeffs(step)
        b = np.zeros((3, J)); s = np.full((3, J), 0.2)
        b[axis] = b1[0][idx[axis]]
        s[axis] = s1[0][idx[axis]]
        other = [k for k in range(3) if k != axis]
        b[other[0]] = 0.7
        b[other[1]] = -0.4
        return b, s

    wl.coeffs = coeffs
    P = oracle_mod.Oracle(wl).algorithm1().reshape(7, *n)
    Pm = np.moveaxis(P, 1 + axis, -1).reshape(7, -1, n1)
    for line in range(Pm.shape[1]):
        np.testing.assert_allclose(Pm[:, line, :], ref, rtol=0, atol=2e-15)


# ----------------------------------------------------------------------------- Algorithm 1
def test_algorithm1_equals_per_column_scheme1_and_prefix(oracle_mod):
    # Algorithm 1 only reorders Eq. 29; columns never interact.
    wl = W.ou_1d(nodes=41, N=9, Q=6, dt=0.02)
    o = oracle_mod.Oracle(wl)
    P = o.algorithm1()
    for m in range(0, wl.N + 1):
        np.testing.assert_array_equal(P[m], o.column(m))
    np.testing.assert_array_equal(o.column(7), o.column_streamed(7))
    np.testing.assert_array_equal(o.algorithm1(5), P[:6])                 # prefix property
    np.testing.assert_array_equal(P[0], o.chi())


def test_time_ordering_of_operators(oracle_mod):
    # Eq. 29: the outermost operator is A_0.  With b switching sign at mid-time, applying the
    # operators in the reverse order gives a different column; the oracle must match the
    # explicit composition A_0(A_1(...chi)).
    wl = W.ou_1d(nodes=33, N=6, Q=4, dt=0.05)
    o = oracle_mod.Oracle(wl)
    u = o.chi()
    for nu in (5, 4, 3, 2, 1, 0):
        b, s = wl.coeffs(nu)
        u = o.apply(b, s, u)
    np.testing.assert_array_equal(u, o.column(6))
    v = o.chi()
    for nu in (0, 1, 2, 3, 4, 5):
        b, s = wl.coeffs(nu)
        v = o.apply(b, s, v)
    assert np.max(np.abs(u - v)) > 1e-3


def test_autonomous_chain(oracle_mod):
    # autonomous coefficients => column m+1 = one application to column m
    wl = W.brownian_1d(nodes=31, N=8, T_max=0.4, Q=6)
    o = oracle_mod.Oracle(wl)
    P = o.algorithm1()
    b, s = wl.coeffs(0)
    for m in range(wl.N):
        np.testing.assert_array_equal(o.apply(b, s, P[m]), P[m + 1])


# ----------------------------------------------------------------------------- vs. truth, 1-D
def brownian_exit_exact(T, x, L, D=0.5, terms=400):
    """Exit probability of dX = sqrt(2D) dW from (0, L) by time T (textbook Fourier series of
    the survival probability; corrected Eq. 31, reading R3: odd n only)."""
    x = np.asarray(x, float)
    S = np.zeros_like(x)
    for n in range(1, 2 * terms, 2):
        S += 4.0 / (n * math.pi) * np.sin(n * math.pi * x / L) * math.exp(-D * (n * math.pi / L) ** 2 * T)
    return 1.0 - S


def test_config1_against_closed_form(oracle_mod):
    # BASELINE config 1 violates Assumption 1 on purpose (off-domain -> 1): the scheme sits
    # within a few 1e-2 of the continuous-time closed form (probe 3.2e-2).
    wl = W.config(1)
    o = oracle_mod.Oracle(wl)
    col = o.column(wl.N)
    exact = brownian_exit_exact(1.0, wl.x[0] + 1.0, 2.0, D=0.5)
    err = np.max(np.abs(col - exact))
    assert err < 5e-2
    assert col[100] == pytest.approx(0.5975, abs=2e-3) and exact[100] == pytest.approx(0.62922, abs=1e-4)
    np.testing.assert_allclose(col, col[::-1], rtol=0, atol=1e-14)        # mirror symmetry


def test_first_order_in_dt_second_order_in_dx_fig1_setup(oracle_mod):
    # PAPER.md:323/329 (Fig. 1): L=10, T=3, Q=3, mesh obeying Assumption 1 / Remark 2 so that
    # every quadrature point stays in the closed box: h >= sqrt(3 dt).  Error ~ O(dt) ~ O(h^2).
    L, T = 10.0, 3.0
    errs, dts = [], []
    for N in (30, 120, 480):
        dt = T / N
        cells = int(math.floor(L / math.sqrt(3.0 * dt) * (1 - 1e-12)))
        wl = W.brownian_1d(nodes=cells + 1, N=N, T_max=T, Q=3, D=0.5, lo=0.0, hi=L)
        col = oracle_mod.Oracle(wl).column(N)
        errs.append(np.max(np.abs(col - brownian_exit_exact(T, wl.x[0], L))))
        dts.append(dt)
    order = np.polyfit(np.log(dts), np.log(errs), 1)[0]
    assert 0.8 < order < 1.3, (order, errs)
    assert errs[-1] < 5e-4 and errs[0] < 1e-2


def test_stable_when_assumption1_fails(oracle_mod):
    # "does not blow up" for any dt on a fixed mesh
    wl = W.brownian_1d(nodes=101, N=5, T_max=50.0, Q=8, lo=0.0, hi=10.0)
    P = oracle_mod.Oracle(wl).algorithm1()
    assert P.min() >= 0.0 and P.max() <= 1.0 + 1e-14
    assert np.all(np.diff(P, axis=0) >= -1e-14)


# ----------------------------------------------------------------------------- invariants
@pytest.mark.parametrize("idx", [2, 3, 4, 5])
def test_invariants_on_reduced_configs(oracle_mod, idx):
    # 0 <= P <= 1, non-decreasing in t, P = g on ABSORB faces
    wl = W.small(idx)
    shrink = {2: 20, 3: 8, 4: 8, 5: 4}[idx]
    o = oracle_mod.Oracle(wl)
    P = o.algorithm1(shrink)
    assert P.min() >= -1e-12 and P.max() <= 1.0 + 1e-12
    assert np.diff(P, axis=0).min() >= -1e-12
    chi = o.chi()
    grid = np.unravel_index(np.arange(wl.J), wl.n)
    on_face = np.zeros(wl.J, bool)
    for k in range(wl.d):
        if wl.face_kind[k][0] == W.FACE_ABSORB:
            on_face |= grid[k] == 0
        if wl.face_kind[k][1] == W.FACE_ABSORB:
            on_face |= grid[k] == wl.n[k] - 1
    for m in range(P.shape[0]):
        np.testing.assert_array_equal(P[m][on_face], chi[on_face])
    assert P[-1].max() > 0 and (idx != 3 or P[-1][~on_face].max() > 1e-3)


# ----------------------------------------------------------------------------- Monte-Carlo
def _mc_exit(wl_coeff, x0, lo, hi, g_lo, g_hi, dt, N, paths, seed):
    """Euler-Maruyama paths (Eq. 11), exit checked at step ends only."""
    rng = np.random.default_rng(seed)
    x = np.full(paths, x0)
    alive = np.ones(paths, bool)
    val = np.zeros(paths)
    for n in range(N):
        b, s = wl_coeff(n, x)
        x = np.where(alive, x + b * dt + s * math.sqrt(dt) * rng.standard_normal(paths), x)
        out_lo = alive & (x < lo)
        out_hi = alive & (x > hi)
        val[out_lo] = g_lo
        val[out_hi] = g_hi
        alive &= ~(out_lo | out_hi)
    return val.mean(), val.std() / math.sqrt(paths)


def test_monte_carlo_brownian(oracle_mod):
    wl = W.brownian_1d(nodes=81, N=40, T_max=1.0, Q=16)
    col = oracle_mod.Oracle(wl).column(wl.N)
    for x0, j in ((0.0, 40), (0.5, 60)):
        mc, se = _mc_exit(lambda n, x: (0.0, 1.0), x0, -1, 1, 1, 1, wl.dt, wl.N, 200000, 1)
        assert abs(col[j] - mc) < 0.03 + 4 * se, (x0, col[j], mc)
        # catches a dropped sqrt(2) (variance halved: P(1,0) ~ 0.37, doubled: ~0.83)
    assert 0.45 < col[40] < 0.70


def test_monte_carlo_time_ordering_with_one_sided_exit(oracle_mod):
    # Only the upper face counts as exit (g=1); the lower face absorbs with g=0.  Drift up in
    # the first half, down in the second: reversing the operator order changes P a lot.
    N, dt = 30, 1.0 / 30
    wl = W.ou_1d(nodes=121, N=N, Q=12, sigma=0.5, dt=dt)
    wl.face_value[:] = [[0.0, 1.0]]
    x = wl.x[0]

    def coeffs(n):
        c = 2.0 if n < N // 2 else -2.0
        return np.full((1, x.size), c), np.full((1, x.size), 0.5)

    wl.coeffs = coeffs
    col = oracle_mod.Oracle(wl).column(N)
    mc, se = _mc_exit(lambda n, xx: (2.0 if n < N // 2 else -2.0, 0.5), 0.0, -1, 1, 0, 1,
                      dt, N, 200000, 2)
    mc_rev, _ = _mc_exit(lambda n, xx: (-2.0 if n < N // 2 else 2.0, 0.5), 0.0, -1, 1, 0, 1,
                         dt, N, 200000, 3)
    assert abs(mc - mc_rev) > 0.15                       # the two orderings are far apart
    assert abs(col[60] - mc) < 0.04 + 4 * se, (col[60], mc, mc_rev)


def test_monte_carlo_2d_coarse(oracle_mod):
    # 2-D: drift in x only, diffusion in both; exit through any face.  Loose (coarse
    # multi-D grids differ from MC by a few 1e-2); pins gross errors of the tensor assembly.
    n = (41, 41)
    N, dt = 20, 0.01
    wl = W.cellular_2d(n=n, N=N, Q=(6, 6), dt=dt)
    wl.x = (np.linspace(0, 1, n[0]), np.linspace(0, 1, n[1]))
    J = wl.J
    wl.coeffs = lambda step: (np.stack([np.full(J, 1.5), np.zeros(J)]),
                              np.stack([np.full(J, 0.6), np.full(J, 0.9)]))
    col = oracle_mod.Oracle(wl).column(N).reshape(n)
    rng = np.random.default_rng(4)
    paths = 200000
    for (x0, y0) in ((0.5, 0.5), (0.75, 0.25)):
        X = np.full(paths, x0); Y = np.full(paths, y0)
        alive = np.ones(paths, bool)
        for _ in range(N):
            X = np.where(alive, X + 1.5 * dt + 0.6 * math.sqrt(dt) * rng.standard_normal(paths), X)
            Y = np.where(alive, Y + 0.9 * math.sqrt(dt) * rng.standard_normal(paths), Y)
            alive &= (X >= 0) & (X <= 1) & (Y >= 0) & (Y <= 1)
        mc = 1.0 - alive.mean()
        i, j = int(round(x0 * 40)), int(round(y0 * 40))
        assert abs(col[i, j] - mc) < 0.05, (x0, y0, col[i, j], mc)
