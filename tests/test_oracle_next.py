"""Pins of the oracle's SURVEY.md section 8(f) additions (all `-m "not gpu"`): PERIODIC
dimensions (R21), the weighted harmonic mean (R22) and the weighted reduction.  As in
test_oracle_pins.py nothing here re-types the oracle's formulas: every expected value comes from
the mathematics (shift invariance, exact shifts, closed forms) or from a library routine."""
import math

import numpy as np
import pytest

from paper_2104_14561_b200 import workloads as W

A, C, P = W.FACE_ABSORB, W.FACE_CLAMP, W.FACE_PERIODIC


def _wl(x, dt, Q, kinds, vals, slope_rule=0):
    x = tuple(np.asarray(a, dtype=np.float64) for a in x)
    return W.Workload("t", x, dt, 1, tuple(Q), np.asarray(kinds, dtype=np.int32).reshape(-1, 2),
                      np.asarray(vals, dtype=np.float64).reshape(-1, 2), None, slope_rule=slope_rule)


# ----------------------------------------------------------------------------- periodic (R21)
def test_periodic_slopes_are_the_interior_rule_across_the_seam(oracle_mod):
    # the periodic extension of the data, shifted by one node, must give the same slopes shifted:
    # the interior rule of Eq. 15 is applied at the seam as anywhere else
    rng = np.random.default_rng(3)
    n = 12
    x = 0.25 * np.arange(n)                               # exact spacing: shifts are exact
    u = rng.uniform(0, 1, n)
    u[-1] = u[0]
    d = oracle_mod.pchip_slopes(x, u, periodic=True)
    assert d[0] == d[-1]
    for s in range(1, n - 1):
        ur = np.concatenate([u[s:-1], u[:s + 1]])            # start the period at node s
        dr = oracle_mod.pchip_slopes(x, ur, periodic=True)
        np.testing.assert_allclose(dr[:-1], np.concatenate([d[s:-1], d[:s]]), rtol=0, atol=1e-15)
    # and away from the seam it is the non-periodic result
    dn = oracle_mod.pchip_slopes(x, u, periodic=False)
    np.testing.assert_array_equal(d[1:-1], dn[1:-1])
    # seam value by hand for a sawtooth: u = (0, 1, 0, ..): differences +,- at node 0 -> 0
    saw = np.array([0.0, 1.0, 0.0, 1.0, 0.0])
    assert oracle_mod.pchip_slopes(np.arange(5.0), saw, periodic=True)[0] == 0.0
    # monotone across the seam is impossible for periodic data unless constant: a ramp with a
    # jump has deltas (1,1,1,-3): node 0 sees (-3, 1) -> 0, node 1 sees (1,1) -> 1
    ramp = np.array([0.0, 1.0, 2.0, 3.0, 0.0])
    np.testing.assert_allclose(oracle_mod.pchip_slopes(np.arange(5.0), ramp, periodic=True),
                               [0.0, 1.0, 1.0, 0.0, 0.0], atol=1e-15)


def test_periodic_pure_shift_crosses_the_seam(oracle_mod):
    # sigma = 0 and b dt = -3 h exactly: u_new(j) = u(j - 3) with indices modulo the period
    n = 17
    x = np.linspace(-1.0, 1.0, n)                          # h = 1/8: exact in binary
    h = x[1] - x[0]
    wl = _wl([x], 0.25, [5], [[P, P]], [[0, 0]])
    o = oracle_mod.Oracle(wl)
    rng = np.random.default_rng(5)
    u = rng.uniform(0, 1, n)
    u[-1] = u[0]
    b = np.full((1, n), -3 * h / wl.dt)
    out = o.apply(b, np.zeros((1, n)), u)
    per = u[:-1]
    expect = np.roll(per, 3)
    np.testing.assert_allclose(out[:-1], expect, rtol=0, atol=1e-15)
    assert abs(out[-1] - out[0]) < 1e-15


@pytest.mark.parametrize("d", [2, 3])
def test_periodic_axis_is_translation_invariant(oracle_mod, d):
    # coefficients that do not depend on the periodic coordinate: the operator commutes with
    # shifts by whole cells along it, INCLUDING across the seam (wrap of the points, slopes at
    # the seam, image node).  Diffusion wide enough that points wrap.
    rng = np.random.default_rng(11 + d)
    n = (10, 7) if d == 2 else (6, 9, 5)
    ax = 0 if d == 2 else 1                                 # the periodic axis
    x = [np.linspace(0.0, 1.0, m) for m in n]
    kinds = [[A, A]] * d
    kinds[ax] = [P, P]
    vals = [[1.0, 0.5]] * d
    wl = _wl(x, 0.01, [4] * d, kinds, vals)
    o = oracle_mod.Oracle(wl)
    J = wl.J
    other = [k for k in range(d) if k != ax]
    shape1 = [1] * d
    def along_others(f):
        return np.broadcast_to(f, n).reshape(-1).copy()
    bs, ss = [], []
    for k in range(d):
        shp = list(n)
        shp[ax] = 1
        bs.append(along_others(rng.uniform(-3, 3, shp)))
        ss.append(along_others(rng.uniform(0.2, 1.5, shp)))
    b, s = np.stack(bs), np.stack(ss)
    u = rng.uniform(0, 1, n)
    idx = [slice(None)] * d
    idx[ax] = -1
    idx0 = list(idx)
    idx0[ax] = 0
    u[tuple(idx)] = u[tuple(idx0)]                          # image node
    out = o.apply(b, s, u.reshape(-1)).reshape(n)
    for shift in (1, 4):
        per = np.take(u, range(n[ax] - 1), axis=ax)
        ur = np.roll(per, shift, axis=ax)
        ur = np.concatenate([ur, np.take(ur, [0], axis=ax)], axis=ax)
        outr = o.apply(b, s, ur.reshape(-1)).reshape(n)
        expect = np.roll(np.take(out, range(n[ax] - 1), axis=ax), shift, axis=ax)
        np.testing.assert_allclose(np.take(outr, range(n[ax] - 1), axis=ax), expect, rtol=0, atol=2e-15)
    # the image node is pushed from x[n-1] and wrapped: same value up to the rounding of the wrap
    np.testing.assert_allclose(np.take(out, 0, axis=ax), np.take(out, n[ax] - 1, axis=ax), rtol=0, atol=2e-15)


def test_periodic_constants_and_row_sums(oracle_mod):
    wl = W.small(6)
    o = oracle_mod.Oracle(wl)
    b, s = wl.coeffs(2)
    np.testing.assert_allclose(o.apply(b, s, np.ones(wl.J)), 1.0, rtol=0, atol=1e-14)
    Pm = o.algorithm1(6)
    assert Pm.min() >= -1e-13 and Pm.max() <= 1 + 1e-13
    g = Pm[-1].reshape(wl.n)
    assert np.all(g[:, 0] == 1.0) and np.all(g[:, -1] == 1.0)
    np.testing.assert_allclose(g[0], g[-1], rtol=0, atol=1e-13)   # image node carries the same values


# ----------------------------------------------------------------------------- weighted (R22)
def test_weighted_slopes_match_scipy_pchip_on_a_nonuniform_grid(oracle_mod):
    # scipy's PchipInterpolator uses the Fritsch-Carlson weighted harmonic mean at interior
    # nodes (its end nodes use a three-point formula: not compared)
    from scipy.interpolate import PchipInterpolator
    rng = np.random.default_rng(2)
    x = np.cumsum(rng.uniform(0.05, 1.0, 30))
    for trial in range(4):
        u = np.cumsum(rng.uniform(-0.3, 1.0, 30)) if trial % 2 else rng.uniform(0, 1, 30)
        d = oracle_mod.pchip_slopes(x, u, weighted=True)
        ref = PchipInterpolator(x, u).derivative()(x)
        np.testing.assert_allclose(d[1:-1], ref[1:-1], rtol=1e-13, atol=1e-14)


def test_weighted_equals_unweighted_on_uniform_grids_and_end_rule(oracle_mod):
    rng = np.random.default_rng(4)
    x = np.linspace(0, 3, 25)
    u = np.cumsum(rng.uniform(0, 1, 25))
    np.testing.assert_allclose(oracle_mod.pchip_slopes(x, u, weighted=True),
                               oracle_mod.pchip_slopes(x, u, weighted=False), rtol=1e-15)
    # end rule by hand: x = (0, 1, 3), u = (0, 1, 2): delta = (1, 1/2), h = (1, 2);
    # node 0: w1 = 2*2+1 = 5, w2 = 2+2*1 = 4 -> 9 / (5/1 + 4/(1/2)) = 9/13
    d = oracle_mod.pchip_slopes(np.array([0.0, 1.0, 3.0]), np.array([0.0, 1.0, 2.0]), weighted=True)
    assert abs(d[0] - 9.0 / 13.0) < 1e-15 and abs(d[1] - 9.0 / 13.0) < 1e-15
    # last node takes (delta_{n-2}, delta_{n-3}) with their own widths: w1 = 2*1+2 = 4, w2 = 1+4 = 5
    # -> 9 / (4/(1/2) + 5/1) = 9/13 as well (symmetric data); an asymmetric check:
    d = oracle_mod.pchip_slopes(np.array([0.0, 1.0, 3.0, 3.5]), np.array([0.0, 1.0, 2.0, 4.0]), weighted=True)
    # node 3: da = delta_2 = 4 (h = 0.5), db = delta_1 = 1/2 (h = 2): w1 = 2*2+0.5 = 4.5, w2 = 2+1 = 3
    assert abs(d[3] - 7.5 / (4.5 / 4.0 + 3.0 / 0.5)) < 1e-15


def test_weighted_rule_keeps_affine_exactness_on_the_radial_grid(oracle_mod):
    wl = W.small(7)
    wl.face_kind[:] = A
    o = oracle_mod.Oracle(wl)
    X = wl.mesh()
    rng = np.random.default_rng(8)
    J = wl.J
    hmin = [np.diff(a).min() for a in wl.x]
    amax = [oracle_mod.gauss_hermite(q)[0][-1] for q in wl.Q]
    b = np.stack([rng.uniform(-1, 1, J) * 0.3 * hmin[k] / wl.dt for k in range(3)])
    s = np.stack([rng.uniform(0, 1, J) * 0.6 * hmin[k] / (math.sqrt(2 * wl.dt) * amax[k]) for k in range(3)])
    c = rng.uniform(-1, 1, 4)
    u = c[0] + sum(c[k + 1] * X[k] for k in range(3))
    out = o.apply(b, s, u)
    expect = c[0] + sum(c[k + 1] * (X[k] + b[k] * wl.dt) for k in range(3))
    idx = np.unravel_index(np.arange(J), wl.n)
    inner = np.ones(J, bool)
    for k in range(3):
        inner &= (idx[k] > 0) & (idx[k] < wl.n[k] - 1)
    np.testing.assert_allclose(out[inner], expect[inner], rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------- reduction
def test_reduce_is_the_weighted_sum(oracle_mod):
    rng = np.random.default_rng(6)
    Pm = rng.uniform(0, 1, (7, 501))
    w = rng.uniform(-1, 1, 501)
    got = oracle_mod.reduce(Pm, w)
    np.testing.assert_allclose(got, Pm @ w, rtol=0, atol=1e-13)
    assert abs(oracle_mod.reduce(np.ones((1, 501)), w)[0] - math.fsum(w)) < 1e-14
    # trapezoid weights integrate a linear P exactly: int_0^2 (1 + 3x) dx = 8
    x = np.linspace(0, 2, 501)
    tw = np.full(501, x[1] - x[0])
    tw[[0, -1]] *= 0.5
    assert abs(oracle_mod.reduce((1 + 3 * x)[None], tw)[0] - 8.0) < 1e-13
