"""Seeded synthetic workloads shaped like the paper's examples (inputs only).

This module builds the *inputs* of the Feynman-Kac exit-time path: the box D, the tensor
grid, dt, N, the Gauss-Hermite order per dimension, the face rules, and the drift b(t_n, x_j)
and diffusion sigma(t_n, x_j) sampled per step.  It holds none of the method's arithmetic
(no quadrature, no interpolation, no operator): it is the one module both the CPU oracle's
tests and the CUDA path's tests/bench import, so that both sides see the same arrays.

The five workloads are BASELINE.json's `configs`, completed as SURVEY.md section 8(d)
proposes (every completion is listed in DESIGN.md "Input recipe").  They stand in for the
paper's examples (PAPER.md:303 1-D Brownian motion, PAPER.md:335 2-D cellular flow,
PAPER.md:385 3-D runaway electrons); none of the paper's figure data exists in this repo.

Only numpy (and math.erf through numpy.vectorize-free formulas) is used.
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass, field
from typing import Callable, Optional, Sequence, Tuple

import numpy as np

FACE_ABSORB = 0
FACE_CLAMP = 1
FACE_PERIODIC = 2
SLOPE_EQ15 = 0        # Eq. 15 as printed: unweighted harmonic mean
SLOPE_WEIGHTED = 1    # Fritsch-Carlson weighted harmonic mean (ref [17]) for non-uniform grids


@dataclass
class Workload:
    """One exit-time problem: everything `fk_create` / `fk_set_coeffs` need.

    x[k]        node coordinates along dimension k (strictly increasing, ends = box faces)
    dt, N       uniform time partition, T_max = N*dt (Eq. 10)
    Q[k]        Gauss-Hermite points along dimension k
    face_kind   [d][2] FACE_ABSORB / FACE_CLAMP / FACE_PERIODIC (both faces of a dimension)
    slope_rule  SLOPE_EQ15 or SLOPE_WEIGHTED
    face_value  [d][2] value g taken by a point leaving through an ABSORB face (1 = "exit")
    coeffs(n)   -> (b, sigma), float64 arrays [d][J], sampled at t_n = n*dt
    autonomous  True when coeffs(n) does not depend on n
    """

    name: str
    x: Tuple[np.ndarray, ...]
    dt: float
    N: int
    Q: Tuple[int, ...]
    face_kind: np.ndarray
    face_value: np.ndarray
    coeffs: Callable[[int], Tuple[np.ndarray, np.ndarray]]
    autonomous: bool = False
    note: str = ""
    extra: dict = field(default_factory=dict)
    slope_rule: int = SLOPE_EQ15

    @property
    def d(self) -> int:
        return len(self.x)

    @property
    def n(self) -> Tuple[int, ...]:
        return tuple(len(a) for a in self.x)

    @property
    def J(self) -> int:
        return int(np.prod(self.n))

    @property
    def updates(self) -> int:
        """Node-step updates U = J*N(N+1)/2 of the full evolution."""
        return self.J * self.N * (self.N + 1) // 2

    def mesh(self):
        """Coordinates of every node, each [J], node index j C-ordered (last dim fastest)."""
        g = np.meshgrid(*self.x, indexing="ij")
        return [np.ascontiguousarray(a.reshape(-1)) for a in g]

    def coeff_table(self, n0: int, n1: int):
        """Stack coeffs(n) for n in [n0, n1): returns (b, sigma) each [n1-n0][d][J]."""
        bs, ss = [], []
        for n in range(n0, n1):
            b, s = self.coeffs(n)
            bs.append(b)
            ss.append(s)
        return np.ascontiguousarray(np.stack(bs)), np.ascontiguousarray(np.stack(ss))


def _faces(kinds, values):
    return (np.asarray(kinds, dtype=np.int32).reshape(-1, 2),
            np.asarray(values, dtype=np.float64).reshape(-1, 2))


# --------------------------------------------------------------------------------------
# config 1: 1-D Brownian exit, autonomous
# --------------------------------------------------------------------------------------
def brownian_1d(nodes: int = 201, N: int = 200, T_max: float = 1.0, Q: int = 16,
                D: float = 0.5, lo: float = -1.0, hi: float = 1.0) -> Workload:
    x = np.linspace(lo, hi, nodes)
    sig = math.sqrt(2.0 * D)
    b = np.zeros((1, nodes))
    s = np.full((1, nodes), sig)
    kinds, vals = _faces([[FACE_ABSORB, FACE_ABSORB]], [[1.0, 1.0]])
    return Workload("cfg1_brownian_1d", (x,), T_max / N, N, (Q,), kinds, vals,
                    lambda n: (b, s), autonomous=True,
                    note="dX=sqrt(2D)dW, D=0.5 => sigma=1; both faces exit",
                    extra={"D": D})


# --------------------------------------------------------------------------------------
# config 2: 1-D time-dependent OU-type drift
# --------------------------------------------------------------------------------------
def ou_1d(nodes: int = 1025, N: int = 1000, T_max: float = 2.0, Q: int = 16,
          sigma: float = 0.3, dt: Optional[float] = None) -> Workload:
    x = np.linspace(-1.0, 1.0, nodes)
    dt = T_max / N if dt is None else dt
    s = np.full((1, nodes), sigma)

    def coeffs(n):
        t = n * dt
        b = (-x + 0.5 * math.sin(2.0 * math.pi * t)).reshape(1, nodes)
        return np.ascontiguousarray(b), s

    kinds, vals = _faces([[FACE_ABSORB, FACE_ABSORB]], [[1.0, 1.0]])
    return Workload("cfg2_ou_1d", (x,), dt, N, (Q,), kinds, vals, coeffs,
                    note="b=-x+0.5 sin(2 pi t), sigma=0.3, T_max=2 at full size")


# --------------------------------------------------------------------------------------
# config 3: 2-D chaotic advection-diffusion (time-periodic cellular flow)
# --------------------------------------------------------------------------------------
def cellular_2d(n=(257, 129), N: int = 2000, T_max: float = 2.0, Q=(8, 8),
                A: float = 1.0, eps: float = 0.25, omega: float = 2.0 * math.pi,
                kappa: float = 1e-3, dt: Optional[float] = None) -> Workload:
    """psi = A sin(pi x) sin(pi y) + eps sin(omega t) sin(pi x) sin(2 pi y); b = (-psi_y, psi_x).

    Same family as the paper's cellular flow, Eq. 33-35; the box and the
    perturbation follow BASELINE.json's config text as completed in SURVEY.md section 8(d).
    """
    x0 = np.linspace(0.0, 2.0, n[0])
    x1 = np.linspace(0.0, 1.0, n[1])
    dt = T_max / N if dt is None else dt
    X, Y = np.meshgrid(x0, x1, indexing="ij")
    X = X.reshape(-1)
    Y = Y.reshape(-1)
    pi = math.pi
    sx, cx = np.sin(pi * X), np.cos(pi * X)
    sy, cy = np.sin(pi * Y), np.cos(pi * Y)
    s2y, c2y = np.sin(2 * pi * Y), np.cos(2 * pi * Y)
    bx0 = -A * pi * sx * cy
    bx1 = -eps * 2 * pi * sx * c2y
    by0 = A * pi * cx * sy
    by1 = eps * pi * cx * s2y
    J = X.size
    sig = np.full((2, J), math.sqrt(2.0 * kappa))

    def coeffs(nstep):
        f = math.sin(omega * nstep * dt)
        b = np.empty((2, J))
        b[0] = bx0 + f * bx1
        b[1] = by0 + f * by1
        return b, sig

    kinds, vals = _faces([[FACE_ABSORB, FACE_ABSORB]] * 2, [[1.0, 1.0]] * 2)
    return Workload("cfg3_cellular_2d", (x0, x1), dt, N, tuple(Q), kinds, vals, coeffs,
                    note="A=1, eps=0.25, omega=2pi, kappa=1e-3; all faces exit")


# --------------------------------------------------------------------------------------
# configs 4 and 5: runaway electrons, Eq. 37-39
# --------------------------------------------------------------------------------------
_erf = np.vectorize(math.erf, otypes=[np.float64])


def _collision_terms(p, Zeff=1.0, delta=0.042, nu_ee=1.0, vT=1.0):
    """C_A, dC_A/dp, C_B, C_F, gamma on p>0."""
    gam = np.sqrt(1.0 + (delta * p) ** 2)
    y = p / gam
    phi = _erf(y)
    dphi = 2.0 / math.sqrt(math.pi) * np.exp(-y * y)
    psi = (phi - y * dphi) / (2.0 * y * y)
    dpsi = dphi - 2.0 * psi / y
    CA = nu_ee * vT ** 2 * psi / y
    dCA_dy = nu_ee * vT ** 2 * (dpsi / y - psi / (y * y))
    dCA_dp = dCA_dy / gam ** 3
    CB = 0.5 * nu_ee * vT ** 2 / y * (Zeff + phi - psi + 0.5 * y * y * delta ** 4)
    CF = 2.0 * nu_ee * vT * psi
    return CA, dCA_dp, CB, CF, gam


def _runaway_parts(P, XI, tau=1e5):
    """Split the (p, xi) drift into a stationary part and the part multiplying E."""
    ok = P > 0.0
    p = np.where(ok, P, 1.0)
    CA, dCA, CB, CF, gam = _collision_terms(p)
    one_m = 1.0 - XI * XI
    bp0 = -gam * p * one_m / tau - CF + 2.0 * CA / p + dCA
    bpE = XI.copy()
    bx0 = -XI * one_m / (tau * gam) - 2.0 * XI * CB / (p * p)
    bxE = one_m / p
    sp = np.sqrt(2.0 * CA)
    sx = np.sqrt(2.0 * CB) / p * np.sqrt(np.maximum(one_m, 0.0))
    for a in (bp0, bpE, bx0, bxE, sp, sx):
        a[~ok] = 0.0          # p = 0 lies on a Dirichlet face; never read (SURVEY.md 8d cfg 4)
    return bp0, bpE, bx0, bxE, sp, sx


def runaway_2d(n=(401, 201), N: int = 5000, T_max: float = 120.0, Q=(8, 8),
               p_max: float = 50.0, dt: Optional[float] = None) -> Workload:
    """(p, xi) rows of Eq. 37 with ramped E(t) = 0.1 + 0.5 t/T_ramp, T_ramp = 120."""
    xp = np.linspace(0.0, p_max, n[0])
    xx = np.linspace(-1.0, 1.0, n[1])
    dt = T_max / N if dt is None else dt
    P, XI = np.meshgrid(xp, xx, indexing="ij")
    P = P.reshape(-1)
    XI = XI.reshape(-1)
    bp0, bpE, bx0, bxE, sp, sx = _runaway_parts(P, XI)
    sig = np.ascontiguousarray(np.stack([sp, sx]))
    J = P.size

    def coeffs(nstep):
        E = 0.1 + 0.5 * (nstep * dt) / 120.0
        b = np.empty((2, J))
        b[0] = bp0 + E * bpE
        b[1] = bx0 + E * bxE
        return b, sig

    kinds, vals = _faces([[FACE_ABSORB, FACE_ABSORB], [FACE_CLAMP, FACE_CLAMP]],
                         [[0.0, 1.0], [0.0, 0.0]])
    return Workload("cfg4_runaway_2d", (xp, xx), dt, N, tuple(Q), kinds, vals, coeffs,
                    note="p in [0,50] exit at p_max (g=1), p=0 g=0, xi faces clamp; E ramp")


def radial_grid(coarse: int = 7, fine: int = 120, r_D: float = 0.7) -> np.ndarray:
    """The paper's non-uniform radial grid (Fig. 8): spacing r_D / coarse (0.1) on
    [0, r_D] and (1 - r_D) / fine (0.0025) on [r_D, 1]: coarse + fine + 1 nodes."""
    return np.concatenate([np.linspace(0.0, r_D, coarse + 1)[:-1], np.linspace(r_D, 1.0, fine + 1)])


def runaway_3d(n=(161, 81, 65), N: int = 2000, T_max: float = 120.0, Q=(6, 6, 6),
               p_max: float = 50.0, seed: int = 20210414, dt: Optional[float] = None,
               r_D: float = 0.7, W: float = 1e-2, dp: float = 20.0, V0: float = 0.003,
               D0: float = 1e-4, xr: Optional[np.ndarray] = None,
               slope_rule: int = SLOPE_EQ15) -> Workload:
    """(p, xi, r) of Eq. 37-38 with E(t, r) = E_amp(t) (1 - r^2/2), seeded random-amplitude ramp.
    xr: radial nodes (default uniform, n[2] of them); radial_grid() gives the paper's
    piecewise-uniform grid."""
    xp = np.linspace(0.0, p_max, n[0])
    xx = np.linspace(-1.0, 1.0, n[1])
    xr = np.linspace(0.0, 1.0, n[2]) if xr is None else np.asarray(xr, dtype=np.float64)
    n = (n[0], n[1], len(xr))
    dt = T_max / N if dt is None else dt
    P, XI, R = np.meshgrid(xp, xx, xr, indexing="ij")
    P = P.reshape(-1)
    XI = XI.reshape(-1)
    R = R.reshape(-1)
    bp0, bpE, bx0, bxE, sp, sx = _runaway_parts(P, XI)
    shape_r = 1.0 - 0.5 * R * R
    bpE = bpE * shape_r
    bxE = bxE * shape_r
    th = np.tanh((R - r_D) / W)
    gp = np.exp(-(P / dp) ** 2)
    Drp = 0.5 * D0 * (1.0 + th) * gp
    dDr = 0.5 * D0 / W * (1.0 - th * th) * gp
    br = V0 * (R > r_D) + dDr
    sr = np.sqrt(2.0 * Drp)
    sig = np.ascontiguousarray(np.stack([sp, sx, sr]))
    J = P.size
    U = np.random.default_rng(seed).random(9)
    knots_t = np.arange(9) * 120.0 / 8.0
    knots_A = (0.1 + 0.5 * np.arange(9) / 8.0) * (1.0 + 0.25 * (2.0 * U - 1.0))

    def E_amp(t):
        return float(np.interp(t, knots_t, knots_A))

    def coeffs(nstep):
        E = E_amp(nstep * dt)
        b = np.empty((3, J))
        b[0] = bp0 + E * bpE
        b[1] = bx0 + E * bxE
        b[2] = br
        return b, sig

    kinds, vals = _faces([[FACE_ABSORB, FACE_ABSORB], [FACE_CLAMP, FACE_CLAMP],
                          [FACE_CLAMP, FACE_ABSORB]],
                         [[0.0, 1.0], [0.0, 0.0], [0.0, 0.0]])
    return Workload("cfg5_runaway_3d", (xp, xx, xr), dt, N, tuple(Q), kinds, vals, coeffs,
                    note="as cfg4 + radial row; r=0 clamp, r=1 absorb g=0; seeded E knots",
                    extra={"E_amp": E_amp, "parts": (bp0, bpE, bx0, bxE, br)},
                    slope_rule=slope_rule)


# --------------------------------------------------------------------------------------
# the paper's own 2-D example: cellular flow, periodic in x1 (Eq. 32-36)
# --------------------------------------------------------------------------------------
def cellular_periodic_2d(n=(129, 65), N: int = 100, T_max: float = 0.05, Q=(4, 4),
                         Pe: float = 10.0, eps: float = 0.15, omega: float = 2.0 * math.pi / 10.0,
                         cells: int = 2, dt: Optional[float] = None) -> Workload:
    """dx = Pe v(x, t) dt + dW on [-pi, pi] x [0, 1] with v of Eq. 33-35 (f = cos(omega t)),
    periodic in x1, P = 1 on x2 = 0 and x2 = 1 (Pe = 10, eps = 0.15,
    omega = 2 pi / 10, n = 2, T_max = 0.05).  The paper gives no grid or step count for this
    example in its text: 129 x 65 nodes and N = 100 are this repo's choice."""
    x0 = np.linspace(-math.pi, math.pi, n[0])
    x1 = np.linspace(0.0, 1.0, n[1])
    dt = T_max / N if dt is None else dt
    X, Y = np.meshgrid(x0, x1, indexing="ij")
    X = X.reshape(-1)
    Y = Y.reshape(-1)
    J = X.size
    snx, cnx = np.sin(cells * X), np.cos(cells * X)
    cpy, spy = np.cos(math.pi * Y), np.sin(math.pi * Y)
    # the last x1 node is the image of the first: give both exactly the same coefficients
    first = np.arange(J).reshape(n)[0]
    last = np.arange(J).reshape(n)[-1]
    sig = np.ones((2, J))

    def coeffs(nstep):
        f = math.cos(omega * nstep * dt)
        b = np.empty((2, J))
        b[0] = Pe * (-math.pi * cpy * (snx + eps * f * cnx))
        b[1] = Pe * (cells * spy * (cnx - eps * f * snx))
        b[:, last] = b[:, first]
        return b, sig

    kinds, vals = _faces([[FACE_PERIODIC, FACE_PERIODIC], [FACE_ABSORB, FACE_ABSORB]],
                         [[0.0, 0.0], [1.0, 1.0]])
    return Workload("cfg6_cellular_periodic_2d", (x0, x1), dt, N, tuple(Q), kinds, vals, coeffs,
                    note="paper's Eq. 33-36: Pe=10, eps=0.15, omega=2pi/10, n=2; periodic x1")


# --------------------------------------------------------------------------------------
# registry: full-size configs (BASELINE.json order) and reduced shapes for parity tests
# --------------------------------------------------------------------------------------
def runaway_3d_radial(**kw) -> Workload:
    """Config 5 on the paper's non-uniform radial grid (0.1 / 0.0025 spacing) with
    the weighted harmonic mean of ref [17]."""
    kw.setdefault("xr", radial_grid())
    kw.setdefault("slope_rule", SLOPE_WEIGHTED)
    wl = runaway_3d(**kw)
    wl.name = "cfg7_runaway_3d_radial"
    return wl


def config(idx: int, **kw) -> Workload:
    """BASELINE.json config `idx` in 1..5 at full size; keyword overrides shrink it.  6 and 7 are
    the SURVEY.md section 8(f) workloads: the paper's periodic cellular flow and the runaway
    problem on the paper's non-uniform radial grid."""
    return {1: brownian_1d, 2: ou_1d, 3: cellular_2d, 4: runaway_2d, 5: runaway_3d,
            6: cellular_periodic_2d, 7: runaway_3d_radial}[idx](**kw)


def small(idx: int) -> Workload:
    """Reduced shapes: same structure, several tiles and ragged tails, oracle-sized."""
    if idx == 1:
        return brownian_1d()
    if idx == 2:
        return ou_1d(nodes=259, N=45, dt=2.0 / 1000)
    if idx == 3:
        return cellular_2d(n=(71, 45), N=37, dt=4e-3)
    if idx == 4:
        return runaway_2d(n=(83, 47), N=33, dt=120.0 / 5000)
    if idx == 5:
        return runaway_3d(n=(37, 23, 19), N=19, dt=120.0 / 2000)
    if idx == 6:
        return cellular_periodic_2d(n=(41, 27), N=35, dt=0.05 / 100)
    if idx == 7:
        return runaway_3d_radial(n=(29, 19, 0), N=13, dt=120.0 / 2000, xr=radial_grid(3, 20))
    raise KeyError(idx)


def exit_everywhere(wl: Workload) -> Workload:
    """Copy of `wl` in which every ABSORB face is an exit face (g = 1).  The runaway configs exit
    only at p = p_max, so for any run the oracle can afford the field is still exactly
    0 at small p -- where the rows with the widest stencils live -- and a comparison there is 0 = 0.
    With p = 0 (and, in 3-D, r = 1) feeding 1 as well, those rows see non-zero data after a few steps.
    Same grid, coefficients and operators as `wl`; only chi and the absorbed constants change."""
    vals = np.array(wl.face_value, dtype=np.float64, copy=True)
    vals[np.asarray(wl.face_kind) == FACE_ABSORB] = 1.0
    return dataclasses.replace(wl, name=wl.name + "_exit_everywhere", face_value=vals)


def random_field(J: int, seed: int, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
    """Seeded rough field on the nodes: exercises the slope sign tests of Eq. 15."""
    return np.random.default_rng(seed).uniform(lo, hi, J)
