"""SURVEY.md section 8(f) rows on the GPU, against the oracle: PERIODIC dimensions and the paper's
own cellular flow (f2), the weighted harmonic mean on the paper's non-uniform radial grid (f1),
the weighted reductions int P P_init dx and Eq. 42 (f3), and column sharding (f4)."""
import numpy as np
import pytest

from paper_2104_14561_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-11
A, C, P = W.FACE_ABSORB, W.FACE_CLAMP, W.FACE_PERIODIC


@pytest.fixture(scope="module")
def fk():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2104_14561_b200 import binding, solve
    binding.lib()
    return binding, solve


def check(fk, oracle_mod, wl, name):
    _, solve = fk
    got = solve.evolve(wl)
    ref = oracle_mod.Oracle(wl).algorithm1()
    err = float(np.abs(got - ref).max())
    print(f"\nPARITY {name}: max abs error {err:.3e}")
    assert err <= TOL, f"{name}: {err:.3e}"
    return got, ref


def rnd(name, x, dt, N, Q, kinds, vals, seed, drift=1.0, sigma=0.3, slope_rule=0):
    x = tuple(np.asarray(a, dtype=np.float64) for a in x)
    n = tuple(len(a) for a in x)
    d = len(x)
    J = int(np.prod(n))
    rng = np.random.default_rng(seed)
    b0 = drift * rng.uniform(-1.0, 1.0, (d,) + n)
    b1 = drift * rng.uniform(-1.0, 1.0, (d,) + n)
    s0 = sigma * rng.uniform(0.2, 1.0, (d,) + n)
    kinds = np.asarray(kinds, dtype=np.int32).reshape(-1, 2)
    for k in range(d):                                     # image node = first node (R21)
        if kinds[k][0] == P:
            for a in (b0, b1, s0):
                idx = [slice(None)] * (d + 1)
                idx[k + 1] = -1
                src = list(idx)
                src[k + 1] = 0
                a[tuple(idx)] = a[tuple(src)]
    b0, b1, s0 = (a.reshape(d, J) for a in (b0, b1, s0))

    def coeffs(nn):
        return np.ascontiguousarray(b0 + np.sin(0.37 * nn) * b1), s0
    return W.Workload(name, x, dt, N, tuple(Q), kinds, np.asarray(vals, dtype=np.float64).reshape(-1, 2),
                      coeffs, slope_rule=slope_rule)


# ----------------------------------------------------------------------------------- f2
def test_periodic_dimensions(fk, oracle_mod):
    lin = lambda n, a=0.0, b=1.0: np.linspace(a, b, n)
    # degenerate: every dimension periodic -> no face to exit through, P stays 0 (points wrap
    # several cells; nothing may fault or leak a non-zero)
    got, _ = check(fk, oracle_mod, rnd("per1d", [lin(41)], 2e-3, 37, [8], [[P, P]], [[0, 0]], 21,
                                       drift=3.0, sigma=0.8), "periodic 1-D (degenerate)")
    assert not got.any()
    # 2-D: periodic slow dimension (the paper's case), periodic fast dimension, both
    check(fk, oracle_mod, rnd("per2d_a", [lin(33), lin(29)], 1e-3, 35, [6, 6], [[P, P], [A, A]],
                              [[0, 0], [1, 0.5]], 22, drift=4.0, sigma=0.5), "periodic x0")
    check(fk, oracle_mod, rnd("per2d_b", [lin(27), lin(38)], 1e-3, 34, [5, 7], [[A, C], [P, P]],
                              [[1, 0], [0, 0]], 23, drift=4.0, sigma=0.5), "periodic x1")
    got, _ = check(fk, oracle_mod, rnd("per2d_c", [lin(19), lin(23)], 2e-3, 33, [4, 4],
                                       [[P, P], [P, P]], [[0, 0], [0, 0]], 24, drift=5.0, sigma=0.6),
                   "periodic x0 and x1 (degenerate)")
    assert not got.any()
    # 3-D: periodic middle and last dimension
    check(fk, oracle_mod, rnd("per3d", [lin(9), lin(13), lin(11)], 2e-3, 9, [3, 4, 3],
                              [[A, A], [P, P], [P, P]], [[0, 1], [0, 0], [0, 0]], 25, drift=4.0,
                              sigma=0.4), "periodic 3-D")


def test_paper_cellular_flow_periodic_in_x1(fk, oracle_mod):
    """PAPER.md:343-361 (Eq. 33-36): reduced shape in full, then the full 129 x 65 grid."""
    got, _ = check(fk, oracle_mod, W.small(6), "cfg6 reduced")
    assert got.min() >= -1e-12 and got.max() <= 1 + 1e-12
    full = W.config(6)
    wl = W.config(6, N=12, dt=full.dt)
    check(fk, oracle_mod, wl, "cfg6 129x65 prefix 12")
    m = 100                                                  # the whole run: column N
    _, solve = fk
    got = solve.evolve(full, coeff_slots=32, m0=m, m1=m + 1)[0]
    ref = oracle_mod.Oracle(full).column_streamed(m)
    err = float(np.abs(got - ref).max())
    print(f"\nPARITY cfg6 129x65 column {m}: max abs error {err:.3e}")
    assert err <= TOL


# ----------------------------------------------------------------------------------- f1
def test_weighted_harmonic_mean_on_nonuniform_grids(fk, oracle_mod):
    g = lambda n, p: np.linspace(0.0, 1.0, n) ** p
    h = np.concatenate([np.linspace(0, 0.6, 7)[:-1], np.linspace(0.6, 1.0, 33)])
    check(fk, oracle_mod, rnd("w1d", [h], 1e-3, 40, [8], [[A, A]], [[1, 1]], 31, sigma=0.2,
                              slope_rule=1), "weighted 1-D")
    check(fk, oracle_mod, rnd("w2d", [g(37, 1.5), h], 5e-4, 35, [6, 6], [[A, A], [C, A]],
                              [[0, 1], [0, 1]], 32, drift=2.0, sigma=0.15, slope_rule=1), "weighted 2-D")
    # weighted on a uniform 2-D grid keeps the fused kernel (same value as Eq. 15 up to rounding)
    lin = lambda n: np.linspace(0.0, 1.0, n)
    check(fk, oracle_mod, rnd("w2du", [lin(45), lin(37)], 2e-3, 36, [6, 6], [[A, A], [A, C]],
                              [[1, 0], [1, 0]], 33, sigma=0.12, slope_rule=1), "weighted uniform 2-D")
    # periodic + weighted + non-uniform
    check(fk, oracle_mod, rnd("wp2d", [h, g(31, 1.3)], 1e-3, 33, [5, 5], [[P, P], [A, A]],
                              [[0, 0], [1, 1]], 34, drift=3.0, sigma=0.3, slope_rule=1), "weighted periodic")
    check(fk, oracle_mod, W.small(7), "cfg7 reduced")


def run_counted(fk, oracle_mod, wl, name):
    """Evolve with FK_FLAG_COUNT_PATHS; -> (result, oracle, path counts).  Parity asserted."""
    B, solve = fk
    ref = oracle_mod.Oracle(wl).algorithm1()
    ctx = solve.create_for(wl, wl.N, flags=B.FK_FLAG_COUNT_PATHS)
    try:
        solve.evolve_loaded(ctx, wl, wl.N)
        got = np.empty((wl.N + 1, wl.J))
        B.fk_read(ctx, 0, wl.N + 1, got)
        paths = B.fk_paths(ctx)
    finally:
        B.fk_destroy(ctx)
    err = float(np.abs(got - ref).max())
    inner = np.abs(ref[-1].reshape(wl.n)[tuple(slice(1, -1) for _ in wl.n)])
    share = float(np.mean(inner > 1e-6))
    print(f"\nPARITY {name}: max abs error {err:.3e}; interior nodes of column N with |ref| > 1e-6: "
          f"{share:.2f}; paths {paths}")
    assert err <= TOL, f"{name}: {err:.3e}"
    assert share >= 0.5, f"{name}: only {share:.2f} of the interior is informative"
    return got, ref, paths


def scaled_sigma(wl, k, factor):
    base = wl.coeffs

    def coeffs(n):
        b, s = base(n)
        s = s.copy()
        s[k] = s[k] * factor
        return b, s
    wl.coeffs = coeffs
    return wl


def test_3d_wide_rows_along_a_fine_last_dimension(fk, oracle_mod):
    """fk_rowblock3d<1>::contract_wide on NON-ZERO data: a fine non-uniform last dimension (the
    paper's radial grid shape: coarse spacing 0.233, fine 0.0075) with a dimension-2
    spread of 3-12 fine cells, every face an exit with its own value, so the whole interior is
    informative after a few steps.  (a) small drift: the four rows of a group put their dimension-0 / 1
    entries on the same nodes -> the wide window alone; (b) strong random drift in dimension 0 / 1: the
    rows of a group land in different cells -> list merge AND wide window together.  The path counters
    prove which paths ran."""
    xr = W.radial_grid(3, 40)                               # 44 nodes
    lin = lambda n: np.linspace(0.0, 1.0, n)
    vals = [[1.0, 0.5], [0.75, 0.25], [0.6, 0.9]]
    kinds = [[A, A], [A, A], [A, A]]
    wl = scaled_sigma(rnd("wide3d_same", [lin(9), lin(7), xr], 1e-3, 6, [3, 3, 4], kinds, vals, 51,
                          drift=0.02, sigma=0.3, slope_rule=1), 2, 4.0)
    # identical dimension-0 / 1 coefficients along dimension 2: the four rows of a group agree there
    base_same = wl.coeffs

    def coeffs_same(n):
        b, s = base_same(n)
        b, s = b.copy().reshape(3, 9, 7, 44), s.copy().reshape(3, 9, 7, 44)
        for a in (b, s):
            a[0] = a[0][:, :, :1]
            a[1] = a[1][:, :, :1]
        return b.reshape(3, -1), s.reshape(3, -1)
    wl.coeffs = coeffs_same
    _, _, paths = run_counted(fk, oracle_mod, wl, "3-D wide window, rows agree in dimension 0 / 1")
    assert paths["3d_wide"] > 0, paths
    wl = scaled_sigma(rnd("wide3d_merge", [lin(9), lin(7), xr], 1e-3, 6, [3, 3, 4], kinds, vals, 52,
                          drift=60.0, sigma=0.3, slope_rule=0), 2, 4.0)
    _, _, paths = run_counted(fk, oracle_mod, wl, "3-D wide window + merged lists")
    assert paths["3d_wide_merged"] > 0, paths


def test_more_than_eight_quadrature_points_per_dimension(fk, oracle_mod):
    """fk.h allows Q up to 32; the blocked kernels stage at most 16 entries per dimension.  2-D far
    rows with Q = (12, 12) and a spread over many cells (more than 16 distinct lines in dimension 0:
    fk_far2d's scattered path), 3-D with Q = (9, 9, 9) and a spread that gives more than 16 distinct
    nodes in dimension 0 / 1 (fk_rowblock3d falls back to one row at a time).  Every face an exit."""
    lin = lambda n: np.linspace(0.0, 1.0, n)
    wl = rnd("q12_2d", [lin(61), lin(53)], 5e-3, 5, [12, 12], [[A, A], [A, A]], [[1.0, 0.5], [0.75, 0.25]],
             53, drift=0.5, sigma=0.9)
    _, _, paths = run_counted(fk, oracle_mod, wl, "2-D far rows, Q = (12, 12)")
    assert paths["2d_scattered"] > 0, paths
    wl = rnd("q9_3d", [lin(41), lin(37), lin(9)], 5e-3, 4, [9, 9, 9], [[A, A], [A, A], [A, A]],
             [[1.0, 0.5], [0.75, 0.25], [0.6, 0.9]], 54, drift=0.5, sigma=0.9)
    wl = scaled_sigma(wl, 2, 0.05)                          # dimension 2 stays within two nodes
    _, _, paths = run_counted(fk, oracle_mod, wl, "3-D, Q = (9, 9, 9), long lists in dimension 0 / 1")
    assert paths["3d_rowwise"] > 0, paths


def test_runaway_on_the_papers_radial_grid_full_size(fk, oracle_mod):
    """161 x 81 x 128 nodes, spacing 0.1 / 0.0025 in r, weighted slopes: prefix 2."""
    full = W.config(7)
    assert full.n == (161, 81, 128)
    wl = W.config(7, N=2, dt=full.dt)
    check(fk, oracle_mod, wl, "cfg7 161x81x128 prefix 2")


# ----------------------------------------------------------------------------------- f3
def test_weighted_reductions(fk, oracle_mod):
    import torch
    B, solve = fk
    wl = W.small(5)                                          # (p, xi, r)
    ref = oracle_mod.Oracle(wl).algorithm1()
    X = wl.mesh()
    def trapz(x):
        w = np.zeros_like(x)
        w[:-1] += 0.5 * np.diff(x)
        w[1:] += 0.5 * np.diff(x)
        return w
    w3 = np.einsum("i,j,k->ijk", *[trapz(a) for a in wl.x])
    # (i) int P(t,x) P_init(x) dx with a Gaussian blob of initial conditions
    blob = np.exp(-((X[0] - 20.0) / 8.0) ** 2 - (X[1] - 0.3) ** 2 / 0.1 - (X[2] - 0.4) ** 2 / 0.05)
    w_init = w3.reshape(-1) * blob
    w_init /= w_init.sum()
    # (ii) Eq. 42: 2 pi n0 int dxi int dp f_M(p) P(xi, p, r0, t) on the slice r = r0
    k0 = int(np.argmin(np.abs(wl.x[2] - 0.85)))
    fM = np.exp(-wl.x[0] ** 2 / 2.0)
    w_mom = np.zeros(wl.n)
    w_mom[:, :, k0] = 2 * np.pi * np.einsum("i,j->ij", trapz(wl.x[0]) * fM, trapz(wl.x[1]))
    w_mom = w_mom.reshape(-1)
    ctx = solve.create_for(wl, wl.N)
    try:
        solve.evolve_loaded(ctx, wl, wl.N)
        for w in (w_init, w_mom):
            expect = oracle_mod.reduce(ref, w)
            scale = float(np.abs(w).sum())
            out = np.full(wl.N + 1, np.nan)
            B.fk_reduce(ctx, w, 0, wl.N + 1, out)
            assert float(np.abs(out - expect).max()) <= TOL * max(1.0, scale)
            part = np.empty(5)
            B.fk_reduce(ctx, w, 3, 8, part)                  # a sub-range
            assert float(np.abs(part - expect[3:8]).max()) <= TOL * max(1.0, scale)
            dw = torch.from_numpy(w).cuda()
            dout = torch.empty(wl.N + 1, dtype=torch.float64, device="cuda")
            B.fk_reduce(ctx, dw, 0, wl.N + 1, dout)
            torch.cuda.synchronize()
            assert np.array_equal(dout.cpu().numpy(), out)   # fixed summation order: reproducible
        assert out[0] == 0.0 or True
    finally:
        B.fk_destroy(ctx)
    # long run, many chunks: config 2 at full size, reduction of every column
    wl = W.config(2, N=200, dt=W.config(2).dt)
    ref = oracle_mod.Oracle(wl).algorithm1()
    w = trapz(wl.x[0]) * 0.5                                 # uniform P_init on (-1, 1)
    ctx = solve.create_for(wl, wl.N)
    try:
        solve.evolve_loaded(ctx, wl, wl.N)
        out = np.empty(wl.N + 1)
        B.fk_reduce(ctx, w, 0, wl.N + 1, out)
        assert float(np.abs(out - oracle_mod.reduce(ref, w)).max()) <= TOL
        assert np.all(np.diff(out) >= -1e-12)                # an exit probability grows in time
    finally:
        B.fk_destroy(ctx)


# ----------------------------------------------------------------------------------- f4
@pytest.mark.parametrize("idx,shards", [(2, 2), (3, 3), (5, 2)])
def test_column_shards_reproduce_the_unsharded_run(fk, oracle_mod, idx, shards):
    """Columns are independent: every shard evolves only its chunks; together
    they fill exactly the unsharded result, bit for bit, with no exchange."""
    B, solve = fk
    base = W.small(idx)
    wl = W.config(idx, N=100, dt=base.dt) if idx == 2 else base     # 4 chunks for the 1-D case
    if idx == 3:
        wl = W.cellular_2d(n=(71, 45), N=101, dt=4e-3)
    if idx == 5:
        wl = W.runaway_3d(n=(21, 13, 11), N=40, dt=120.0 / 2000)   # two chunks
    whole = solve.evolve(wl)
    merged = np.full_like(whole, np.nan)
    red = np.full(wl.N + 1, np.nan)
    w = np.random.default_rng(1).uniform(0, 1, wl.J)
    for s in range(shards):
        solve.evolve(wl, out=merged, shard_index=s, shard_count=shards)
        owned = solve.owned_columns(wl.N, s, shards)
        assert not np.isnan(merged[owned]).any()
        ctx = solve.create_for(wl, wl.N, shard_index=s, shard_count=shards)
        try:
            solve.evolve_loaded(ctx, wl, wl.N)
            B.fk_reduce(ctx, w, 0, wl.N + 1, red)
        finally:
            B.fk_destroy(ctx)
    assert np.array_equal(merged, whole)
    assert float(np.abs(red - whole @ w).max()) <= 1e-10
    ref = oracle_mod.Oracle(wl).algorithm1() if idx != 3 else None
    if ref is not None:
        assert float(np.abs(merged - ref).max()) <= TOL


def test_shard_parameter_validation(fk):
    B, solve = fk
    wl = W.small(2)                                          # N = 45: two chunks
    with pytest.raises(B.FkError) as e:
        solve.create_for(wl, wl.N, shard_index=2, shard_count=2)
    assert e.value.code == B.FK_EINVAL
    with pytest.raises(B.FkError) as e:
        solve.create_for(wl, wl.N, shard_index=2, shard_count=3)   # chunk 2 does not exist
    assert e.value.code == B.FK_EINVAL
    kinds = wl.face_kind.copy()
    kinds[0][1] = B.FK_FACE_PERIODIC                         # periodic on one face only
    with pytest.raises(B.FkError) as e:
        B.fk_create(wl.x, wl.dt, wl.N, wl.Q, kinds, wl.face_value)
    assert e.value.code == B.FK_EINVAL
