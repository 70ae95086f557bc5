"""Edge cases and full-size checks of the CUDA path against the oracle (through the C ABI).

* degenerate shapes: minimal grids (3 nodes per dimension), Q = 1, N = 1, N a multiple of 32
* non-uniform tensor grids, in the fused 2-D kernel and in the generic kernels
* 2-D problems whose rows all leave the fused kernel's halo, or only some (mixed steps)
* BASELINE.json configs 2 and 3 at FULL size, in the launch configuration bench.py times:
  columns 0..N' of the full run are exactly the prefix problem N' (Eq. 29), which
  the oracle finishes in seconds; plus the invariants of P on sampled late columns.
"""
import numpy as np
import pytest

from paper_2104_14561_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-11
A, C = W.FACE_ABSORB, W.FACE_CLAMP


@pytest.fixture(scope="module")
def fk():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2104_14561_b200 import binding, solve
    binding.lib()
    return binding, solve


def make(name, x, dt, N, Q, kinds, vals, seed, drift=1.0, sigma=0.3, autonomous=False):
    """Seeded smooth-random coefficients on the grid `x` (inputs only)."""
    x = tuple(np.asarray(a, dtype=np.float64) for a in x)
    d = len(x)
    J = int(np.prod([len(a) for a in x]))
    rng = np.random.default_rng(seed)
    b0 = drift * rng.uniform(-1.0, 1.0, (d, J))
    b1 = drift * rng.uniform(-1.0, 1.0, (d, J))
    s0 = sigma * rng.uniform(0.2, 1.0, (d, J))

    def coeffs(n):
        f = 0.0 if autonomous else np.sin(0.37 * n)
        return np.ascontiguousarray(b0 + f * b1), s0

    return W.Workload(name, x, dt, N, tuple(Q), np.asarray(kinds, dtype=np.int32).reshape(-1, 2),
                      np.asarray(vals, dtype=np.float64).reshape(-1, 2), coeffs,
                      autonomous=autonomous)


def check(fk, oracle_mod, wl, tol=TOL):
    _, solve = fk
    got = solve.evolve(wl)
    ref = oracle_mod.Oracle(wl).algorithm1()
    assert got.shape == ref.shape
    err = float(np.abs(got - ref).max())
    assert err <= tol, f"{wl.name}: max abs error {err:.3e}"
    return got


def test_minimal_grids_and_orders(fk, oracle_mod):
    lin = lambda n: np.linspace(0.0, 1.0, n)
    check(fk, oracle_mod, make("min1d", [lin(3)], 0.01, 1, [1], [[A, A]], [[1, 0.5]], 1))
    check(fk, oracle_mod, make("min2d", [lin(3), lin(3)], 0.01, 33, [1, 2], [[A, A], [A, C]],
                               [[1, 0], [0.25, 0]], 2))
    check(fk, oracle_mod, make("min3d", [lin(3), lin(4), lin(3)], 0.02, 5, [2, 1, 3],
                               [[C, A], [A, A], [C, C]], [[0, 1], [0.5, 1], [0, 0]], 3))
    # N a multiple of 32: column N is the first lane of the last chunk
    check(fk, oracle_mod, make("n64", [lin(40), lin(21)], 2e-3, 64, [4, 4], [[A, A], [A, A]],
                               [[1, 1], [1, 1]], 4))


def test_nonuniform_grids(fk, oracle_mod):
    g = lambda n, p: np.linspace(0.0, 1.0, n) ** p           # graded towards 0
    h = np.concatenate([np.linspace(0, 0.6, 7)[:-1], np.linspace(0.6, 1.0, 33)])   # two spacings
    check(fk, oracle_mod, make("nu1d", [h], 1e-3, 40, [8], [[A, A]], [[1, 1]], 5, sigma=0.2))
    check(fk, oracle_mod, make("nu2d", [g(37, 1.5), h], 5e-4, 35, [6, 6], [[A, A], [C, A]],
                               [[0, 1], [0, 1]], 6, drift=2.0, sigma=0.15))
    check(fk, oracle_mod, make("nu3d", [g(9, 1.3), h[::3].copy(), g(11, 0.8)], 1e-3, 7, [3, 4, 3],
                               [[A, A], [C, C], [C, A]], [[0, 1], [0, 0], [0, 0.5]], 7))


def test_3d_odd_quadrature_sum_and_odd_last_dimension(fk, oracle_mod):
    """A row of the operator's offset table is 8 * sum(Q_k) bytes: with an odd sum(Q_k) every other
    row starts 8 bytes off a 16-byte boundary, which the L2 bulk prefetch of fk_rowblock3d (rows of
    the plane three steps ahead, so n0 > 3) must round (it needs a 16-byte aligned start and size).
    Odd n2 as well, so that group starts jb take both parities.  Every face value non-zero."""
    lin = lambda n: np.linspace(0.0, 1.0, n)
    for name, n, Q, seed in (("odd555", (9, 7, 13), (5, 5, 5), 21), ("odd665", (8, 6, 65), (6, 6, 5), 22),
                             ("odd311", (7, 5, 11), (3, 1, 1), 23)):
        wl = make(name, [lin(n[0]), lin(n[1]), lin(n[2])], 2e-3, 9, Q, [[A, A], [C, A], [C, A]],
                  [[0.5, 1.0], [0.0, 0.75], [0.0, 0.25]], seed, drift=1.0, sigma=0.1)
        got = check(fk, oracle_mod, wl)
        assert float(np.abs(got[-1].reshape(n)[1:-1, 1:-1, 1:-1]).max()) > 1e-3   # informative


def test_2d_far_rows_only_and_mixed(fk, oracle_mod):
    lin = lambda n: np.linspace(-1.0, 1.0, n)
    # sigma sqrt(2 dt) a_max ~ 14 cells: every row leaves the 2-node halo -> generic kernels only
    check(fk, oracle_mod, make("far2d", [lin(41), lin(53)], 0.02, 34, [8, 8], [[A, A], [C, C]],
                               [[1, 0], [0, 0]], 8, drift=0.5, sigma=0.8))
    # reach grows with the node index: near rows (fused) and far rows (generic) in every step
    wl = make("mix2d", [lin(61), lin(49)], 4e-3, 36, [6, 8], [[A, A], [A, C]], [[1, 1], [0, 0]], 9,
              drift=1.5, sigma=0.05)
    j1 = np.tile(np.arange(49), 61)
    scale = 1.0 + 12.0 * (j1 / 48.0) ** 2
    base = wl.coeffs

    def coeffs(n):
        b, s = base(n)
        s = s.copy()
        s[1] *= scale
        return b, s
    wl.coeffs = coeffs
    check(fk, oracle_mod, wl)


def test_2d_far_rows_beyond_node_32768_of_dimension_1(fk, oracle_mod):
    """fk_assemble packs a far row's first and last dimension-1 node into one int (16 bits each): with
    more than 32768 nodes along dimension 1 the last node reaches the sign bit and must be unpacked
    unsigned, or fk_far2d sees an empty window and returns c_j alone.  Reach of 3-14 cells (banded and
    scattered groups), a box so thin in dimension 0 that its faces feed every node: no 0 = 0 compare."""
    B, solve = fk
    n1 = 40001
    wl = make("wide_n1", [np.linspace(0.0, 3e-4, 4), np.linspace(-1.0, 1.0, n1)], 1e-6, 3, [2, 4],
              [[A, A], [A, A]], [[1.0, 0.5], [0.25, 1.0]], 31, drift=1.0, sigma=0.3)
    ref = oracle_mod.Oracle(wl).algorithm1()
    ctx = solve.create_for(wl, wl.N)
    try:
        B.fk_profile(ctx, True)
        solve.evolve_loaded(ctx, wl, wl.N)
        got = np.empty((wl.N + 1, wl.J))
        B.fk_read(ctx, 0, wl.N + 1, got)
        prof = B.fk_profile_read(ctx)
    finally:
        B.fk_destroy(ctx)
    assert prof["far2d"][1] == wl.N, prof
    high = ref[-1].reshape(4, n1)[1:3, 32768:-1]             # updated rows beyond node 32768
    assert float(np.mean(np.abs(high) > 1e-3)) > 0.9         # informative
    err = float(np.abs(got - ref).max())
    assert err <= TOL, f"{wl.name}: max abs error {err:.3e}"


def test_reset_straight_after_a_failed_evolve(fk):
    """fk_reset without a sync after an fk_evolve that raised the device's error flag: the refresh
    of the host copy queued by that fk_evolve must not land after the reset cleared it."""
    B, solve = fk
    wl = W.small(3)
    b, s = wl.coeff_table(0, wl.N)
    s_bad = s.copy()
    s_bad[3, 0, wl.J // 2 + 1] = -0.1
    for _ in range(3):
        ctx = solve.create_for(wl, wl.N)
        try:
            B.fk_set_coeffs_range(ctx, 0, wl.N, b, s_bad)
            B.fk_evolve(ctx, wl.N, 0)                        # queued; raises the flag on the device
            B.fk_reset(ctx)                                  # no fk_check / sync in between
            B.fk_set_coeffs_range(ctx, 0, wl.N, b, s)
            B.fk_evolve(ctx, wl.N, 0)
            B.fk_evolve(ctx, 0, 0)                           # entry check only
            out = np.empty((1, wl.J))
            B.fk_read(ctx, wl.N, wl.N + 1, out)
            B.fk_check(ctx)
        finally:
            B.fk_destroy(ctx)


def test_two_multistep_contexts_with_different_lines(fk, oracle_mod):
    """fk_line1d's dynamic shared-memory limit is a per-function attribute, shared by every context:
    a second FK_FLAG_MULTISTEP context with a shorter line must not break launches of the first."""
    B, solve = fk
    long_wl = W.config(2, N=40, dt=W.config(2).dt)           # J = 1025: 197 KB of shared memory
    short_wl = W.small(1)                                    # J = 201
    ref = oracle_mod.Oracle(long_wl).algorithm1()
    a = solve.create_for(long_wl, long_wl.N, flags=B.FK_FLAG_MULTISTEP)
    try:
        b = solve.create_for(short_wl, 1, flags=B.FK_FLAG_MULTISTEP)
        try:
            B.fk_profile(a, True)
            solve.evolve_loaded(b, short_wl, 1)
            solve.evolve_loaded(a, long_wl, long_wl.N)
            got = np.empty((long_wl.N + 1, long_wl.J))
            B.fk_read(a, 0, long_wl.N + 1, got)
            assert B.fk_profile_read(a)["line1d"][1] > 0
        finally:
            B.fk_destroy(b)
    finally:
        B.fk_destroy(a)
    assert float(np.abs(got - ref).max()) <= TOL


def test_2d_lines_handed_over_at_either_end(fk, oracle_mod):
    """The per-step plan (fk_api.cu plan_2d) gives the lines at either end of dimension 0 on which
    at least half of the rows are far to fk_far2d whole and runs the fused kernel on the rest: reach
    that grows towards the LAST lines (suffix hand-over), towards both ends, and a CLAMP face in
    dimension 0 (the first line is updated, not Dirichlet).  All kernels must run, result vs oracle."""
    B, solve = fk
    lin = lambda n: np.linspace(-1.0, 1.0, n)
    for name, kinds, shape in (("top", [[A, A], [A, C]], lambda t: t ** 3),
                               ("both", [[C, A], [C, C]], lambda t: (2 * t - 1) ** 4)):
        wl = make("plan_" + name, [lin(57), lin(45)], 4e-3, 35, [6, 8], kinds, [[1, 0], [0, 1]], 41,
                  drift=1.0, sigma=0.05)
        j0 = np.repeat(np.arange(57), 45)
        scale = 1.0 + 14.0 * shape(j0 / 56.0)
        base = wl.coeffs

        def coeffs(n, base=base, scale=scale):
            b, s = base(n)
            s = s.copy()
            s[1] *= scale
            return b, s
        wl.coeffs = coeffs
        ref = oracle_mod.Oracle(wl).algorithm1()
        ctx = solve.create_for(wl, wl.N)
        try:
            B.fk_profile(ctx, True)
            solve.evolve_loaded(ctx, wl, wl.N)
            got = np.empty((wl.N + 1, wl.J))
            B.fk_read(ctx, 0, wl.N + 1, got)
            prof = B.fk_profile_read(ctx)
            upd = B.fk_profile_updates(ctx)
        finally:
            B.fk_destroy(ctx)
        assert prof["fused"][1] == wl.N and prof["far2d"][1] == wl.N, prof
        # every updated row is owned by exactly one of the two kernels
        n_upd = (57 - (kinds[0][0] == A) - (kinds[0][1] == A)) * (45 - (kinds[1][0] == A) - (kinds[1][1] == A))
        assert upd["fused"] + upd["far2d"] == pytest.approx(n_upd * wl.N * (wl.N + 1) / 2)
        assert upd["far2d"] > 0.05 * upd["fused"]
        err = float(np.abs(got - ref).max())
        assert err <= TOL, f"{wl.name}: max abs error {err:.3e}"


@pytest.mark.parametrize("idx,nprefix", [(2, 24), (3, 12)])
def test_full_size_config_prefix_and_invariants(fk, oracle_mod, idx, nprefix):
    import torch
    B, solve = fk
    wl = W.config(idx)
    ref = oracle_mod.Oracle(wl).algorithm1(nprefix)          # columns 0..nprefix of the full run
    ctx = solve.create_for(wl, wl.N)
    try:
        solve.evolve_loaded(ctx, wl, wl.N)                   # the launches bench.py times
        got = np.empty((nprefix + 1, wl.J))
        B.fk_read(ctx, 0, nprefix + 1, got)
        err = float(np.abs(got - ref).max())
        assert err <= TOL, f"config {idx} full size, columns 0..{nprefix}: {err:.3e}"
        # invariants on late columns: 0 <= P <= 1, non-decreasing in t,
        # P = 1 on the absorbing faces (all faces of configs 2 and 3)
        cols = sorted({wl.N // 2, wl.N // 2 + 1, wl.N - 1, wl.N})
        late = np.empty((2, wl.J))
        for m in (cols[0], cols[2]):
            B.fk_read(ctx, m, m + 2, late)
            assert late.min() >= -1e-12 and late.max() <= 1.0 + 1e-12
            # monotonicity in t is a property of the exact P, not a theorem for the scheme in
            # multi-D (slope weights can be negative): loose bound, worst value printed
            worst = float((late[1] - late[0]).min())
            print(f"config {idx}: min over nodes of P(t_{m + 1}) - P(t_{m}) = {worst:.3e}")
            assert worst >= -1e-6
            grid = late[1].reshape(wl.n)
            for k in range(wl.d):
                assert np.all(np.take(grid, 0, axis=k) == 1.0)
                assert np.all(np.take(grid, -1, axis=k) == 1.0)
    finally:
        B.fk_destroy(ctx)


def test_negative_sigma_and_nonfinite_coefficients_are_reported(fk):
    """negative sigma is FK_EINVAL; NaN / Inf only with the validate flag."""
    B, solve = fk
    for idx in (2, 3, 5):                                   # 1-D, 2-D (fused kernel), 3-D
        wl = W.small(idx)
        b, s = wl.coeff_table(0, wl.N)
        interior = wl.J // 2 + 1                            # not on a face in any of the shapes
        # (1) negative sigma at an updated node of one step
        s_bad = s.copy()
        s_bad[3, 0, interior] = -0.1
        ctx = solve.create_for(wl, wl.N)
        try:
            B.fk_set_coeffs_range(ctx, 0, wl.N, b, s_bad)
            B.fk_evolve(ctx, wl.N, 0)                       # queued; the flag is raised on the device
            with pytest.raises(B.FkError) as e:
                B.fk_check(ctx)
            assert e.value.code == B.FK_EINVAL and "negative sigma" in str(e.value)
            with pytest.raises(B.FkError) as e:
                B.fk_read(ctx, 0, wl.N + 1, np.empty((wl.N + 1, wl.J)))
            assert e.value.code == B.FK_EINVAL
            # good coefficients + fk_reset clear it
            B.fk_reset(ctx)
            B.fk_set_coeffs_range(ctx, 0, wl.N, b, s)
            B.fk_evolve(ctx, wl.N, 0)
            B.fk_check(ctx)
        finally:
            B.fk_destroy(ctx)
        # (2) a negative sigma on a Dirichlet node is never read
        s_ok = s.copy()
        s_ok[:, :, 0] = -1.0                                # node 0 lies on an ABSORB face in all three
        ctx = solve.create_for(wl, wl.N)
        try:
            B.fk_set_coeffs_range(ctx, 0, wl.N, b, s_ok)
            B.fk_evolve(ctx, wl.N, 0)
            B.fk_check(ctx)
        finally:
            B.fk_destroy(ctx)
        # (3) NaN drift: reported only with FK_FLAG_VALIDATE
        b_nan = b.copy()
        b_nan[1, 0, interior] = np.nan
        for flags, raises in ((B.FK_FLAG_VALIDATE, True), (0, False)):
            ctx = solve.create_for(wl, wl.N, flags=flags)
            try:
                B.fk_set_coeffs_range(ctx, 0, wl.N, b_nan, s)
                B.fk_evolve(ctx, wl.N, 0)
                if raises:
                    with pytest.raises(B.FkError) as e:
                        B.fk_check(ctx)
                    assert e.value.code == B.FK_EINVAL and "NaN" in str(e.value)
                else:
                    B.fk_check(ctx)
            finally:
                B.fk_destroy(ctx)


def test_results_do_not_depend_on_what_freed_device_memory_held(fk, oracle_mod):
    """Operator buffers come from plain cudaMalloc: poison freed device memory with NaN patterns
    first; Dirichlet rows (g != 1 faces) and every padded slot must still be exact."""
    import torch
    lin = lambda n: np.linspace(0.0, 1.0, n)
    wl = make("poison2d", [lin(45), lin(37)], 2e-3, 40, [6, 6], [[A, A], [A, C]],
              [[0.25, 0.75], [0.5, 0]], 11, drift=1.0, sigma=0.12)
    ref = oracle_mod.Oracle(wl).algorithm1()
    _, solve = fk
    for _ in range(2):
        junk = torch.full((96 << 20,), float("nan"), dtype=torch.float64, device="cuda")   # 768 MB
        torch.cuda.synchronize()
        del junk
        torch.cuda.empty_cache()                            # hand the pages back to the driver
        got = solve.evolve(wl)
        assert np.isfinite(got).all()
        assert float(np.abs(got - ref).max()) <= TOL
