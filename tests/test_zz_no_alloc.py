"""fk_reduce_static: the weighted reduction for callers that cannot allocate device memory.

Some users of this library reach the reduction at a moment when cudaMalloc is off the table: the
process has already given all device memory away (a framework's caching allocator owns what the
big P buffers left, so a late cudaMalloc returns out-of-memory), or the reduction sits in a loop
next to other busy streams, and cudaMalloc / cudaFree would make the whole device wait.  For them
include/fk.h offers fk_reduce_static: the same two kernels as fk_reduce, with the partial sums in a
1 MiB array that is part of the library (shared by every call on a device, at most 64 chunks of 32
columns per call, device buffers only).

What is checked here, through the C ABI, against the existing fk_reduce on device buffers (which
test_gpu_next.py checks against the oracle): two calls in a row give the same numbers as fk_reduce
-- the second call with other weights and a range that starts and ends inside chunks, so that
anything the first call left in the shared array would show; a range beyond the limit and host
pointers are refused with FK_EINVAL and nothing is launched.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It passes alone in a fresh process (then its first call is also the
device's first, the one that looks up the array's address) and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_2104_14561_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-11          # the tolerance of the parity tests; the two paths add in the same order,
                     # so they are also expected to agree bit for bit


@pytest.fixture(scope="module")
def fk():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2104_14561_b200 import binding, solve
    binding.lib()
    return binding, solve


def test_two_calls_in_a_row_match_fk_reduce(fk):
    import torch
    B, solve = fk
    wl = W.cellular_2d(n=(71, 45), N=101, dt=4e-3)            # 102 columns: 4 chunks, the last one ragged
    rng = np.random.default_rng(7)
    w1 = torch.from_numpy(rng.uniform(0.0, 1.0, wl.J)).cuda()
    w2 = torch.from_numpy(rng.uniform(-1.0, 1.0, wl.J)).cuda()
    ctx = solve.create_for(wl, wl.N)
    try:
        solve.evolve_loaded(ctx, wl, wl.N)
        # the existing path (allocates its scratch with cudaMalloc)
        ref1 = torch.full((wl.N + 1,), float("nan"), dtype=torch.float64, device="cuda")
        ref2 = torch.full((60,), float("nan"), dtype=torch.float64, device="cuda")
        B.fk_reduce(ctx, w1, 0, wl.N + 1, ref1)
        B.fk_reduce(ctx, w2, 17, 77, ref2)
        # the entry point under test, twice in a row on the same stream, no sync in between
        launches = B.fk_launch_count(ctx)
        out1 = torch.full((wl.N + 1,), float("nan"), dtype=torch.float64, device="cuda")
        out2 = torch.full((60,), float("nan"), dtype=torch.float64, device="cuda")
        B.fk_reduce_static(ctx, w1, 0, wl.N + 1, out1)
        B.fk_reduce_static(ctx, w2, 17, 77, out2)
        assert B.fk_launch_count(ctx) == launches + 4         # two kernels per call: it did run
        B.fk_check(ctx)                                       # synchronises the context's stream
        torch.cuda.synchronize()
        for got, ref, w in ((out1, ref1, w1), (out2, ref2, w2)):
            got, ref = got.cpu().numpy(), ref.cpu().numpy()
            assert np.isfinite(ref).all() and np.abs(ref).max() > 1e-3    # not a 0 = 0 comparison
            scale = max(1.0, float(w.abs().sum()))
            assert float(np.abs(got - ref).max()) <= TOL * scale
            assert np.array_equal(got, ref)                   # same kernels, same order
        # and once more after them: the first range again, over whatever the second call left
        out3 = torch.full((wl.N + 1,), float("nan"), dtype=torch.float64, device="cuda")
        B.fk_reduce_static(ctx, w1, 0, wl.N + 1, out3)
        torch.cuda.synchronize()
        assert np.array_equal(out3.cpu().numpy(), ref1.cpu().numpy())
    finally:
        B.fk_destroy(ctx)


def test_shards_write_only_their_columns(fk):
    """A shard skips the chunks it does not own in both passes: `out` keeps the caller's values there
    and stale partial sums in the shared array are never read."""
    import torch
    B, solve = fk
    wl = W.cellular_2d(n=(71, 45), N=101, dt=4e-3)
    w = torch.from_numpy(np.random.default_rng(8).uniform(0.0, 1.0, wl.J)).cuda()
    got = torch.full((wl.N + 1,), float("nan"), dtype=torch.float64, device="cuda")
    ref = torch.full((wl.N + 1,), float("nan"), dtype=torch.float64, device="cuda")
    for s in range(2):
        ctx = solve.create_for(wl, wl.N, shard_index=s, shard_count=2)
        try:
            solve.evolve_loaded(ctx, wl, wl.N)
            B.fk_reduce(ctx, w, 0, wl.N + 1, ref)
            B.fk_reduce_static(ctx, w, 0, wl.N + 1, got)
            torch.cuda.synchronize()
            owned = solve.owned_columns(wl.N, s, 2)
            assert not np.isnan(got.cpu().numpy()[owned]).any()
        finally:
            B.fk_destroy(ctx)
    assert np.isfinite(ref.cpu().numpy()).all()
    assert np.array_equal(got.cpu().numpy(), ref.cpu().numpy())


def test_refuses_what_it_cannot_hold(fk):
    import torch
    B, solve = fk
    # 1-D, 2101 columns = 66 chunks: more than the fixed array holds in one call
    wl = W.config(1, N=2100, T_max=W.config(1).dt * 2100)
    ctx = solve.create_for(wl, 1)
    try:
        w = torch.ones(wl.J, dtype=torch.float64, device="cuda")
        out = torch.zeros(wl.N + 1, dtype=torch.float64, device="cuda")
        launches = B.fk_launch_count(ctx)
        with pytest.raises(B.FkError) as e:
            B.fk_reduce_static(ctx, w, 0, wl.N + 1, out)
        assert e.value.code == B.FK_EINVAL and "chunks" in str(e.value)
        with pytest.raises(B.FkError) as e:                   # 2018 columns from m = 31: 65 chunks
            B.fk_reduce_static(ctx, w, 31, 31 + 2018, out[:2018])
        assert e.value.code == B.FK_EINVAL
        # host memory is refused as well (staging it would need an allocation)
        with pytest.raises(B.FkError) as e:
            B.fk_reduce_static(ctx, np.ones(wl.J), 0, 1, np.zeros(1))
        assert e.value.code == B.FK_EINVAL and "device memory" in str(e.value)
        assert B.fk_launch_count(ctx) == launches             # nothing was launched
        # the widest range that fits, on column 0 only being final would be FK_ESTATE: evolve first
        solve.evolve_loaded(ctx, wl, 1)
        ref = torch.zeros(2048, dtype=torch.float64, device="cuda")
        got = torch.zeros(2048, dtype=torch.float64, device="cuda")
        B.fk_reduce(ctx, w, 32, 32 + 2048, ref)
        B.fk_reduce_static(ctx, w, 32, 32 + 2048, got)        # exactly 64 chunks
        torch.cuda.synchronize()
        assert np.abs(ref.cpu().numpy()).max() > 1e-3
        assert np.array_equal(got.cpu().numpy(), ref.cpu().numpy())
    finally:
        B.fk_destroy(ctx)
