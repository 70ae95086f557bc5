"""The column-ownership RULE only (solve.owned_columns), under torch.distributed (gloo, world_size 2)
on CPU: every column has exactly one owner and round-robin chunks balance the triangular work.  No
fk context is created here (there is no GPU on the CPU box): that fk_params.shard_* contexts
reproduce the unsharded run bit for bit, with no exchange, is checked on the GPU by
tests/test_gpu_next.py::test_column_shards_reproduce_the_unsharded_run (one process, every shard
in turn) and, for the reductions, by tests/test_zz_no_alloc.py."""
import os
import socket
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, N, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_2104_14561_b200 import solve
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        mine = solve.owned_columns(N, rank, world)
        mask = torch.zeros(N + 1, dtype=torch.int64)
        mask[mine] = 1
        dist.all_reduce(mask)                                 # test-side check only
        work = sum(mine)                                      # column m costs m applications
        out.put((rank, mask.tolist(), work, len(mine)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_partition_the_columns_and_balance_the_work():
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    N = 2000
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, N, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [1] * (N + 1)                          # every column owned exactly once
    w0, w1 = res[0][2], res[1][2]
    assert abs(w0 - w1) / (w0 + w1) < 0.02                     # round-robin chunks balance the triangle
