"""World-size-2 CPU (gloo) test of the N > 1 path's host logic (tier framing 5).

The kernels cannot run here, so each rank forms its shard's partial sketch with the oracle (test
infrastructure) using the row range `shard_rows` hands it, the partials are summed with
`sharding.all_reduce_sketch` -- the call bench.py makes after every apply -- and the result must equal the
oracle's sketch of the whole matrix: this pins the row bookkeeping (ranges tile [0, m) exactly, the global
row index enters the hash).  The bench's timing rule (`sharding.max_over_ranks`: the slowest rank's time, the
same value on every rank) and its rank-0-only reporting are covered on the same two-rank group.
"""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_20195_b200.sharding import all_reduce_sketch, max_over_ranks, shard_rows  # noqa: E402


def test_shard_rows_tile_the_matrix_exactly():
    for m in (0, 1, 3, 4, 5, 4096, 4099, (1 << 20) + 7):
        for world in (1, 2, 3, 8):
            got = [shard_rows(m, world, r) for r in range(world)]
            assert got[0][0] == 0
            for (b0, n0), (b1, _) in zip(got, got[1:]):
                assert b0 + n0 == b1
            assert got[-1][0] + got[-1][1] == m
            assert all(b % 4 == 0 or n == 0 for b, n in got)
    with pytest.raises(ValueError):
        shard_rows(10, 2, 2)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, m: int, n: int, d: int, zeta: int, out_dir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        import workloads as wl

        seed = wl.sketch_seed(3)
        A = wl.gaussian(m, n, 11)                       # every rank generates the same matrix, keeps its rows
        begin, rows = shard_rows(m, world, rank)
        part = oracle.f64_sketch(seed, d, zeta, A[begin:begin + rows], row_begin=begin)
        t = torch.from_numpy(part)
        all_reduce_sketch(t, dist)
        # the bench's collective leg around it: every rank learns the slowest rank's time; only rank 0 reports
        slowest = max_over_ranks(10.0 + 5.0 * rank, dist)
        h16 = torch.full((8,), 1.0 + rank, dtype=torch.float16)
        all_reduce_sketch(h16, dist)                       # FP16 sketches are reduced in FP16
        np.save(os.path.join(out_dir, "leg%d.npy" % rank), np.array([slowest, float(h16[0])]))
        if rank == 0:
            np.save(os.path.join(out_dir, "sum.npy"), t.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_row_sharded_sketch_equals_whole(tmp_path):
    import oracle
    import workloads as wl

    m, n, d, zeta, world = 4099, 16, 32, 4, 2          # ragged: the last rank gets 2047 rows
    oracle.build()
    port = _free_port()
    mp.spawn(_worker, args=(world, port, m, n, d, zeta, str(tmp_path)), nprocs=world, join=True)
    got = np.load(tmp_path / "sum.npy")
    assert sorted(p.name for p in tmp_path.glob("sum*.npy")) == ["sum.npy"]          # one reporter
    for r in range(world):
        slowest, h = np.load(tmp_path / ("leg%d.npy" % r))
        assert slowest == 10.0 + 5.0 * (world - 1) and h == sum(1.0 + k for k in range(world))
    want = oracle.f64_sketch(wl.sketch_seed(3), d, zeta, wl.gaussian(m, n, 11))
    # F64 partial sums: equal up to the rounding order of the final scaling (each rank scales its partial)
    assert np.allclose(got, want, rtol=0, atol=1e-12 * np.abs(want).max())
    assert np.linalg.norm(got - want) <= 1e-14 * np.linalg.norm(want)


def test_collective_helpers_are_the_identity_without_a_process_group():
    t = torch.arange(6, dtype=torch.float32)
    assert all_reduce_sketch(t.clone()).equal(t)
    assert max_over_ranks(3.25) == 3.25
