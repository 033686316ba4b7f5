"""The N = 2 data path of the row-sharded sketch minus the second GPU.

No box with two GPUs is available to this build, so the two shards of `sharding.shard_rows(m, 2, r)` are sketched on ONE
device into private sketches -- each with its global `row_begin`, exactly what rank r does -- rank 0's partial goes through
`sharding.all_reduce_sketch` on a real NCCL communicator (one rank: the collective call, its stream ordering and the
in-place result are exercised; the sum over ranks is the tensor add below), rank 1's partial is added, and the result must
equal the oracle's sketch of the whole matrix bit for bit (integer-valued input: every FP16 / FP32 sum is exact in any order).
"""
import socket

import numpy as np
import pytest

import oracle
import workloads as wl
from workloads import sketch_seed

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_row_shards_on_one_device_through_a_one_rank_nccl_all_reduce():
    import torch.distributed as dist

    import paper_2606_20195_b200 as ss
    from paper_2606_20195_b200.sharding import all_reduce_sketch, max_over_ranks, shard_rows

    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    m, n, d, zeta = 200003, 64, 128, 4            # ragged: the shards are 100004 and 99999 rows
    seed = sketch_seed(515)
    A = wl.integer_valued(m, n, 61)
    want = oracle.f64_sketch(seed, d, zeta, A, threads=8)
    assert np.abs(want).max() < 1024
    Ad = torch.from_numpy(A).cuda()
    sk = ss.Sketch(m, d, zeta, seed)
    shards = [shard_rows(m, 2, r) for r in range(2)]
    assert shards[0][0] == 0 and shards[0][1] + shards[1][1] == m and shards[1][0] == shards[0][1]
    own = not dist.is_initialized()
    if own:
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % _free_port(), rank=0, world_size=1,
                                device_id=torch.device("cuda", 0))
    try:
        for name in ("f16", "f32"):
            parts = []
            for rb, rows in shards:
                Ar = Ad[rb:rb + rows]
                assert sk.plan(n, f16=name == "f16", rows=rows, row_begin=rb)["variant"] == "tmem"      # the kernel bench.py times
                parts.append(sk.apply_f16acc(Ar, row_begin=rb, rows=rows) if name == "f16" else sk.apply_f32acc(Ar, row_begin=rb, rows=rows))
            # neither shard alone is the answer
            assert not np.array_equal(parts[0].float().cpu().numpy().astype(np.float64), want)
            total = all_reduce_sketch(parts[0], dist)            # NCCL, sketch dtype, in place
            assert total.data_ptr() == parts[0].data_ptr()
            total += parts[1]                                    # what the second rank's contribution adds in the reduction
            torch.cuda.synchronize()
            assert np.array_equal(total.float().cpu().numpy().astype(np.float64), want), name
        assert max_over_ranks(2.5, dist, torch.device("cuda", 0)) == 2.5
    finally:
        if own:
            dist.destroy_process_group()
        sk.close()
