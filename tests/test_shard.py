"""Multi-rank host logic on CPU: two gloo processes (no GPU, no data-path collective exists)."""
import os
import socket

import numpy as np
import pytest

from paper_2005_11468_b200 import shard, synth


def test_reactor_ranges_partition_the_batch():
    for n in (0, 1, 7, 64, 65536, 65537):
        for world in (1, 2, 3, 8):
            r = [shard.reactor_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.reactor_range(10, 2, 2)


def test_rank_state_seeds_are_distinct_and_rank0_is_the_single_gpu_workload():
    assert shard.state_seed(1, 0) == 2001
    seeds = {shard.state_seed(c, r) for c in range(5) for r in range(8)}
    assert len(seeds) == 40
    mech, b0 = synth.make_config("C1", 16)
    b1 = synth.make_states(mech.n_species, 16, seed=shard.state_seed(1, 1), **synth.CONFIGS["C1"]["state"])
    assert not np.array_equal(b0.T, b1.T) and b0.Y.shape == b1.Y.shape


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
        mx = shard.max_over_ranks(ms)
        lo, hi = shard.reactor_range(1001, rank, world)
        out.put((rank, mx, lo, hi, shard.whole_job_rate(100, 4, mx, world)))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_agree_on_the_max_time_and_cover_the_batch():
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]                       # both ranks hold the max
    assert (res[0][2], res[0][3], res[1][2], res[1][3]) == (0, 501, 501, 1001)
    assert res[0][4] == res[1][4] == pytest.approx(2 * 100 * 4 / 15e-3)


def test_max_over_ranks_without_a_process_group_is_the_identity():
    assert shard.max_over_ranks(3.5) == 3.5
