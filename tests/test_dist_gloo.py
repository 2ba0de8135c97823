"""N > 1 path on CPU: world_size-2 `gloo` processes exercising paper_2505_12414_b200.dist
(toy / event sharding, rank-ordered combine of the K+1 partial sums, gather of per-toy rows).
The per-shard sums come from the CPU oracle here (no GPU in this suite); on GPUs the same calls
take the shard sums from mf_nll_grad.  SURVEY.md §8(e)."""
import os
import socket

import numpy as np
import pytest

import mf_datagen as dg
from paper_2505_12414_b200 import dist as mfd


def test_shard_toys_partition():
    for n in (0, 1, 7, 4096, 4097):
        for world in (1, 2, 3, 8):
            blocks = [mfd.shard_toys(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and sum(c for _, c in blocks) == n
            for (f0, c0), (f1, _) in zip(blocks, blocks[1:]):
                assert f0 + c0 == f1
            assert max(c for _, c in blocks) - min(c for _, c in blocks) <= 1


def test_shard_events_whole_items():
    for n in (0, 1, 63, 64, 65, 10_000, 1_000_000):
        for world in (1, 2, 8):
            blocks = [mfd.shard_events(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and sum(c for _, c in blocks) == n
            for r, (f, c) in enumerate(blocks):
                assert f % 64 == 0 or c == 0
                if r + 1 < world and blocks[r + 1][1] > 0:
                    assert c % 64 == 0
                    assert f + c == blocks[r + 1][0]


def test_ordered_sum_is_compensated_and_propagates_inf():
    rows = np.array([[1e16, 1.0], [1.0, 1e-16], [-1e16, 1.0]])
    out = mfd.ordered_sum(rows)
    assert out[0] == 1.0 and out[1] == 2.0 + 1e-16
    bad = mfd.ordered_sum(np.array([[np.inf, np.nan], [1.0, 1.0]]))
    assert bad[0] == np.inf and np.isnan(bad[1])


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    import torch.distributed as dist

    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # (a) one dataset split by events: shard sums combined in rank order
        m = dg.gen_mass(10_000, seed=0)
        first, count = mfd.shard_events(m.size, rank, world)
        nll, g, _ = oracle.nll_grad(oracle.MASS, m[first:first + count], dg.MASS_START, dg.MASS_LO, dg.MASS_HI)
        total = mfd.combine_partials(np.concatenate([[nll], g]))
        # (b) toys split by toy: every rank evaluates its block, rows gathered in toy order
        T = 5
        toys = dg.gen_mass_toys(T, 500, first_seed=0)
        f, c = mfd.shard_toys(T, rank, world)
        rows = np.array([oracle.nll_grad(oracle.MASS, toys[t], dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI)[0]
                         for t in range(f, f + c)]).reshape(c, 1)
        allrows = mfd.gather_toy_rows(rows, T)
        q.put((rank, total, allrows[:, 0]))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_world_size_2_gloo():
    import torch.multiprocessing as mp

    import oracle
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=150) for _ in range(world)], key=lambda x: x[0])
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    # every rank holds bit-identical totals
    assert np.array_equal(got[0][1], got[1][1]) and np.array_equal(got[0][2], got[1][2])
    # and they are the unsharded oracle's values
    m = dg.gen_mass(10_000, seed=0)
    nll, g, _ = oracle.nll_grad(oracle.MASS, m, dg.MASS_START, dg.MASS_LO, dg.MASS_HI)
    ref = np.concatenate([[nll], g])
    assert np.all(np.abs(got[0][1] - ref) <= 1e-12 * (1 + np.abs(ref)))
    toys = dg.gen_mass_toys(5, 500, first_seed=0)
    for t in range(5):
        o = oracle.nll_grad(oracle.MASS, toys[t], dg.MASS_TRUTH, dg.MASS_LO, dg.MASS_HI)[0]
        assert got[0][2][t] == o
