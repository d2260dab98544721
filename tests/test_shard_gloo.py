"""CPU, world_size 2, gloo: the N>1 host path of bench.py -- read sharding, gather of the per-read records and the
max-over-ranks of the timed region.  The per-rank "mapper" here is the oracle (no GPU in this test); what is checked is that
sharding + gathering reproduces the unsharded result read for read."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1403_2136_b200.shard import shard_bounds, shard_range  # noqa: E402


def test_shard_bounds_cover_exactly():
    for n in (0, 1, 2, 7, 100, 100_000, 1_000_003):
        for w in (1, 2, 3, 4, 8):
            b = shard_bounds(n, w)
            assert b[0] == 0 and b[-1] == n and len(b) == w + 1
            sizes = [b[i + 1] - b[i] for i in range(w)]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
            assert [shard_range(n, r, w) for r in range(w)] == list(zip(b[:-1], b[1:]))
    with pytest.raises(ValueError):
        shard_bounds(5, 0)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_reads, out_dir):
    import torch.distributed as dist
    import gen
    import oracle
    from paper_1403_2136_b200.shard import gather_records, max_over_ranks, shard_range as sr
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        genome = gen.make_genome(6000, 77)[0]
        r = gen.make_reads(genome, n_reads, 40, 78, sub_rate=0.1)
        lo, hi = sr(n_reads, rank, world)
        local = oracle.map_reads(genome, 500, -1, r["reads"][lo:hi], r["lens"][lo:hi], strands=3)
        full = gather_records(torch.from_numpy(local), n_reads)
        t = max_over_ranks(10.0 + rank)
        np.save(os.path.join(out_dir, f"full{rank}.npy"), full.numpy())
        np.save(os.path.join(out_dir, f"t{rank}.npy"), np.array([t]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_reads", [9, 10])
def test_sharded_map_equals_unsharded(tmp_path, oracle_mod, n_reads):
    import gen
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_reads, str(tmp_path)), nprocs=world, join=True)
    genome = gen.make_genome(6000, 77)[0]
    r = gen.make_reads(genome, n_reads, 40, 78, sub_rate=0.1)
    want = oracle_mod.map_reads(genome, 500, -1, r["reads"], r["lens"], strands=3)
    for rank in range(world):
        got = np.load(tmp_path / f"full{rank}.npy")
        assert got.shape == want.shape and (got == want).all()
        assert float(np.load(tmp_path / f"t{rank}.npy")[0]) == 11.0        # max over ranks of 10 + rank
