"""Multi-GPU host logic on CPU: world_size-2 `gloo` processes.  The path has no data-path
collective (focal points are independent): ranks own disjoint focal slices, torch.distributed carries
only the barrier and the max / sum over ranks that bench.py uses for its timing."""
import os
import socket

import numpy as np
import pytest

from paper_2106_04649_b200 import configs, gen, shard


def test_focal_slices_partition_every_count():
    for nfoc in (1, 2, 7, 64, 256, 601):
        for world in (1, 2, 3, 4, 8):
            got = [i for r in range(world) for i in shard.focal_slice(nfoc, r, world)]
            assert got == list(range(nfoc))
            sizes = [len(shard.focal_slice(nfoc, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.focal_slice(4, 2, 2)


def test_replica_config_moves_the_focal_depth_only():
    cfg = configs.get(1)
    assert shard.replica_config(cfg, 0, 4) is cfg
    c2 = shard.replica_config(cfg, 2, 4)
    assert c2.focal == "single:850.0" and c2.n == cfg.n and c2.seed == cfg.seed and c2.A_R == cfg.A_R


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = configs.scaled(2, n=12, nt=64, nfoc=12, focal="line:300")
        mine = list(shard.focal_slice(cfg.nfoc, rank, world))
        gd, td = gen.first_arrivals(cfg, focs=mine)          # each rank generates only its own focal points
        dist.barrier()
        t_max = shard.max_over_ranks(10.0 + rank, dist)      # the max-over-ranks timing of bench.py
        n_sum = shard.sum_over_ranks(float(len(mine)), dist)
        q.put((rank, mine, float(gd.astype(np.float64).sum()), td.shape, t_max, n_sum))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_focal_sharding():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port, world = _free_port(), 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = configs.scaled(2, n=12, nt=64, nfoc=12, focal="line:300")
    gd_all, td_all = gen.first_arrivals(cfg)
    owned = []
    for rank, mine, gsum, tshape, t_max, n_sum in res:
        owned += mine
        assert tshape == (len(mine), cfg.n)
        assert gsum == float(gd_all[mine].astype(np.float64).sum())     # shards see the same bytes as the whole job
        assert t_max == 11.0 and n_sum == float(cfg.nfoc)
    assert owned == list(range(cfg.nfoc))


# ---------------------------------------------------------------- receiver-row sharding (section 8(e), NEXT-3)
def _row_worker(rank, world, port, q, n, nb, rpr, rf, nplanes):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ld = ((n + 15) // 16) * 16
        full = [_row_truth(p, nb, rpr * ld, rf) for p in range(nplanes)]
        mine = shard.row_slice(n, rank, world)
        planes = []
        for p in range(nplanes):                      # a rank starts with its own rows only (the rest is stale: -1)
            t = torch.full((nb, rpr * ld, rf), -1.0)
            t[:, rpr * mine.start:rpr * mine.stop] = full[p][:, rpr * mine.start:rpr * mine.stop]
            t[:, rpr * n:] = 0.0                      # pad rows are zero and must stay zero
            planes.append(t)
        shard.allgather_operand_rows(planes, rpr, n, rank, world, dist)
        # the exchange that bench.py --parallel rows uses (buffers allocated once, all_gather_into_tensor), driven twice on
        # a stand-in for the context: it must give the same planes
        again = []
        for p in range(nplanes):
            t = torch.full((nb, rpr * ld, rf), -1.0)
            t[:, rpr * mine.start:rpr * mine.stop] = full[p][:, rpr * mine.start:rpr * mine.stop]
            t[:, rpr * n:] = 0.0
            again.append(t)

        class FakeContext:
            nrec = n
            acked = 0

            def operand(self, slot):
                class V:
                    rows_per_rec = rpr
                return again, V

            def operand_exchanged(self, slot):
                self.acked += 1
        fake = FakeContext()
        exchange = shard.distributed_exchange(fake, dist)
        exchange(0)
        exchange(0)
        same = fake.acked == 2 and all(bool(torch.equal(a, b)) for a, b in zip(again, planes))
        ok = same and all(bool(torch.equal(planes[p][:, :rpr * n], full[p][:, :rpr * n])) and float(planes[p][:, rpr * n:].abs().max()) == 0.0
                 for p in range(nplanes))
        q.put((rank, ok))
    finally:
        dist.destroy_process_group()


def _row_truth(p, nb, rows, rf):
    import torch
    g = torch.Generator().manual_seed(1234 + p)
    return torch.randn((nb, rows, rf), generator=g)


def test_row_slices_partition():
    for n in (1, 5, 37, 601, 3901):
        for world in (1, 2, 3, 8):
            if world > n:
                continue
            got = [i for r in range(world) for i in shard.row_slice(n, r, world)]
            assert got == list(range(n))


@pytest.mark.parametrize("world,n,rpr,nplanes", [(2, 37, 1, 1), (3, 37, 2, 2)])
def test_gloo_allgather_of_operand_rows(world, n, rpr, nplanes):
    """The exchange step of the row-sharded path on CPU tensors: uneven row blocks, one- and two-plane operands
    (regimes 1/2 and the two-rows-per-receiver split operand of regime 3), pad rows untouched."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_row_worker, args=(r, world, port, q, n, 5, rpr, 12, nplanes)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(r, True) for r in range(world)]
