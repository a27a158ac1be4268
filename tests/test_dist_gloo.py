"""N>1 host logic on CPU: world_size-2 gloo run of the batch partition and the Welford merge."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2604_07248_b200 import shard


def test_partition_covers_batch():
    for B in (0, 1, 7, 32, 33):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                s, c = shard.partition(B, world, r)
                seen += list(range(s, s + c))
            assert seen == list(range(B))
            sizes = [shard.partition(B, world, r)[1] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_chan_merge_equals_single_pass():
    rng = np.random.default_rng(0)
    x = rng.random((11, 6, 6)) ** 2
    def acc(a):
        return a.shape[0], torch.from_numpy(a.mean(0)), torch.from_numpy(((a - a.mean(0)) ** 2).sum(0))
    n, m, s = shard.chan_merge(*acc(x[:4]), *acc(x[4:]))
    assert n == 11
    np.testing.assert_allclose(m.numpy(), x.mean(0), rtol=1e-12)
    np.testing.assert_allclose(s.numpy() / (n - 1), x.var(0, ddof=1), rtol=1e-11)
    n0, m0, s0 = shard.chan_merge(0, torch.zeros(6, 6), torch.zeros(6, 6), *acc(x))
    assert n0 == 11 and torch.equal(m0, acc(x)[1])


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(5)
    I = rng.random((9, 8, 8))                       # 9 "realisations" of an intensity map
    s, c = shard.partition(9, world, rank)
    mine = I[s:s + c]
    mean = torch.from_numpy(mine.mean(0))
    M2 = torch.from_numpy(((mine - mine.mean(0)) ** 2).sum(0))
    n, m, v = shard.merge_welford(c, mean, M2)
    rec = torch.full((c * 4,), rank, dtype=torch.uint8)[: 4 * min(c, 4)]
    rec = torch.full((16,), rank, dtype=torch.uint8)
    allrec = shard.gather_stats(rec)
    ok = (n == 9 and np.allclose(m.numpy(), I.mean(0), rtol=1e-12)
          and np.allclose(v.numpy() / 8, I.var(0, ddof=1), rtol=1e-11)
          and allrec.tolist() == [0] * 16 + [1] * 16)
    q.put((rank, bool(ok)))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo():
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
    assert res == [(0, True), (1, True)]
