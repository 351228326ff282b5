"""The N>1 path on CPU (gloo, world_size 2): how bench.py deals row blocks to ranks and reduces the
per-rank figures.  The sweep itself has no collective (pairs are independent)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, k, stride, out):
    import torch
    import torch.distributed as dist
    import bench
    from oracle import famsa_oracle
    from paper_1603_06958_b200 import synth
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seqs, offsets = synth.family(0, k=k, seed=3)
    perm = famsa_oracle.sort_perm(offsets)
    lens = np.diff(offsets)[perm].astype(np.float64)
    prefix = np.concatenate([[0.0], np.cumsum(lens)])
    blocks = bench.rank_blocks(k, stride, rank)
    cells = sum(lens[i] * prefix[i] for a, b in blocks for i in range(a, b))
    pairs = sum(famsa_oracle.rows_pairs(a, b) for a, b in blocks)
    ms, cells_all, pairs_all = bench.reduce_over_ranks(dist, 10.0 + rank, cells, pairs, torch.device("cpu"))
    out.put((rank, blocks, cells, pairs, ms, cells_all, pairs_all))
    dist.barrier()
    dist.destroy_process_group()


def _gather_worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    k = 50
    rng = np.random.default_rng(100 + rank)
    m = 17 if rank == 0 else 49                                  # forests of different sizes, one of them full
    a = rng.integers(1, k, m).astype(np.int64); b = (a * rng.random(m)).astype(np.int64); w = rng.random(m).astype(np.float32)
    parts = bench.gather_forests(dist, a, b, w, k, torch.device("cpu"))
    out.put((rank, [(x.tolist(), y.tolist(), z.tolist()) for x, y, z in parts], (a.tolist(), b.tolist(), w.tolist())))
    dist.barrier()
    dist.destroy_process_group()


def test_gather_forests_gloo():
    """The one exchange step of the multi-GPU guide tree (bench.gather_forests): a padded all_gather."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_gather_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    mine = {r: own for r, _, own in res}
    for r, parts, _ in res:
        assert len(parts) == 2
        for src in range(2):
            assert tuple(parts[src]) == tuple(mine[src])         # every rank holds every rank's edges, unpadded


@pytest.mark.parametrize("stride", [2, 1])
def test_two_ranks_gloo(stride):
    import torch.multiprocessing as mp
    k, world = 5000, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000) + stride
    procs = [ctx.Process(target=_worker, args=(r, world, port, k, stride, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, b0, c0, p0, ms0, ca0, pa0), (_, b1, c1, p1, ms1, ca1, pa1) = res
    assert ms0 == ms1 == 11.0                                   # MAX over ranks
    assert ca0 == ca1 == pytest.approx(c0 + c1) and pa0 == pa1 == p0 + p1   # SUM over ranks
    if stride == 2:
        assert not set(b0) & set(b1)                             # disjoint batches ...
        rows = sorted(i for a, b in b0 + b1 for i in range(a, b))
        assert rows == list(range(k))                            # ... that together cover every row
        assert p0 + p1 == k * (k - 1) // 2
    else:
        assert b0 == b1 and b0[0][0] == 0 and b0[-1][1] == k     # replicas of the whole job


def test_step_blocks_cover():
    import bench
    k = 415519
    for stride in (1, 16):
        seen = []
        for off in range(stride):
            seen += bench.step_blocks(k, stride, offset=off)
        rows = sorted(seen)
        assert rows[0][0] == 0 and rows[-1][1] == k and len(rows) == (k + 1023) // 1024
        assert all(rows[n][1] == rows[n + 1][0] for n in range(len(rows) - 1))


def test_strong_scaling_deal():
    """--strong: the N=1 batch is dealt block by block; the ranks' batches partition it."""
    import bench
    k, stride = 415519, 16
    whole = bench.rank_blocks(k, stride, 0, 1, True)
    assert whole == bench.step_blocks(k, stride)
    parts = [bench.rank_blocks(k, stride, r, 4, True) for r in range(4)]
    assert sorted(b for p in parts for b in p) == sorted(whole)
    assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
