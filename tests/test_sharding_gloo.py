"""Host logic of the multi-GPU path on CPU: world_size = 2 over gloo (DESIGN.md
section 9).  Streams shard with no data-path collective: every rank creates the shard
(n_total, first, n_local) that paper_1204_6193_b200.sharding hands it; here the ranks' rows come
from the oracle's shard constructor (same rng_create_shard semantics), are gathered, and must
equal the rows of one unsharded generator.  The all-reduce(MAX) that bench.py applies to the
per-rank step time is exercised the same way."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_1204_6193_b200 import sharding  # noqa: E402
from paper_1204_6193_b200 import workloads as W  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n_per_rank: int, n: int):
    import oracle
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        for kind in (W.LCG64, W.LCG64_LEAPFROG, W.XORWOW, W.PHILOX4X32_10, W.XS1024W, W.PHILOX4X32_7, W.LCG32,
                     W.XS1024W_SKIP, W.LCG64_BOTH, W.LFIB521, W.LFIB1279, W.LCG32_LEAPFROG,
                     W.MWC, W.MWC_MULTI):
            # bench.py's weak-scaling layout (the lagged Fibonacci kinds come in 256-stream instances)
            per = 256 if kind in (W.LFIB521, W.LFIB1279) else n_per_rank
            n_total, first, n_local = sharding.weak_scaling_shard(rank, world, per)
            mine = oracle.Rng(kind, n_local, W.MASTER_SEED, first=first, n_total=n_total).fill_u32(n)
            parts = [torch.empty(n_local * n, dtype=torch.int64) for _ in range(world)]
            dist.all_gather(parts, torch.from_numpy(mine.astype(np.int64)))
            if rank == 0:
                whole = oracle.Rng(kind, n_total, W.MASTER_SEED).fill_u32(n)
                got = torch.cat(parts).numpy().astype(np.uint32)
                assert np.array_equal(got, whole), f"kind {kind}: gathered shards != unsharded rows"
            # strong-scaling layout with an uneven split (granule 32 keeps xs1024 instances whole)
            total = 32 * 7
            f2, m2 = sharding.shard_range(rank, world, total, granule=32)
            sizes = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
            dist.all_gather(sizes, torch.tensor([f2, m2]))
            if rank == 0:
                cover = sorted((int(t[0]), int(t[1])) for t in sizes)
                assert cover[0][0] == 0 and sum(m for _, m in cover) == total
                assert all(cover[i][0] + cover[i][1] == cover[i + 1][0] for i in range(world - 1))
                assert all(f % 32 == 0 and m % 32 == 0 for f, m in cover)
        # the timing reduction of bench.py: max over ranks
        t = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert float(t.item()) == float(world)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_over_gloo_reproduce_the_unsharded_streams():
    mp.spawn(_worker, args=(2, _free_port(), 64, 24), nprocs=2, join=True)


def _gpu_worker(rank: int, world: int, port: int, n_per_rank: int, n: int):
    """the PRODUCT's shards (rng_create_shard through the binding, kernels on cuda:0 shared by both ranks -- no
    rank's kernel waits for another's), gathered over gloo and compared with the unsharded oracle"""
    import oracle
    import paper_1204_6193_b200 as pkg
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        for kind in (W.LCG64, W.LCG64_LEAPFROG, W.XORWOW, W.PHILOX4X32_10, W.XS1024W, W.PHILOX4X32_7, W.LCG32,
                     W.XS1024W_SKIP, W.LCG64_BOTH, W.LFIB521, W.LFIB1279):
            per = 256 if kind in (W.LFIB521, W.LFIB1279) else n_per_rank
            n_total, first, n_local = sharding.weak_scaling_shard(rank, world, per)
            g = pkg.Rng(kind, n_local, W.MASTER_SEED, first=first, n_total=n_total)
            out = torch.empty(n_local * n, dtype=torch.int32, device="cuda")
            g.fill_u32(out, n)
            red = torch.empty(2 * n_local, dtype=torch.int32, device="cuda")
            g.draw_reduce(red, 7)
            g.close()
            parts = [torch.empty(n_local * n, dtype=torch.int32) for _ in range(world)]
            dist.all_gather(parts, out.cpu())
            reds = [torch.empty(2 * n_local, dtype=torch.int32) for _ in range(world)]
            dist.all_gather(reds, red.cpu())
            if rank == 0:
                o = oracle.Rng(kind, n_total, W.MASTER_SEED)
                assert np.array_equal(torch.cat(parts).numpy().view(np.uint32), o.fill_u32(n)), f"kind {kind}: fill"
                assert np.array_equal(torch.cat(reds).numpy().view(np.uint32), o.draw_reduce(7)), f"kind {kind}: draw"
        # bench.py's timing reduction on device-timed values
        t = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert float(t.item()) == float(world)
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
def test_two_ranks_of_product_shards_reproduce_the_unsharded_streams():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device (no CPU fallback exists)")
    from paper_1204_6193_b200 import build
    build.build()
    mp.spawn(_gpu_worker, args=(2, _free_port(), 2048 + 64, 40), nprocs=2, join=True)


def test_shard_range_properties():
    for world in (1, 2, 3, 8):
        for total in (32, 64, 32 * 9, 32 * 1000):
            cover = [sharding.shard_range(r, world, total, 32) for r in range(world)]
            assert cover[0][0] == 0 and sum(m for _, m in cover) == total
            assert max(m for _, m in cover) - min(m for _, m in cover) <= 32
    with pytest.raises(ValueError):
        sharding.shard_range(2, 2, 64)
    with pytest.raises(ValueError):
        sharding.shard_range(0, 2, 65, 32)
    assert sharding.weak_scaling_shard(3, 8, 1 << 20) == (8 << 20, 3 << 20, 1 << 20)
