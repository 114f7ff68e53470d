"""N > 1 path on CPU: world_size-2 (and 3) gloo process groups run the pixel-shard partition and the one
gradient all-reduce of paper_2410_01136_b200/sharding.py; each rank's per-shard numbers come from the ORACLE
restricted to its pixel range (tests may use the oracle), and the reduced result must equal the whole-map
oracle.  This covers the host-side logic of DESIGN.md section 9; the GPU kernels of a shard are covered by
tests/test_gpu_parity.py::test_pixel_shards_match_full_plan."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

from paper_2410_01136_b200 import sharding  # noqa: E402


def test_pixel_shards_cover_and_balance():
    for npix, world in ((768, 1), (768, 2), (768, 5), (12 * 256 * 256, 8), (5, 8)):
        sh = sharding.pixel_shards(npix, world)
        assert len(sh) == world and sh[0][0] == 0
        assert sum(c for _, c in sh) == npix
        for (b0, c0), (b1, _) in zip(sh, sh[1:]):
            assert b1 == b0 + c0
        counts = [c for _, c in sh]
        assert max(counts) - min(counts) <= 1
    assert sharding.shard_of(10, 2, 3) == (7, 3)
    with pytest.raises(ValueError):
        sharding.shard_of(10, 3, 3)
    assert [c for _, c in sharding.batch_shards(256, 8)] == [32] * 8
    assert [c for _, c in sharding.batch_shards(2, 4)] == [1, 1, 0, 0]


def test_strided_shards_cover_and_balance():
    for npix, world in ((768, 1), (768, 2), (768, 5), (12 * 256 * 256, 8), (5, 8)):
        seen = np.zeros(npix, dtype=np.int64)
        counts = []
        for r in range(world):
            begin, stride, count = sharding.strided_shard_of(npix, r, world)
            assert begin == r and stride == world
            if count:
                assert begin + (count - 1) * stride < npix
                seen[begin::stride][:count] += 1
            counts.append(count)
        assert np.all(seen == 1) and sum(counts) == npix and max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        sharding.strided_shard_of(10, 3, 3)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir, strided=False):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from harness import parity
        from harness import workloads as wl
        oracle.set_num_threads(2)
        w = wl.config(2).scaled(nside=4, n_los=64, batch=3)           # FULL16, batch 3, 192 pixels
        if strided:
            begin, stride, count = sharding.strided_shard_of(w.npix, rank, world)
            pix = begin + stride * np.arange(count)
        else:
            begin, count = sharding.shard_of(w.npix, rank, world)
            pix = np.arange(begin, begin + count)
        cots = w.cotangents()
        local = parity.oracle_forward(w, pix=pix)
        g_local = parity.oracle_vjp(w, tuple(np.ascontiguousarray(c[..., pix]) for c in cots), pix=pix)
        g = sharding.reduce_gradient(torch.from_numpy(g_local.copy()))
        if strided:   # the gradient is what the shards exchange; the maps stay interleaved on their ranks
            full_Q = torch.from_numpy(parity.oracle_forward(w)[1]) if rank == 0 else None
        else:
            full_Q = sharding.gather_maps(torch.from_numpy(local[1]), w.npix)
        if rank == 0:
            ref = parity.oracle_forward(w)
            g_ref = parity.oracle_vjp(w, cots)
            np.save(os.path.join(out_dir, "ok.npy"),
                    np.array([np.abs(g.numpy() - g_ref).max() / np.abs(g_ref).max(),
                              np.abs(full_Q.numpy() - ref[1]).max(), float(full_Q.shape[-1] == w.npix)]))
        # every rank must hold the same reduced gradient
        gs = [torch.empty_like(g) for _ in range(world)]
        dist.all_gather(gs, g)
        assert all(torch.equal(gs[0], x) for x in gs)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,strided", [(2, False), (3, False), (2, True), (3, True)])
def test_gloo_pixel_shards_reduce_to_the_full_gradient(world, strided, tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path), strided), nprocs=world, join=True)
    rel_g, dq, shape_ok = np.load(tmp_path / "ok.npy")
    assert rel_g < 1e-13          # float64 partial sums in a different order
    assert dq == 0.0 and shape_ok == 1.0


def _bench_worker(rank, world, port, out_dir):
    """bench.py's rank_workload: rank 0 is the config as stated, other ranks are distinct, seeded chains."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        from harness import workloads as wl
        w = bench.rank_workload(0, rank)
        t = torch.from_numpy(w.params.astype(np.float64).ravel().copy())
        ts = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(ts, t)
        if rank == 0:
            assert np.array_equal(w.params, wl.config(0).params)
            assert not torch.equal(ts[0], ts[1])
            assert torch.all((ts[1] / ts[0] - 1).abs() <= 0.05 + 1e-6)
        vals = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)                  # the bench's max-over-ranks timing reduction
        assert vals.item() == world
    finally:
        dist.destroy_process_group()


def test_gloo_bench_rank_workloads_are_distinct_chains(tmp_path):
    mp.spawn(_bench_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
