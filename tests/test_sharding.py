"""`-m "not gpu"`: the N > 1 layout (contiguous proposal shards, no data-path collective) on CPU with gloo,
world_size 2.  The per-rank evaluation here is the oracle (tests may use it); what is under test is the host
logic of paper_1904_02863_b200/sharding.py: ranges, rank order, ragged sizes, the gather."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1904_02863_b200 import inputs
from paper_1904_02863_b200.sharding import gather_lnl, shard_range, shard_sizes


@pytest.mark.parametrize("n,world", [(0, 1), (1, 2), (7, 2), (8, 2), (4096, 8), (65537, 8), (5, 8)])
def test_shard_ranges_partition(n, world):
    edges = [shard_range(n, r, world) for r in range(world)]
    assert edges[0][0] == 0 and edges[-1][1] == n
    assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
    sizes = shard_sizes(n, world)
    assert sum(sizes) == n and max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def _worker(rank, world, port, n_prop, out_path):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    cfg = inputs.CONFIGS["C1"].reduced(f_max=40.0, batch=n_prop)
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    th = inputs.proposals(cfg)
    lo, hi = shard_range(n_prop, rank, world)
    lnl, _, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th[lo:hi], n_threads=1)
    full = gather_lnl(torch.from_numpy(lnl), n_prop)
    if rank == 0:
        ref, _, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, n_threads=1)
        np.save(out_path, np.stack([full.numpy(), ref]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_matches_unsharded(tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = str(tmp_path / "lnl.npy")
    mp.spawn(_worker, args=(2, port, 13, out), nprocs=2, join=True)
    got, ref = np.load(out)
    assert got.shape == (13,) and np.array_equal(got, ref)      # same arithmetic, same order: identical bits


# ---- bin sharding (NEXT-4 host logic) ----
def _bin_worker(rank, world, port, n_prop, out_path):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1904_02863_b200.sharding import bin_shard_edges, lnl_from_parts, reduce_parts_rank_ordered
    cfg = inputs.CONFIGS["C2"].reduced(f_max=22.0, batch=n_prop)          # 257 bins, long-signal shape
    f, S, dets = inputs.frequency_grid(cfg), inputs.psd(cfg), inputs.detectors(cfg)
    d = inputs.make_data(cfg, oracle.waveform)
    th = inputs.proposals(cfg)
    lo, hi = bin_shard_edges(cfg.n_bins, world)[rank]
    _, parts, _ = oracle.lnl(f[lo:hi], cfg.delta_f, d[:, lo:hi], S[:, lo:hi], dets, cfg.gmst, th, n_threads=1)
    total = reduce_parts_rank_ordered(torch.from_numpy(parts))
    lnl = lnl_from_parts(total)
    if rank == 0:
        ref, ref_parts, _ = oracle.lnl(f, cfg.delta_f, d, S, dets, cfg.gmst, th, n_threads=1)
        np.save(out_path, np.stack([lnl.numpy(), ref, (np.abs(total.numpy() - ref_parts)).max(axis=(1, 2)),
                                    np.abs(ref_parts).max(axis=(1, 2))]))
    dist.barrier()
    dist.destroy_process_group()


def test_bin_sharded_two_rank_gloo(tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = str(tmp_path / "bins.npy")
    mp.spawn(_bin_worker, args=(2, port, 5, out), nprocs=2, join=True)
    lnl, ref, perr, pmax = np.load(out)
    # the two half-band sums are added after, not inside, the compensated bin loop: equal up to rounding of the split
    assert np.all(perr <= 1e-13 * pmax)
    np.testing.assert_allclose(lnl, ref, rtol=0, atol=1e-12 * pmax.max())
