"""N>1 path on CPU: world_size-2 gloo.  Each rank integrates its shard of the Philox counter range (here with the
oracle standing in for the kernel: the host logic under test is the range split and the accumulator all-reduce)."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n_total, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_1305_0708_b200 import shard
    from oracle import integrate as oint, sm as osm
    dist.init_process_group('gloo', init_method='tcp://127.0.0.1:%d' % port, rank=rank, world_size=world)
    first, n = shard.shard_range(1000, n_total, rank, world)
    w, ok = oint.weights(2, 77, first, n, 500.0, osm.default_params())
    acc = shard.combine_acc(oint.accumulate(w, ok))
    if rank == 0:
        np.save(out, np.array(acc))
    dist.destroy_process_group()


def test_shard_ranges_cover_batch():
    from paper_1305_0708_b200 import shard
    for n, world in ((10, 3), (1 << 22, 8), (5, 8), (0, 2)):
        parts = [shard.shard_range(7, n, r, world) for r in range(world)]
        assert sum(p[1] for p in parts) == n
        pos = 7
        for s, m in parts:
            assert s == pos
            pos += m


def test_two_rank_integration_equals_single(tmp_path):
    from oracle import integrate as oint, sm as osm
    s = socket.socket()
    s.bind(('127.0.0.1', 0))
    port = s.getsockname()[1]
    s.close()
    n_total = 301
    out = str(tmp_path / 'acc.npy')
    mp.spawn(_worker, args=(2, port, n_total, out), nprocs=2, join=True)
    got = np.load(out)
    w, ok = oint.weights(2, 77, 1000, n_total, 500.0, osm.default_params())
    ref = oint.accumulate(w, ok)
    assert got[2] == n_total and got[3] == ref[3]
    assert abs(got[0] - ref[0]) <= 1e-13 * ref[0] and abs(got[1] - ref[1]) <= 1e-13 * ref[1]


def _grid_worker(rank, world, port, n_total, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_1305_0708_b200 import api, shard
    from oracle import integrate as oint, sm as osm, vegas
    dist.init_process_group('gloo', init_method='tcp://127.0.0.1:%d' % port, rank=rank, world_size=world)
    cfg, nb = 2, 16
    grid = vegas.uniform_grid(12, nb)
    for it in range(2):                      # two grid-optimisation steps, every rank on its shard of the counters
        first, n = shard.shard_range(it * n_total, n_total, rank, world)
        bins = np.zeros((n, 12), dtype=np.int64)
        w, ok = oint.weights(cfg, 77, first, n, 500.0, osm.default_params(), grid=grid, bins_out=bins)
        hist = shard.combine_hist(torch.from_numpy(vegas.accumulate(bins, w, nb)))
        g = torch.from_numpy(grid.copy())
        api.hg_grid_refine(hist, 1.0, g)     # host-only call of the library: no GPU needed
        grid = g.numpy()
    np.save(out % rank, grid)
    dist.destroy_process_group()


def test_two_rank_grid_optimisation_equals_single(tmp_path):
    """Sharded grid optimisation: histograms summed over the ranks (shard.combine_hist), then the same refinement on
    every rank: both ranks end with the grid a single process gets on the whole range."""
    from paper_1305_0708_b200 import build
    build.build()
    import torch
    from paper_1305_0708_b200 import api
    from oracle import integrate as oint, sm as osm, vegas
    s = socket.socket()
    s.bind(('127.0.0.1', 0))
    port = s.getsockname()[1]
    s.close()
    n_total = 601
    out = str(tmp_path / 'grid%d.npy')
    mp.spawn(_grid_worker, args=(2, port, n_total, out), nprocs=2, join=True)
    g0, g1 = np.load(out % 0), np.load(out % 1)
    assert np.array_equal(g0, g1)
    grid = vegas.uniform_grid(12, 16)
    for it in range(2):
        bins = np.zeros((n_total, 12), dtype=np.int64)
        w, ok = oint.weights(2, 77, it * n_total, n_total, 500.0, osm.default_params(), grid=grid, bins_out=bins)
        g = torch.from_numpy(grid.copy())
        api.hg_grid_refine(torch.from_numpy(vegas.accumulate(bins, w, 16)), 1.0, g)
        grid = g.numpy()
    assert np.allclose(g0, grid, rtol=0, atol=1e-12) and not np.allclose(grid, vegas.uniform_grid(12, 16), atol=1e-3)
