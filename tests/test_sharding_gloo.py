"""N > 1 host logic on CPU: grid sharding + gloo all-gather of map slabs (world_size 2 and 3).
The per-slab map function here is the ORACLE (allowed in tests); the GPU path plugs mi_map in."""
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

from paper_1909_10690_b200 import sharding as sh  # noqa: E402


def test_slab_bounds_cover_the_axis_exactly():
    for n2 in (1, 2, 5, 41):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                b, e = sh.slab_bounds(n2, r, world)
                assert 0 <= b <= e <= n2
                seen += list(range(b, e))
            assert seen == list(range(n2))
    with pytest.raises(ValueError):
        sh.slab_bounds(4, 2, 2)


def test_slab_range_is_a_node_range_of_the_whole_grid():
    n = (41, 41, 41)
    seen = []
    for r in range(4):
        begin, end = sh.slab_range(n, r, 4)
        assert begin[:2] == (0, 0) and end[:2] == (41, 41)
        assert (begin[2], end[2]) == sh.slab_bounds(41, r, 4)
        seen += list(range(begin[2], end[2]))
    assert seen == list(range(41))
    assert sh.slab_range((3, 3, 1), 1, 2) is None                  # more ranks than planes
    with pytest.raises(ValueError):
        sh.map_sharded(lambda b, e: None, n, 1, 0, 2, dist=None)    # world > 1 needs torch.distributed
    with pytest.raises(ValueError):
        sh.batch_sharded(lambda b, e: None, 10, 1, 0, 2, dist=None)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


# a grid whose step (2/6) is not representable: a slab whose interior nodes were re-derived from the slab's
# own end points would differ from the full grid by an ulp; node ranges of the whole grid cannot
GRID_N = 7
GRID_LO_HI = ((-1.0, -1.0, -1.0), (1.0, 1.0, 1.0))


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle as orc
    from paper_1909_10690_b200 import phantoms as ph
    cfg = ph.config_c1(grid_n=GRID_N)
    lo, hi = GRID_LO_HI

    def map_fn(begin, end):
        return orc.mi_map_range(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                                cfg.family, lo, hi, cfg.n, begin, end, q=cfg.q)

    full, am = sh.map_sharded(map_fn, cfg.n, 1 + len(cfg.q), rank, world, dist=dist)
    np.save(os.path.join(out_dir, "map_%d.npy" % rank), full.numpy())
    np.save(os.path.join(out_dir, "am_%d.npy" % rank), am.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_map_equals_single_rank_map_gloo(world, tmp_path):
    import oracle as orc
    from paper_1909_10690_b200 import phantoms as ph
    cfg = ph.config_c1(grid_n=GRID_N)
    lo, hi = GRID_LO_HI
    ref = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                     cfg.family, lo, hi, cfg.n, q=cfg.q)
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        m = np.load(tmp_path / ("map_%d.npy" % r))
        am = np.load(tmp_path / ("am_%d.npy" % r))
        assert m.shape == ref["map"].shape
        assert np.array_equal(m, ref["map"])                 # bit for bit: every rank's nodes are the full grid's
        assert np.array_equal(am, ref["argmax"])


# ------------------------------------------------------------------------------------------------ 12-DOF composite grid
def test_affine12_grid_is_the_3_to_the_12_product():
    d = np.arange(1, 13) * 0.01
    assert sh.affine12_count() == 531441
    mid = (3 ** 12 - 1) // 2
    assert np.array_equal(sh.affine12_grid(d, mid, mid + 1)[0], np.eye(3, 4))
    first, last = sh.affine12_grid(d, 0, 1)[0], sh.affine12_grid(d, 3 ** 12 - 1, 3 ** 12)[0]
    assert np.allclose(first, np.eye(3, 4) - d.reshape(3, 4)) and np.allclose(last, np.eye(3, 4) + d.reshape(3, 4))
    # entry k moves with period 3^k; a chunk equals the same rows of a bigger chunk
    T = sh.affine12_grid(d, 0, 3 ** 5)
    for k in range(5):
        col = T.reshape(-1, 12)[:, k] - np.eye(3, 4).reshape(12)[k]
        want = ((np.arange(3 ** 5) // 3 ** k) % 3 - 1) * d[k]
        assert np.allclose(col, want)
    assert np.array_equal(sh.affine12_grid(d, 100, 140), sh.affine12_grid(d, 0, 200)[100:140])
    assert len(np.unique(sh.affine12_grid(d, 0, 3 ** 6).reshape(-1, 12), axis=0)) == 3 ** 6


def _batch_worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n = 83

    def eval_fn(b, e):
        i = np.arange(b, e, dtype=np.float64)
        return np.stack([i * i, -i], axis=1)

    full = sh.batch_sharded(eval_fn, n, 2, rank, world, dist=dist)
    np.save(os.path.join(out_dir, "batch_%d.npy" % rank), full.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_batch_sharded_gathers_every_share_gloo(world, tmp_path):
    mp.spawn(_batch_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    i = np.arange(83, dtype=np.float64)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / ("batch_%d.npy" % r)), np.stack([i * i, -i], axis=1))
