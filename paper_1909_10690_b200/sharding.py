"""Multi-GPU plumbing for one exhaustive map: shard the parameter grid across ranks, gather the map.

Every map voxel is a separate MI evaluation, so the path shards by TRANSFORMS with no
exchange inside it: each rank owns a contiguous slab of the slowest grid axis (p2), holds both
volumes (<= 105 MB, replicated) in its own context, maps its slab with `mi_map_range` -- whose node
parameters are those of the WHOLE grid, so the sharded map equals the single-GPU map bit for bit --
and the slabs are concatenated with one all-gather of doubles (<= 551 KB at C5).  This module holds
host logic only (index arithmetic + torch.distributed calls); it never touches the method's
arithmetic, so it can be exercised with the gloo backend on CPU by passing any `map_fn`.
"""
from __future__ import annotations

import numpy as np


def axis_values(lo: float, hi: float, n: int) -> np.ndarray:
    """Grid values of include/mi.h: lo + k*(hi-lo)/(n-1) in double, n == 1 -> lo."""
    if n == 1:
        return np.array([lo], dtype=np.float64)
    return np.array([lo + k * (hi - lo) / (n - 1) for k in range(n)], dtype=np.float64)


def slab_bounds(n2: int, rank: int, world: int):
    """Contiguous [k_begin, k_end) slab of the p2 axis for `rank`; sizes differ by at most one."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    base, rem = divmod(int(n2), int(world))
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def slab_range(n, rank: int, world: int):
    """Node range (begin[3], end[3]) of the rank's p2 slab on the grid of n nodes, or None if the slab
    is empty (more ranks than p2 planes).  These are the `begin`, `end` arguments of mi_map_range."""
    n = [int(v) for v in n]
    b, e = slab_bounds(n[2], rank, world)
    if e <= b:
        return None
    return (0, 0, b), (n[0], n[1], e)


def map_sharded(map_fn, n, nch: int, rank: int, world: int, dist=None, device=None):
    """Run `map_fn(begin, end) -> array (nch, end[2]-begin[2], n1, n0)` on this rank's slab (the GPU
    path passes a closure over mi_map_range) and return the full (nch, n2, n1, n0) float64 map on
    every rank plus the per-channel arg max (ties -> lowest index).

    `dist` is `torch.distributed` (already initialised); it may be None only for world == 1."""
    import torch

    if world > 1 and dist is None:
        raise ValueError("map_sharded: world = %d needs an initialised torch.distributed" % world)
    n = [int(v) for v in n]
    sub = slab_range(n, rank, world)
    plane = n[1] * n[0]
    base = (n[2] + world - 1) // world           # padded slab depth so all_gather sees equal shapes
    local = torch.zeros((nch, base, n[1], n[0]), dtype=torch.float64, device=device)
    if sub is not None:
        depth = sub[1][2] - sub[0][2]
        m = map_fn(*sub)
        m = m if isinstance(m, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(m))
        local[:, :depth] = m.to(local.device).reshape(nch, depth, n[1], n[0])
    if world == 1:
        parts = [local]
    else:
        parts = [torch.empty_like(local) for _ in range(world)]
        dist.all_gather(parts, local)
    full = torch.empty((nch, n[2], n[1], n[0]), dtype=torch.float64, device=local.device)
    for r in range(len(parts)):
        b, e = slab_bounds(n[2], r, world)
        if e > b:
            full[:, b:e] = parts[r][:, : e - b]
    flat = full.reshape(nch, n[2] * plane)
    best = flat.max(dim=1, keepdim=True).values
    idx = torch.arange(flat.shape[1], device=flat.device).expand_as(flat)
    argmax = torch.where(flat == best, idx, torch.full_like(idx, flat.shape[1])).min(dim=1).values
    return full, argmax


# ---- composite grids over all 12 affine degrees of freedom ---------------------------
def affine12_count() -> int:
    return 3 ** 12


def affine12_grid(delta12, begin: int = 0, end: int | None = None) -> np.ndarray:
    """The paper's 12-dimensional exhaustive idea: "Using 12 dimensions and only 3 individual parameter
    (i.e. a minus parameter, a plus parameter and zero) in each dimension or direction we have
    3^12 = 531441" measurements.  Read literally on the 12 entries of the physical 3x4
    [A|t]: transform number i has entry k (row-major; k = 3, 7, 11 are the translations) equal to the
    identity's entry plus (digit_k(i) - 1) * delta12[k], where digit_k is the k-th base-3 digit of i
    (entry 0 fastest).  Returns transforms [begin, end) as an (end - begin, 3, 4) float64 array; the
    identity is number (3^12 - 1) / 2.  Host logic only: the matrices go to mi_eval_batch."""
    d = np.asarray(delta12, dtype=np.float64).reshape(12)
    end = affine12_count() if end is None else int(end)
    idx = np.arange(int(begin), end, dtype=np.int64)
    T = np.tile(np.eye(3, 4).reshape(1, 12), (idx.size, 1))
    for k in range(12):
        digit = (idx // 3 ** k) % 3
        T[:, k] += (digit - 1).astype(np.float64) * d[k]
    return T.reshape(-1, 3, 4)


def batch_bounds(n: int, rank: int, world: int):
    """Contiguous [begin, end) share of n independent transforms for `rank` (sizes differ by at most one)."""
    return slab_bounds(n, rank, world)


def batch_sharded(eval_fn, n: int, nch: int, rank: int, world: int, dist=None, device=None):
    """Evaluate transforms [0, n) split across ranks: `eval_fn(begin, end) -> (end - begin, nch)` values for
    this rank's share; returns the (n, nch) float64 result on every rank (one all-gather of doubles)."""
    import torch

    if world > 1 and dist is None:
        raise ValueError("batch_sharded: world = %d needs an initialised torch.distributed" % world)
    b, e = batch_bounds(n, rank, world)
    base = (int(n) + world - 1) // world
    local = torch.zeros((base, nch), dtype=torch.float64, device=device)
    if e > b:
        v = eval_fn(b, e)
        v = v if isinstance(v, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(v, dtype=np.float64))
        local[: e - b] = v.to(local.device).reshape(e - b, nch)
    if world == 1:
        parts = [local]
    else:
        parts = [torch.empty_like(local) for _ in range(world)]
        dist.all_gather(parts, local)
    full = torch.empty((int(n), nch), dtype=torch.float64, device=local.device)
    for r in range(len(parts)):
        rb, re = batch_bounds(n, r, world)
        if re > rb:
            full[rb:re] = parts[r][: re - rb]
    return full
