"""CPU oracle for the capture-range analysis of an exhaustive MI map -- TEST INFRASTRUCTURE, not
product code (same rules as oracle/__init__.py: only tests/, smoke() and bench.py's cpu_baseline leg
may import it; it shares nothing with the CUDA library).

What the paper does with its maps (section 3; section 3.1, Figs. 2-5):
"The gradient descent will see those MI results and try to register the image with the minimum
value it can reach"; the figures show "the paths the gradient descent algorithm will take", regions
"converging to the central point" and regions "converging to other points not related to our goal".
The paper drew those paths with an external viewer and prints no algorithm for them, so the
read-out is restated here in its exact, parameter-free, discrete form (reading A17):

* `map_gradient`  -- the finite-difference gradient field of the map in parameter units: central
  differences inside, one-sided differences on the faces (what `numpy.gradient(edge_order=1)`
  computes; pinned against it).
* `map_basins`    -- discrete steepest ascent (or descent) on the parameter grid: every node steps
  to its best neighbour (6- or 26-neighbourhood) while that neighbour is strictly better, until a
  local extremum is reached; label = that extremum, steps = moves taken; capture fraction = share
  of the cube whose path ends where the path of the target node (the ground truth, or the global
  extremum) ends -- the "central region converging to the central point" of Fig. 2a as a number.

Plain numpy, fp64, no blocking or reordering.  Maps are (n2, n1, n0) arrays, p0 fastest, linear
index t = (k2*n1 + k1)*n0 + k0 as in mi_map's map_out (one channel).

Pins (tests/test_oracle_analysis_pins.py): numpy.gradient; exact gradients of linear and quadratic
maps; a concave quadratic has one basin and steps = Chebyshev / Manhattan distance to the peak;
two peaks split the cube at the bisecting plane; brute force with independent Python loops on tiny
random maps; invariants (labels are fixed points, values never decrease along a path).
"""
from __future__ import annotations

import numpy as np


def map_gradient(m, lo, hi):
    """Gradient field (3, n2, n1, n0): component d is dM/dp_d in units of parameter d.
    Grid step h_d = (hi[d] - lo[d]) / (n[d] - 1) (mi_map's inclusive grid); an axis with one node
    has gradient 0.  Interior: (M[k+1] - M[k-1]) / (2 h); faces: (M[1] - M[0]) / h and
    (M[n-1] - M[n-2]) / h."""
    m = np.asarray(m, dtype=np.float64)
    assert m.ndim == 3
    g = np.zeros((3,) + m.shape, dtype=np.float64)
    for d, axis in ((0, 2), (1, 1), (2, 0)):          # parameter d lives on array axis 2 - d
        n = m.shape[axis]
        if n == 1:
            continue
        h = (float(hi[d]) - float(lo[d])) / (n - 1)
        mm = np.moveaxis(m, axis, 0)
        gg = np.moveaxis(g[d], axis, 0)               # a view: writes land in g[d]
        gg[1:-1] = (mm[2:] - mm[:-2]) / (2.0 * h)
        gg[0] = (mm[1] - mm[0]) / h
        gg[-1] = (mm[-1] - mm[-2]) / h
    return g


def neighbour_offsets(connectivity):
    """(dk2, dk1, dk0) of the neighbourhood in increasing linear-index order."""
    assert connectivity in (6, 26)
    offs = []
    for d2 in (-1, 0, 1):
        for d1 in (-1, 0, 1):
            for d0 in (-1, 0, 1):
                nz = (d2 != 0) + (d1 != 0) + (d0 != 0)
                if nz == 0 or (connectivity == 6 and nz != 1):
                    continue
                offs.append((d2, d1, d0))
    return offs


def next_pointer(m, direction=1, connectivity=26):
    """next[t] = the node t steps to: the neighbour with the largest direction*M if that is strictly
    larger than direction*M[t] (ties between neighbours: the lowest linear index), else t itself."""
    assert direction in (1, -1)
    v = direction * np.asarray(m, dtype=np.float64)
    n2, n1, n0 = v.shape
    idx = np.arange(v.size, dtype=np.int64).reshape(v.shape)
    best_v = v.copy()
    best_i = idx.copy()
    pv = np.full((n2 + 2, n1 + 2, n0 + 2), -np.inf)
    pv[1:-1, 1:-1, 1:-1] = v
    pi = np.full((n2 + 2, n1 + 2, n0 + 2), -1, dtype=np.int64)
    pi[1:-1, 1:-1, 1:-1] = idx
    for d2, d1, d0 in neighbour_offsets(connectivity):          # increasing linear index
        cv = pv[1 + d2:1 + d2 + n2, 1 + d1:1 + d1 + n1, 1 + d0:1 + d0 + n0]
        ci = pi[1 + d2:1 + d2 + n2, 1 + d1:1 + d1 + n1, 1 + d0:1 + d0 + n0]
        better = cv > best_v                                    # strict: earlier candidates keep ties
        best_v = np.where(better, cv, best_v)
        best_i = np.where(better, ci, best_i)
    return best_i.reshape(-1)


def map_basins(m, direction=1, connectivity=26, target=-1):
    """Follow next[] from every node to its fixed point.  Returns a dict: label (n2,n1,n0) int64 linear
    index of the extremum reached, steps (n2,n1,n0) int32 moves taken, n_extrema, target (the node
    used: `target`, or for -1 the global extremum, lowest index on ties), target_label, captured
    (nodes with label == target_label), capture_fraction."""
    m = np.asarray(m, dtype=np.float64)
    nxt = next_pointer(m, direction, connectivity)
    n = nxt.size
    cur = np.arange(n, dtype=np.int64)
    steps = np.zeros(n, dtype=np.int32)
    while True:
        nx = nxt[cur]
        moved = nx != cur
        if not moved.any():
            break
        steps += moved
        cur = nx
    if target < 0:
        target = int(np.argmax(direction * m.reshape(-1)))      # first maximum = lowest index
    assert 0 <= target < n
    tl = int(cur[target])
    captured = int((cur == tl).sum())
    return {"label": cur.reshape(m.shape), "steps": steps.reshape(m.shape),
            "n_extrema": int((nxt == np.arange(n)).sum()), "target": int(target), "target_label": tl,
            "captured": captured, "capture_fraction": captured / float(n), "max_steps": int(steps.max())}
