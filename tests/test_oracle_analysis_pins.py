"""Pins of the capture-range analysis oracle (oracle/map_analysis.py) against what mathematics and
library routines fix -- no GPU, no CUDA library.  A dropped term, a wrong sign, a swapped axis or a
wrong tie rule fails at least one of them."""
import itertools

import numpy as np
import pytest

from oracle import map_analysis as ma


def grid_axes(n, lo, hi):
    return [np.array([lo[d]]) if n[d] == 1 else lo[d] + np.arange(n[d]) * (hi[d] - lo[d]) / (n[d] - 1) for d in range(3)]


def make_map(fn, n, lo, hi):
    p0, p1, p2 = grid_axes(n, lo, hi)
    return fn(p0[None, None, :], p1[None, :, None], p2[:, None, None]) + np.zeros((n[2], n[1], n[0]))


# ------------------------------------------------------------------------------------------------ gradient
def test_gradient_equals_numpy_gradient():
    rng = np.random.default_rng(3)
    n, lo, hi = (7, 5, 9), (-3.0, 0.5, -10.0), (3.0, 2.5, 10.0)
    m = rng.normal(size=(n[2], n[1], n[0]))
    h = [(hi[d] - lo[d]) / (n[d] - 1) for d in range(3)]
    g2, g1, g0 = np.gradient(m, h[2], h[1], h[0], edge_order=1)      # numpy: array axes (2, 1, 0) order
    g = ma.map_gradient(m, lo, hi)
    assert np.allclose(g[0], g0, rtol=1e-14, atol=0) and np.allclose(g[1], g1, rtol=1e-14, atol=0)
    assert np.allclose(g[2], g2, rtol=1e-14, atol=0)


def test_gradient_of_linear_and_quadratic_maps_closed_form():
    n, lo, hi = (9, 6, 5), (-4.0, -2.5, 0.0), (4.0, 2.5, 8.0)
    # linear: every difference quotient is the slope, faces included (components must not be swapped)
    g = ma.map_gradient(make_map(lambda a, b, c: 2.0 * a - 3.0 * b + 0.5 * c + 7.0, n, lo, hi), lo, hi)
    assert np.allclose(g[0], 2.0, atol=1e-12) and np.allclose(g[1], -3.0, atol=1e-12) and np.allclose(g[2], 0.5, atol=1e-12)
    # quadratic a^2: central differences are exact (2a) inside; the one-sided faces are off by h
    g = ma.map_gradient(make_map(lambda a, b, c: a * a + 0 * b + 0 * c, n, lo, hi), lo, hi)
    a = grid_axes(n, lo, hi)[0]
    assert np.allclose(g[0][:, :, 1:-1], (2 * a[1:-1])[None, None, :], atol=1e-12)
    assert np.allclose(g[0][:, :, 0], 2 * a[0] + 1.0, atol=1e-12) and np.allclose(g[0][:, :, -1], 2 * a[-1] - 1.0, atol=1e-12)
    assert np.all(g[1] == 0) and np.all(g[2] == 0)


def test_gradient_singleton_axis_is_zero():
    m = np.arange(12, dtype=np.float64).reshape(4, 1, 3)
    g = ma.map_gradient(m, (0, 5, 0), (2, 5, 3))
    assert np.all(g[1] == 0) and np.allclose(g[0], 1.0) and np.allclose(g[2], 3.0)


# ------------------------------------------------------------------------------------------------ basins
def brute_basins(m, direction, connectivity):
    """Independent restatement with plain Python loops (tiny maps only)."""
    n2, n1, n0 = m.shape
    lin = lambda k2, k1, k0: (k2 * n1 + k1) * n0 + k0
    label = np.zeros(m.shape, dtype=np.int64)
    steps = np.zeros(m.shape, dtype=np.int32)
    for s2, s1, s0 in itertools.product(range(n2), range(n1), range(n0)):
        k, cnt = (s2, s1, s0), 0
        while True:
            best, bv = k, direction * m[k]
            cands = []
            for d in itertools.product((-1, 0, 1), repeat=3):
                nz = sum(x != 0 for x in d)
                if nz == 0 or (connectivity == 6 and nz != 1):
                    continue
                q = (k[0] + d[0], k[1] + d[1], k[2] + d[2])
                if 0 <= q[0] < n2 and 0 <= q[1] < n1 and 0 <= q[2] < n0:
                    cands.append(q)
            for q in sorted(cands, key=lambda q: lin(*q)):          # lowest linear index wins ties
                if direction * m[q] > bv:
                    best, bv = q, direction * m[q]
            if best == k:
                break
            k, cnt = best, cnt + 1
        label[s2, s1, s0], steps[s2, s1, s0] = lin(*k), cnt
    return label, steps


@pytest.mark.parametrize("direction", [1, -1])
@pytest.mark.parametrize("connectivity", [6, 26])
def test_basins_brute_force_on_tiny_random_maps(direction, connectivity):
    rng = np.random.default_rng(11)
    for shape in [(4, 4, 4), (3, 5, 2), (1, 6, 4), (5, 1, 1)]:
        m = rng.normal(size=shape)
        m.reshape(-1)[rng.integers(0, m.size, m.size // 3)] = 0.25      # plateaus: the tie rules matter
        r = ma.map_basins(m, direction, connectivity)
        label, steps = brute_basins(m, direction, connectivity)
        assert np.array_equal(r["label"], label) and np.array_equal(r["steps"], steps)
        assert r["n_extrema"] == len(np.unique(label))
        assert r["target"] == int(np.argmax(direction * m.reshape(-1)))


def test_concave_quadratic_has_one_basin_and_known_path_lengths():
    n, lo, hi = (9, 7, 5), (-4.0, -3.0, -2.0), (4.0, 3.0, 2.0)
    peak = (1.0, -1.0, 0.0)                                            # grid node (5, 2, 2)
    m = make_map(lambda a, b, c: -((a - peak[0]) ** 2 + (b - peak[1]) ** 2 + (c - peak[2]) ** 2), n, lo, hi)
    k2, k1, k0 = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    d = np.stack([np.abs(k0 - 5), np.abs(k1 - 2), np.abs(k2 - 2)])
    t_peak = (2 * n[1] + 2) * n[0] + 5
    for conn, dist in ((26, d.max(axis=0)), (6, d.sum(axis=0))):
        r = ma.map_basins(m, 1, conn)
        assert r["n_extrema"] == 1 and r["target"] == t_peak and r["capture_fraction"] == 1.0
        assert np.all(r["label"] == t_peak)
        assert np.array_equal(r["steps"], dist)                        # Chebyshev / Manhattan distance
    # descent on the negated map is the same problem (PAPER.md:73 speaks of the minimum)
    r = ma.map_basins(-m, -1, 26)
    assert r["n_extrema"] == 1 and np.all(r["label"] == t_peak)


def test_two_equal_peaks_split_the_cube_at_the_bisecting_plane():
    n, lo, hi = (11, 5, 5), (-5.0, -2.0, -2.0), (5.0, 2.0, 2.0)
    f = lambda a, b, c: np.maximum(-((a + 3) ** 2 + b * b + c * c), -((a - 3) ** 2 + b * b + c * c))
    m = make_map(f, n, lo, hi)
    r = ma.map_basins(m, 1, 6, target=(2 * 5 + 2) * 11 + 8)            # the node of the peak at a = +3
    left, right = (2 * 5 + 2) * 11 + 2, (2 * 5 + 2) * 11 + 8
    lab = r["label"]
    assert np.all(lab[:, :, :5] == left) and np.all(lab[:, :, 6:] == right)
    # on the bisecting plane a = 0 both a-neighbours are equally better: the tie goes to the lower
    # linear index, i.e. to the peak at a = -3
    assert np.all(lab[:, :, 5] == left) and r["n_extrema"] == 2
    assert r["target_label"] == right and r["captured"] == 5 * 5 * 5
    assert r["capture_fraction"] == pytest.approx(125 / 275)


def test_basin_invariants_on_a_rough_map():
    rng = np.random.default_rng(5)
    m = rng.normal(size=(9, 8, 7))
    for conn in (6, 26):
        r = ma.map_basins(m, 1, conn, target=100)
        lab, flat = r["label"].reshape(-1), m.reshape(-1)
        nxt = ma.next_pointer(m, 1, conn)
        assert np.array_equal(lab[lab], lab)                          # labels are fixed points
        assert np.array_equal(nxt[lab], lab)
        assert np.all(flat[nxt] >= flat)                              # a step never goes down
        assert np.all(flat[lab] >= flat)
        assert np.array_equal(r["steps"].reshape(-1) == 0, nxt == np.arange(m.size))
        assert r["captured"] == int((lab == lab[100]).sum()) and r["target"] == 100
        # a path from t has one more step than the path from next[t]
        moved = nxt != np.arange(m.size)
        assert np.array_equal(r["steps"].reshape(-1)[moved], r["steps"].reshape(-1)[nxt[moved]] + 1)
