"""Pins of the multi-metric gradient oracle (oracle/multimetric.py): no GPU, no CUDA library."""
import numpy as np
from scipy.spatial.transform import Rotation

import oracle as orc
from oracle import map_analysis as ma
from oracle import multimetric as mm
from paper_1909_10690_b200 import phantoms as ph


def test_compose_matrix_against_scipy_and_the_map_families():
    rng = np.random.default_rng(2)
    for _ in range(5):
        p = np.concatenate([rng.uniform(-9, 9, 3), rng.uniform(-25, 25, 3), rng.uniform(0.7, 1.3, 3)])
        T = mm.compose_matrix(p)
        # R = Rz(az) Ry(ay) Rx(ax): scipy's extrinsic "xyz" sequence
        R = Rotation.from_euler("xyz", p[3:6], degrees=True).as_matrix()
        assert np.allclose(T[:, :3], R @ np.diag(p[6:9]), atol=1e-14)
        assert np.array_equal(T[:, 3], p[:3])
        # y = R S x + t on a point
        x = rng.normal(size=3)
        assert np.allclose(T[:, :3] @ x + T[:, 3], R @ (p[6:9] * x) + p[:3], atol=1e-13)
    ident = np.array([0, 0, 0, 0, 0, 0, 1, 1, 1.0])
    assert np.array_equal(mm.compose_matrix(ident), np.eye(3, 4))
    for fam, sl, p3 in ((0, slice(0, 3), (1.5, -2, 0.25)), (1, slice(3, 6), (4, -3, 2)), (3, slice(6, 9), (1.05, 0.97, 1.02))):
        p = ident.copy()
        p[sl] = p3
        assert np.array_equal(mm.compose_matrix(p), orc.family_matrix(fam, p3))


def test_gradient_components_equal_central_differences_of_the_family_maps():
    """Each parameter group against an exhaustive 3x3x3 map of its own family around p (step = delta):
    the centre node's central difference of the right channel -- Tsallis for translations, Shannon
    for rotations and scales."""
    cfg = ph.get_config("C1")
    q = 0.5
    p = np.array([0, 0, 0, 0, 0, 0, 1, 1, 1.0])
    delta = np.array([1.0, 1.0, 0.5, 2.0, 3.0, 1.0, 0.02, 0.05, 0.03])
    args = (cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, cfg.ranges)
    grad, vals = mm.multimetric_gradient(*args, p, delta, q, interp=1)
    for fam, sl, ch in ((0, slice(0, 3), 1), (1, slice(3, 6), 0), (3, slice(6, 9), 0)):
        lo, hi = p[sl] - delta[sl], p[sl] + delta[sl]
        r = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                       fam, lo, hi, (3, 3, 3), q=(q,), interp=1)
        g = ma.map_gradient(r["map"][ch], lo, hi)[:, 1, 1, 1]
        assert np.allclose(grad[sl], g, rtol=0, atol=1e-12), (fam, grad[sl], g)
        assert np.allclose(vals, r["map"][:, 1, 1, 1], atol=1e-12)
    # the translation components really come from the Tsallis channel: they differ from Shannon's
    r = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                   0, p[:3] - delta[:3], p[:3] + delta[:3], (3, 3, 3), q=(q,), interp=1)
    g_sh = ma.map_gradient(r["map"][0], p[:3] - delta[:3], p[:3] + delta[:3])[:, 1, 1, 1]
    assert np.max(np.abs(grad[:3] - g_sh)) > 1e-3
    # the Shannon translation gradient points towards the ground-truth shift (1.5, -2, 0.5)
    assert np.dot(g_sh, cfg.truth) > 0


def test_skipped_components_and_pseudo_additive_form():
    cfg = ph.get_config("C1")
    p = np.array([0.5, 0, 0, 1, 0, 0, 1, 1, 1.0])
    delta = np.array([1, 0, 0, 0, 0, -1, 0.05, 0, 0.0])
    args = (cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, cfg.ranges)
    g0, v0 = mm.multimetric_gradient(*args, p, delta, 2.0, interp=0)
    assert np.all(g0[[1, 2, 3, 4, 5, 7, 8]] == 0) and g0[0] != 0 and g0[6] != 0
    g1, v1 = mm.multimetric_gradient(*args, p, delta, 2.0, interp=0, form=1)
    assert v1[0] == v0[0] and v1[1] != v0[1]          # Shannon unchanged, Tsallis form changes
    assert g1[6] == g0[6] and g1[0] != g0[0]


def test_register_follows_its_rule_and_reaches_the_map_maximum():
    """The driver on the C1 pair, translations only: every move has the current step length, a halving
    happens exactly when the direction turns back, and the end point sits next to the maximum of the
    Tsallis q = 0.5 translation map (the metric its translation group ascends), which the exhaustive
    oracle map locates independently."""
    cfg = ph.get_config("C1")
    args = (cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, cfg.ranges)
    p0 = np.array([0, 0, 0, 0, 0, 0, 1, 1, 1.0])
    delta = np.array([0.5, 0.5, 0.5, 0, 0, 0, 0, 0, 0.0])
    r = mm.register(*args, p0, delta, (1.0, 0, 0), (0.1, 1, 1), 40, 0.5, interp=1)
    tr = r["trace"]
    assert r["iterations"] == len(tr) - 1 and np.array_equal(tr[0], p0)
    assert np.all(tr[:, 3:] == p0[3:])                       # rotation and scale never move (step 0)
    moves = np.linalg.norm(np.diff(tr[:, :3], axis=0), axis=1)
    L = 1.0
    for k in range(len(moves)):
        if moves[k] == 0:
            assert k == len(moves) - 1                       # the last iteration may not move
            continue
        assert np.isclose(moves[k], L) or np.isclose(moves[k], L / 2)
        if np.isclose(moves[k], L / 2) and not np.isclose(moves[k], L):
            d0, d1 = np.diff(tr[:, :3], axis=0)[k - 1], np.diff(tr[:, :3], axis=0)[k]
            assert np.dot(d0, d1) < 0                        # halved exactly where the direction turned back
            L = L / 2
    assert r["steps"][0] < 0.1 * 2 and r["iterations"] < 40  # stopped on the step length, not the cap
    # independent check of where it ends: the exhaustive Tsallis map at 0.5-voxel resolution
    m = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, *cfg.ranges, 0, (-1, -4, -2), (4, 1, 3),
                   (11, 11, 11), q=(0.5,), interp=1)
    k2, k1, k0 = np.unravel_index(int(m["argmax"][1]), (11, 11, 11))
    peak = np.array([-1 + 0.5 * k0, -4 + 0.5 * k1, -2 + 0.5 * k2])
    assert np.max(np.abs(r["p"][:3] - peak)) <= 0.75, (r["p"][:3], peak)
    # and it climbed: the Tsallis value at the end exceeds the one at the start
    _, v0 = mm.multimetric_gradient(*args, p0, delta, 0.5, interp=1)
    assert r["values"][1] > v0[1]


def test_seed_from_map_reproduces_the_nodes_transform():
    """The hand-off map -> register (reading A22): for every family the nine parameters of a node compose to the
    very transform the map evaluated at that node (compose_matrix(seed) == family_matrix(node)): exactly for
    translation / Euler / scale, to rounding for log-scale and for the versor -> Euler conversion."""
    lo, hi, n = (-0.3, -0.2, -0.25), (0.3, 0.25, 0.2), (5, 4, 3)
    for fam in range(5):
        for index in (0, 7, 23, 59):
            p = mm.seed_from_map(fam, lo, hi, n, index)
            k = (index % 5, (index // 5) % 4, index // 20)
            node = [lo[d] + k[d] * (hi[d] - lo[d]) / (n[d] - 1) for d in range(3)]
            want = orc.family_matrix(fam, node)
            got = mm.compose_matrix(p)
            if fam in (0, 1, 3):
                assert np.array_equal(got, want), (fam, index)
            else:
                assert np.max(np.abs(got - want)) <= 1e-14, (fam, index)
    assert np.array_equal(mm.seed_from_map(0, lo, hi, n, 59), [0.3, 0.25, 0.2, 0, 0, 0, 1, 1, 1])
    assert np.array_equal(mm.seed_from_map(3, (1, 1, 1), (1, 1, 1), (1, 1, 1), 0), [0, 0, 0, 0, 0, 0, 1, 1, 1])
