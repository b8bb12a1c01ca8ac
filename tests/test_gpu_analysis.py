"""GPU parity of the capture-range analysis calls (mi_map_gradient, mi_map_basins) against the CPU
oracle (oracle/map_analysis.py), through the C ABI.  Labels, steps and counts are integer work:
bit-exact.  The gradient is one IEEE double subtraction and one division per component: both sides
do the same two correctly rounded operations, so it is compared for equality as well."""
import numpy as np
import pytest

from oracle import map_analysis as ma
from paper_1909_10690_b200 import phantoms as ph

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mi():
    from paper_1909_10690_b200 import build
    build.build()
    from paper_1909_10690_b200 import binding
    return binding


def rough_map(shape, seed, plateaus=True):
    rng = np.random.default_rng(seed)
    m = rng.normal(size=shape)
    if plateaus:
        m.reshape(-1)[rng.integers(0, m.size, m.size // 4)] = 0.5
    return m


def check_basins(mi, m, direction, conn, target):
    ref = ma.map_basins(m, direction, conn, target)
    got = mi.mi_map_basins(m, direction, conn, target)
    assert np.array_equal(got["label"], ref["label"])
    assert np.array_equal(got["steps"], ref["steps"])
    for k in ("n_extrema", "target", "target_label", "captured", "max_steps"):
        assert got[k] == ref[k], k
    assert got["capture_fraction"] == ref["capture_fraction"]
    return got


def test_gradient_equals_oracle_exactly(mi):
    for shape, lo, hi in [((9, 8, 7), (-3, -2, 0), (3, 2, 9)), ((1, 1, 5), (0, 0, 0), (4, 1, 1)), ((41, 41, 41), (-10,) * 3, (10,) * 3),
                          ((2, 300, 1), (0, -7, 0.5), (0, 7, 1.5)), ((1, 1, 1), (0, 0, 0), (0, 0, 0))]:
        m = rough_map(shape, 1, plateaus=False)
        lo3, hi3 = list(lo), list(hi)
        for d in range(3):                      # an axis with one node may have lo == hi
            if shape[2 - d] == 1:
                hi3[d] = lo3[d]
        g = mi.mi_map_gradient(m, lo3, hi3)
        assert np.array_equal(g, ma.map_gradient(m, lo3, hi3)), shape


def test_basins_equal_oracle_on_rough_maps(mi):
    for shape in [(4, 4, 4), (9, 8, 7), (1, 1, 1), (1, 6, 40), (33, 1, 1), (41, 41, 41), (30, 50, 70)]:
        m = rough_map(shape, 7)
        for direction in (1, -1):
            for conn in (6, 26):
                check_basins(mi, m, direction, conn, -1)
        check_basins(mi, m, 1, 26, m.size // 2)


def test_basins_long_paths_need_many_doubling_rounds(mi):
    # a monotone ramp along a 1 x 1 x 5000 line: one path of 4999 moves (13 doubling rounds)
    m = np.arange(5000, dtype=np.float64).reshape(1, 1, 5000)
    r = check_basins(mi, m, 1, 6, 0)
    assert r["max_steps"] == 4999 and r["n_extrema"] == 1 and r["capture_fraction"] == 1.0
    # a serpentine ridge through a 2D sheet: path length ~ n0*n1/2
    n0, n1 = 64, 63
    m = np.full((1, n1, n0), -1.0)
    v = 0.0
    for k1 in range(0, n1, 2):
        cols = range(n0) if (k1 // 2) % 2 == 0 else range(n0 - 1, -1, -1)
        for k0 in cols:
            m[0, k1, k0] = v
            v += 1.0
        if k1 + 1 < n1:
            m[0, k1 + 1, cols[-1]] = v
            v += 1.0
    r = check_basins(mi, m, 1, 6, 0)
    assert r["max_steps"] > 2000


def test_basins_device_pointers_and_no_arrays(mi):
    import torch
    m = rough_map((20, 21, 22), 3)
    ref = ma.map_basins(m, 1, 26, -1)
    md = torch.from_numpy(m).cuda()
    got = mi.mi_map_basins(md, 1, 26, -1)
    assert got["label"].is_cuda and np.array_equal(got["label"].cpu().numpy(), ref["label"])
    assert np.array_equal(got["steps"].cpu().numpy(), ref["steps"])
    g = mi.mi_map_gradient(md, (0, 0, 0), (1, 1, 1))
    assert g.is_cuda and np.array_equal(g.cpu().numpy(), ma.map_gradient(m, (0, 0, 0), (1, 1, 1)))
    only = mi.mi_map_basins(m, 1, 26, -1, want_arrays=False)
    assert only["label"] is None and only["captured"] == ref["captured"]


def test_analysis_argument_errors(mi):
    m = np.zeros((3, 3, 3))
    for kw in (dict(direction=0), dict(connectivity=18), dict(target=27), dict(target=-2)):
        with pytest.raises(mi.MIError) as ei:
            mi.mi_map_basins(m, **kw)
        assert ei.value.status == mi.MI_ERR_INVALID_ARG
    with pytest.raises(mi.MIError) as ei:
        mi.mi_map_gradient(m, (0, 0, 0), (1, 0, 1))          # three nodes on an axis of zero length
    assert ei.value.status == mi.MI_ERR_INVALID_ARG


def test_capture_range_of_a_real_map_shannon_and_tsallis(mi):
    """End to end on the C1 translation map (9^3 half-step grid): every channel's basins equal the
    oracle's on the oracle's own map and on the GPU map; the Shannon channel captures the node next to
    the ground truth (P11: the arg max is within one step of it)."""
    import oracle as orc
    cfg = ph.config_c1(grid_n=9)
    ref = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                     cfg.family, cfg.lo, cfg.hi, cfg.n, q=cfg.q, interp=1)
    with mi.mi_create(cfg.fixed, cfg.moving, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins) as ctx:
        gm, am = mi.mi_map(ctx, cfg.family, cfg.lo, cfg.hi, cfg.n, cfg.q, 1)
    for ch in range(gm.shape[0]):
        r = check_basins(mi, ref["map"][ch], 1, 26, -1)
        g = mi.mi_map_basins(gm[ch], 1, 26, -1)
        # the two maps differ by ~1e-10 nats: the same arg max, and the same basins wherever the
        # oracle's map has no near-tie between a node's best and second-best neighbour
        assert g["target"] == r["target"] == int(am[ch])
    sh = mi.mi_map_basins(gm[0], 1, 26, -1)
    k2, k1, k0 = np.unravel_index(sh["target"], gm.shape[1:])
    p = [cfg.lo[d] + k * (cfg.hi[d] - cfg.lo[d]) / (cfg.n[d] - 1) for d, k in enumerate((k0, k1, k2))]
    assert max(abs(p[d] - cfg.truth[d]) for d in range(3)) <= 1.0
    assert 0.0 < sh["capture_fraction"] <= 1.0


def test_multimetric_gradient_equals_oracle(mi):
    """mi_multimetric_gradient (one mi_eval_batch of 2*9 + 1 transforms) against oracle/multimetric.py: MI values
    within 1e-4 nats, so each central difference within 1e-4 / delta_k; skipped components are exactly 0."""
    from oracle import multimetric as mm
    cfg = ph.get_config("C1")
    args = (cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, cfg.ranges)
    cases = [(np.array([0, 0, 0, 0, 0, 0, 1, 1, 1.0]), np.array([1.0, 1.0, 0.5, 2.0, 3.0, 1.0, 0.02, 0.05, 0.03]), 0.5, 0),
             (np.array([1.2, -1.5, 0.4, 3, -2, 1, 1.03, 0.98, 1.01]), np.array([0.5, 0.5, 0.5, 1, 1, 1, 0.01, 0.01, 0.01]), 2.0, 0),
             (np.array([0.5, 0, 0, 1, 0, 0, 1, 1, 1.0]), np.array([1, 0, 0, 0, 0, -1, 0.05, 0, 0.0]), 2.0, 1)]
    with mi.mi_create(cfg.fixed, cfg.moving, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins) as ctx:
        for p, delta, q, form in cases:
            mi.mi_set_tsallis_form(ctx, form)
            for interp in (0, 1):
                g_ref, v_ref = mm.multimetric_gradient(*args, p, delta, q, interp=interp, form=form)
                g, v = mi.mi_multimetric_gradient(ctx, p, delta, q, interp)
                assert np.max(np.abs(v - v_ref)) <= 1e-4
                tol = np.where(delta > 0, 1e-4 / np.maximum(delta, 1e-300), 0.0)
                assert np.all(np.abs(g - g_ref) <= tol), (g, g_ref)
                assert np.all(g[delta <= 0] == 0)
        with pytest.raises(mi.MIError):
            mi.mi_multimetric_gradient(ctx, cases[0][0], cases[0][1], -1.0, 1)


def test_register_follows_the_oracle_trajectory(mi):
    """mi_register against oracle/multimetric.register: same rule, gradients equal to ~1e-9, so the visited
    points agree to 1e-6 and the step halvings fall on the same iterations."""
    from oracle import multimetric as mm
    cfg = ph.get_config("C1")
    args = (cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, cfg.ranges)
    p0 = np.array([0, 0, 0, 0, 0, 0, 1, 1, 1.0])
    runs = [(np.array([0.5, 0.5, 0.5, 0, 0, 0, 0, 0, 0.0]), (1.0, 0, 0), (0.1, 1, 1), 40, 0.5),
            (np.array([0.5, 0.5, 0.5, 1, 1, 1, 0.02, 0.02, 0.02]), (0.5, 0.5, 0.01), (0.1, 0.1, 0.002), 12, 0.5)]
    with mi.mi_create(cfg.fixed, cfg.moving, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins) as ctx:
        for delta, step0, step_min, iters, q in runs:
            ref = mm.register(*args, p0, delta, step0, step_min, iters, q, interp=1)
            got = mi.mi_register(ctx, p0, delta, step0, step_min, iters, q, 1)
            assert got["iterations"] == ref["iterations"]
            assert np.max(np.abs(got["trace"] - ref["trace"])) <= 1e-6
            assert np.allclose(got["steps"], ref["steps"], rtol=0, atol=0)
            assert np.max(np.abs(got["values"] - ref["values"])) <= 1e-4
            assert np.array_equal(got["p"], got["trace"][-1])
        r0 = mi.mi_register(ctx, p0, runs[0][0], (0, 0, 0), (1, 1, 1), 5, 0.5, 1)     # nothing may move
        assert r0["iterations"] == 1 and np.array_equal(r0["p"], p0)


def test_coarse_map_seeds_the_registration(mi):
    """SURVEY 8(f)-2's hand-off end to end on the GPU: a coarse exhaustive map (the exhaustive
    search as the robust start) -> mi_seed_from_map at its arg max -> mi_register (multi-metric ascent,
    PAPER.md:199, 210).  Translation on the C1 pair: coarse 5^3 map on integer voxels, Tsallis q = 0.5 channel
    for the translation group as the paper recommends; the ascent must end within one FINE step (0.5 voxel) of
    the maximum of the fine 0.5-voxel map, and equal the oracle's trajectory from the same seed.  Rotation on
    the quarter-resolution C3 pair: coarse 5^3 Euler map over +-6 deg (Shannon), ascent over the rotation group
    ends within one fine step (1 deg) of the fine map's maximum."""
    import oracle as orc
    from oracle import multimetric as mm
    cfg = ph.get_config("C1")
    with mi.mi_create(cfg.fixed, cfg.moving, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins) as ctx:
        coarse, am = mi.mi_map(ctx, 0, cfg.lo, cfg.hi, cfg.n, (0.5,), 1)
        p0 = mi.mi_seed_from_map(0, cfg.lo, cfg.hi, cfg.n, am[1])           # arg max of the Tsallis channel
        assert np.array_equal(p0, mm.seed_from_map(0, cfg.lo, cfg.hi, cfg.n, int(am[1])))
        delta = np.array([0.5, 0.5, 0.5, 0, 0, 0, 0, 0, 0.0])
        got = mi.mi_register(ctx, p0, delta, (0.5, 0, 0), (0.05, 1, 1), 40, 0.5, 1)
        fine, fam = mi.mi_map(ctx, 0, (-1, -4, -2), (4, 1, 3), (11, 11, 11), (0.5,), 1)
    ref = mm.register(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, cfg.ranges, p0, delta,
                      (0.5, 0, 0), (0.05, 1, 1), 40, 0.5, interp=1)
    assert got["iterations"] == ref["iterations"] and np.max(np.abs(got["trace"] - ref["trace"])) <= 1e-6
    k2, k1, k0 = np.unravel_index(int(fam[1]), (11, 11, 11))
    peak = np.array([-1 + 0.5 * k0, -4 + 0.5 * k1, -2 + 0.5 * k2])
    assert np.max(np.abs(got["p"][:3] - peak)) <= 0.5 + 1e-9, (got["p"][:3], peak)
    assert got["values"][1] >= coarse[1].max() - 1e-9                       # it did not fall below its seed

    c3 = ph.get_config("C3", res=0.25, grid_n=5)
    lo, hi, n = (-6.0,) * 3, (6.0,) * 3, (5, 5, 5)
    with mi.mi_create(c3.fixed, c3.moving, c3.fixed_spacing, c3.moving_spacing, c3.nbins) as ctx:
        coarse, am = mi.mi_map(ctx, 1, lo, hi, n, (), 1)
        p0 = mi.mi_seed_from_map(1, lo, hi, n, am[0])
        assert np.array_equal(p0[:3], [0, 0, 0]) and np.array_equal(p0[6:], [1, 1, 1])
        delta = np.array([0, 0, 0, 1.0, 1.0, 1.0, 0, 0, 0])
        got = mi.mi_register(ctx, p0, delta, (0, 1.0, 0), (1, 0.1, 1), 30, 0.5, 1)
        centre = p0[3:6]
        flo, fhi = tuple(centre - 3.0), tuple(centre + 3.0)
        fine, fam = mi.mi_map(ctx, 1, flo, fhi, (7, 7, 7), (), 1)
    k2, k1, k0 = np.unravel_index(int(fam[0]), (7, 7, 7))
    peak = np.array([flo[0] + k0, flo[1] + k1, flo[2] + k2])
    assert np.max(np.abs(got["p"][3:6] - peak)) <= 1.0 + 1e-9, (got["p"][3:6], peak)
    assert got["values"][0] >= coarse[0].max() - 1e-9


def test_partial_volume_gradient_needs_a_step_its_quantisation_resolves(mi):
    """Partial-volume weights are quantised to 1/32 voxel (reading A21), so PV MI is piecewise constant in the
    transform.  mi_pv_min_delta names the smallest finite-difference steps that quantisation resolves;
    mi_multimetric_gradient / mi_register refuse anything smaller instead of returning a silent zero, and at the
    smallest accepted step the two arms really see different histograms and every gradient component is non-zero.
    Trilinear has no bound."""
    cfg = ph.get_config("C1")
    p = np.array([0.7, -0.4, 0.3, 2.0, -1.0, 1.5, 1.02, 0.99, 1.01])
    with mi.mi_create(cfg.fixed, cfg.moving, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins) as ctx:
        dmin = mi.mi_pv_min_delta(ctx)
        ms = np.asarray(cfg.moving_spacing, dtype=np.float64)
        assert np.array_equal(dmin[:3], ms / 32.0) and np.all(dmin[3:] > 0)
        g, _ = mi.mi_multimetric_gradient(ctx, p, dmin, 0.5, mi.MI_INTERP_PARTIAL_VOLUME)
        assert np.all(g != 0.0), g
        for k in range(9):
            e = np.zeros(9)
            e[k] = dmin[k]
            T = np.stack([mi.mi_compose_matrix(p), mi.mi_compose_matrix(p + e)])
            _, h, _ = mi.mi_eval_batch_pv(ctx, T, (), hist_out=True)
            assert not np.array_equal(h[0], h[1]), "PV histogram unchanged by the smallest accepted step of parameter %d" % k
            small = np.zeros(9)
            small[k] = 0.99 * dmin[k]
            with pytest.raises(mi.MIError) as err:
                mi.mi_multimetric_gradient(ctx, p, small, 0.5, mi.MI_INTERP_PARTIAL_VOLUME)
            assert err.value.status == mi.MI_ERR_INVALID_ARG and "mi_pv_min_delta" in str(err.value)
            mi.mi_multimetric_gradient(ctx, p, small, 0.5, mi.MI_INTERP_TRILINEAR)      # no bound without quantisation
        with pytest.raises(mi.MIError):
            mi.mi_register(ctx, p, 0.5 * dmin, (0.5, 0.5, 0.01), (0.1, 0.1, 0.002), 3, 0.5, mi.MI_INTERP_PARTIAL_VOLUME)
        r = mi.mi_register(ctx, p, dmin, (0.5, 0.5, 0.01), (0.1, 0.1, 0.002), 3, 0.5, mi.MI_INTERP_PARTIAL_VOLUME)
        assert r["iterations"] >= 1
