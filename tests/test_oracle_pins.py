"""Pins for the CPU oracle (no GPU): each checks the oracle against something other than itself --
closed forms, library routines, brute force, invariants (DESIGN.md pins P1..P12)."""
import math
import os

import numpy as np
import pytest
import scipy.ndimage as ndi
import scipy.stats
from scipy.spatial.transform import Rotation

import oracle as orc
from paper_1909_10690_b200 import phantoms as ph

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")
IDENT = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], dtype=np.float32)


def golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()
                out[k] = float(v)
    return out


def levels_volume(K, dims, axis=None):
    """K equiprobable levels, one per bin of a K-bin [0,1] histogram."""
    nx, ny, nz = dims
    if axis is None:
        idx = np.arange(nx * ny * nz) % K
        return ((idx + 0.5) / K).astype(np.float32).reshape(nz, ny, nx)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    src = (i, j, k)[axis]
    return ((src % K + 0.5) / K).astype(np.float32)


# ---------------------------------------------------------------- P1: identity self-pair
def test_p1_identity_levels_closed_form():
    g = golden()
    vol = levels_volume(64, (8, 8, 8))
    for interp in (0, 1):
        h, nv = orc.joint_hist(vol, vol, IDENT, 64, 0, 1, 0, 1, interp)
        assert nv == 512
        assert np.array_equal(h, np.diag(np.full(64, 8, dtype=np.uint32)))
        vals, det = orc.entropies(h, [2.0, 0.5], detail=True)
        assert vals[0] == pytest.approx(g["p1_shannon_K64"], abs=1e-12)
        assert det[0] == pytest.approx(math.log(64), abs=1e-12)
        assert vals[1] == pytest.approx(g["p1_tsallis_q2_K64"], abs=1e-12)
        assert vals[2] == pytest.approx(g["p1_tsallis_q0.5_K64"], abs=1e-11)


def test_p1_identity_any_volume_is_diagonal_and_I_equals_HA():
    vol = ph.config_c1().fixed
    h, nv = orc.joint_hist(vol, vol, IDENT, 64, 0, 1, 0, 1, 1)
    assert nv == vol.size
    assert np.count_nonzero(h - np.diag(np.diag(h))) == 0
    vals, det = orc.entropies(h, detail=True)
    assert vals[0] == pytest.approx(det[0], abs=1e-12)
    # H(A) against scipy on the marginal computed by numpy from the raw intensities
    a = np.clip(np.floor(vol.astype(np.float64) * 64), 0, 63).astype(int)
    assert det[0] == pytest.approx(scipy.stats.entropy(np.bincount(a.ravel(), minlength=64)), abs=1e-12)


# ---------------------------------------------------------------- P2 / P3: exact independence
def test_p2_p3_independence_closed_forms():
    g = golden()
    fixed = levels_volume(4, (4, 4, 4), axis=0)
    moving = levels_volume(4, (4, 4, 4), axis=1)
    h, nv = orc.joint_hist(fixed, moving, IDENT, 4, 0, 1, 0, 1, 0)
    assert nv == 64 and np.all(h == 4)
    add = orc.entropies(h, [2.0, 0.5], form=orc.TSALLIS_ADDITIVE)
    pse = orc.entropies(h, [2.0, 0.5], form=orc.TSALLIS_PSEUDO_ADDITIVE)
    assert add[0] == pytest.approx(g["p2_shannon_indep"], abs=1e-14)
    assert add[1] == pytest.approx(g["p3_additive_q2_K4"], abs=1e-14)
    assert add[2] == pytest.approx(g["p3_additive_q0.5_K4"], abs=1e-13)
    assert pse[1] == pytest.approx(g["p3_pseudo_q2_K4"], abs=1e-14)
    assert pse[2] == pytest.approx(g["p3_pseudo_q0.5_K4"], abs=1e-13)


def test_table1_ratios_golden():
    g = golden()
    assert round(116.21 / 0.8388, 2) == g["t1_translation_xeon8"]
    assert round(86.30 / 1.6471, 2) == g["t1_rotation_xeon64"]
    assert round(99.46 / 0.3076, 2) == g["t1_scale_i7"]


# ---------------------------------------------------------------- P4: q -> 1
@pytest.mark.parametrize("form", [0, 1])
def test_p4_tsallis_converges_to_shannon_linearly(form):
    rng = np.random.default_rng(7)
    h = rng.integers(0, 50, size=(16, 16)).astype(np.uint32)
    sh = orc.entropies(h)[0]
    assert orc.entropies(h, [1.0], form=form)[1] == sh  # q == 1 returns Shannon exactly
    prev = None
    for eps in (1e-1, 1e-2, 1e-3, 1e-4):
        d = [abs(orc.entropies(h, [1 + s * eps], form=form)[1] - sh) for s in (1, -1)]
        if prev is not None:
            for a, b in zip(prev, d):
                assert 5.0 < a / b < 20.0  # one decade in |q-1| -> about one decade in the gap
        prev = d
    assert max(prev) < 5e-3


# ---------------------------------------------------------------- P5: inequalities, symmetry
def test_p5_bounds_and_symmetry():
    cfg = ph.config_c1()
    nb = 64
    for shift in [(0, 0, 0), (1, -2, 1), (3, 0, -1)]:
        M = IDENT.copy(); M[:, 3] = shift
        Mi = IDENT.copy(); Mi[:, 3] = [-s for s in shift]
        h, nv = orc.joint_hist(cfg.fixed, cfg.moving, M, nb, 0, 1, 0, 1, 1)
        vals, (HA, HB, HAB) = orc.entropies(h, detail=True)
        assert -1e-12 <= vals[0] <= min(HA, HB) + 1e-12
        assert HAB <= HA + HB + 1e-12 and max(HA, HB) <= HAB + 1e-12
        assert HA <= math.log(nb) + 1e-12 and HAB <= 2 * math.log(nb)
        # I(A;B) = I(B;A): swapping the volumes with the inverse integer shift transposes h exactly
        ht, nvt = orc.joint_hist(cfg.moving, cfg.fixed, Mi, nb, 0, 1, 0, 1, 1)
        assert nvt == nv and np.array_equal(ht, h.T)
        assert orc.entropies(ht)[0] == pytest.approx(vals[0], abs=1e-12)


def test_entropy_matches_scipy_on_random_histogram():
    rng = np.random.default_rng(3)
    h = rng.integers(0, 1000, size=(32, 32)).astype(np.uint32)
    h[rng.random((32, 32)) < 0.5] = 0
    vals, (HA, HB, HAB) = orc.entropies(h, [0.3, 1.7], detail=True)
    p = h / h.sum()
    assert HA == pytest.approx(scipy.stats.entropy(p.sum(1)), abs=1e-12)
    assert HB == pytest.approx(scipy.stats.entropy(p.sum(0)), abs=1e-12)
    assert HAB == pytest.approx(scipy.stats.entropy(p.ravel()), abs=1e-12)
    # KL form of MI: sum p log(p / (pa pb))
    pa, pb = p.sum(1, keepdims=True), p.sum(0, keepdims=True)
    m = p > 0
    assert vals[0] == pytest.approx(np.sum(p[m] * np.log(p[m] / (pa @ pb)[m])), abs=1e-12)
    for k, q in enumerate([0.3, 1.7]):
        S = lambda x: (1 - np.sum(x[x > 0] ** q)) / (q - 1)
        assert vals[1 + k] == pytest.approx(S(p.sum(1)) + S(p.sum(0)) - S(p.ravel()), rel=1e-12)


def test_empty_overlap_gives_zeros():
    cfg = ph.config_c1()
    M = IDENT.copy(); M[0, 3] = 1000.0
    h, nv = orc.joint_hist(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, 1)
    assert nv == 0 and h.sum() == 0
    assert np.all(orc.entropies(h, [0.5, 2.0]) == 0.0)


# ---------------------------------------------------------------- P6: ramp reproduction
def rand_affine(rng, dims, mag=0.15):
    A = np.eye(3) + rng.uniform(-mag, mag, (3, 3))
    t = rng.uniform(-2, 2, 3)
    c = (np.array(dims) - 1) / 2.0
    m0 = c - A @ c + t
    return np.concatenate([A, m0[:, None]], axis=1).astype(np.float32)


def test_p6_trilinear_reproduces_a_ramp_under_any_affine():
    rng = np.random.default_rng(11)
    fd, md = (13, 11, 9), (12, 14, 10)
    coeffs = (0.031, -0.017, 0.023, 0.4)
    moving = ph.ramp_volume(md, coeffs)
    for _ in range(5):
        M = rand_affine(rng, md)
        val, ok = orc.resample(fd, moving, M, 1)
        k, j, i = np.meshgrid(np.arange(fd[2]), np.arange(fd[1]), np.arange(fd[0]), indexing="ij")
        Md = M.astype(np.float64)
        c = [Md[r, 0] * i + Md[r, 1] * j + Md[r, 2] * k + Md[r, 3] for r in range(3)]
        inside = np.ones_like(ok)
        interior = np.ones_like(ok)
        for r in range(3):
            inside &= (c[r] >= -0.5) & (c[r] < md[r] - 0.5)
            interior &= (c[r] >= 0) & (c[r] <= md[r] - 1)
        # validity region [-0.5, n-0.5) (reading A6); compare away from fp32-vs-fp64 edge ties
        edge = np.zeros_like(ok)
        for r in range(3):
            edge |= (np.abs(c[r] + 0.5) < 1e-4) | (np.abs(c[r] - (md[r] - 0.5)) < 1e-4)
        assert np.array_equal(ok[~edge], inside[~edge])
        expect = coeffs[0] * c[0] + coeffs[1] * c[1] + coeffs[2] * c[2] + coeffs[3]
        sel = ok & interior
        assert sel.sum() > 50
        assert np.max(np.abs(val[sel] - expect[sel])) < 2e-6


# ---------------------------------------------------------------- P7: worked 2x2x2 example
def test_p7_worked_example_2x2x2():
    mv = np.arange(8, dtype=np.float32).reshape(2, 2, 2) / 8 + 0.0625  # v[z][y][x]
    def at(c, interp=1):
        M = np.zeros((3, 4), dtype=np.float32); M[:, 3] = c
        val, ok = orc.resample((1, 1, 1), mv, M, interp)
        return float(val[0, 0, 0]), bool(ok[0, 0, 0])
    assert at((0.5, 0.5, 0.5)) == (pytest.approx(float(mv.mean()), abs=1e-7), True)
    v, ok = at((0.25, 0, 0))
    assert ok and v == pytest.approx(0.75 * mv[0, 0, 0] + 0.25 * mv[0, 0, 1], abs=1e-7)
    v, ok = at((0, 0.25, 0))
    assert ok and v == pytest.approx(0.75 * mv[0, 0, 0] + 0.25 * mv[0, 1, 0], abs=1e-7)
    v, ok = at((0, 0, 0.25))
    assert ok and v == pytest.approx(0.75 * mv[0, 0, 0] + 0.25 * mv[1, 0, 0], abs=1e-7)
    # validity edges: [-0.5, n-0.5), clamped to the edge voxel inside the half-voxel border
    assert at((-0.5, 0, 0)) == (float(mv[0, 0, 0]), True)
    assert at((-0.500001, 0, 0))[1] is False
    assert at((1.4999, 1, 1)) == (float(mv[1, 1, 1]), True)
    assert at((1.5, 0, 0))[1] is False
    # nearest neighbour: round half up, same region
    assert at((0.5, 0, 0), 0) == (float(mv[0, 0, 1]), True)
    assert at((0.4999, 0, 0), 0) == (float(mv[0, 0, 0]), True)
    assert at((-0.5, 0, 0), 0) == (float(mv[0, 0, 0]), True)
    assert at((1.5, 0, 0), 0)[1] is False
    assert at((0, 1.5, 0), 0)[1] is False and at((0, 0, -0.51), 0)[1] is False


def test_p7_integer_shift_equals_slicing_for_both_interpolators():
    cfg = ph.config_c1()
    M = IDENT.copy(); M[:, 3] = (2, -1, 3)
    for interp in (0, 1):
        val, ok = orc.resample((32, 32, 32), cfg.moving, M, interp)
        assert np.array_equal(val[:29, 1:, :30], cfg.moving[3:, :31, 2:])
        assert ok[:29, 1:, :30].all() and ok.sum() == 29 * 31 * 30


# ---------------------------------------------------------------- P8: library routine
def test_p8_matches_scipy_map_coordinates_on_interior_points():
    rng = np.random.default_rng(5)
    fd, md = (17, 15, 12), (16, 18, 13)
    moving = ph.random_volume(md, 9)
    for _ in range(4):
        M = rand_affine(rng, md, 0.2)
        val, ok = orc.resample(fd, moving, M, 1)
        k, j, i = np.meshgrid(np.arange(fd[2]), np.arange(fd[1]), np.arange(fd[0]), indexing="ij")
        Md = M.astype(np.float64)
        c = [Md[r, 0] * i + Md[r, 1] * j + Md[r, 2] * k + Md[r, 3] for r in range(3)]
        interior = ok.copy()
        for r in range(3):
            interior &= (c[r] >= 0) & (c[r] <= md[r] - 1)
        ref = ndi.map_coordinates(moving.astype(np.float64), [c[2], c[1], c[0]], order=1)
        assert interior.sum() > 100
        assert np.max(np.abs(val[interior] - ref[interior])) < 2e-6
        # nearest neighbour = rounding the same coordinates (away from .5 ties)
        valn, okn = orc.resample(fd, moving, M, 0)
        tie = np.zeros_like(ok)
        for r in range(3):
            tie |= np.abs((c[r] + 0.5) - np.round(c[r] + 0.5)) < 1e-4
        jn = [np.floor(c[r] + 0.5).astype(int) for r in range(3)]
        sel = okn & ~tie
        assert np.array_equal(valn[sel], moving[jn[2][sel], jn[1][sel], jn[0][sel]])


# ---------------------------------------------------------------- P9: histogram invariants
def test_p9_histogram_counts_and_numpy_cross_check():
    cfg = ph.config_c1()
    nb = 64
    rng = np.random.default_rng(2)
    fbins_np = np.clip(np.floor(cfg.fixed.astype(np.float64) * nb), 0, nb - 1).astype(int)
    assert np.array_equal(orc.prebin(cfg.fixed, nb, 0, 1), fbins_np)
    for interp in (0, 1):
        M = rand_affine(rng, (32, 32, 32), 0.05)
        h, nv = orc.joint_hist(cfg.fixed, cfg.moving, M, nb, 0, 1, 0, 1, interp)
        val, ok = orc.resample((32, 32, 32), cfg.moving, M, interp)
        assert h.sum() == nv == ok.sum()
        b = np.clip(np.floor(val.astype(np.float32) * np.float32(nb)), 0, nb - 1).astype(int)
        ref = np.bincount(fbins_np[ok] * nb + b[ok], minlength=nb * nb).reshape(nb, nb)
        assert np.array_equal(h, ref)  # row = fixed bin, column = moving bin
        h2, _, _ = np.histogram2d(fbins_np[ok], b[ok], bins=[np.arange(nb + 1)] * 2)
        assert np.array_equal(h, h2.astype(np.uint32))
    # all-valid transform (identity): row sums equal the fixed-bin histogram whatever the moving image
    h, nv = orc.joint_hist(cfg.fixed, cfg.moving, IDENT, nb, 0, 1, 0, 1, 1)
    assert nv == cfg.fixed.size
    assert np.array_equal(h.sum(1), np.bincount(fbins_np.ravel(), minlength=nb))


def test_binning_edges():
    v = np.array([-1.0, 0.0, 0.2499999, 0.25, 0.5, 0.999999, 1.0, 7.0], dtype=np.float32)
    assert orc.prebin(v, 4, 0.0, 1.0).tolist() == [0, 0, 0, 1, 2, 3, 3, 3]
    v = np.array([10.0, 12.5, 15.0, 19.99, 20.0], dtype=np.float32)
    assert orc.prebin(v, 10, 10.0, 20.0).tolist() == [0, 2, 5, 9, 9]


# ---------------------------------------------------------------- P10: brute force on 4^3
def brute_force_hist(fixed, moving, M, nb, interp):
    """Independent pure-Python loops in double; inputs are dyadic so fp32 == fp64 exactly."""
    nz, ny, nx = fixed.shape
    mz, my, mx = moving.shape
    h = [[0] * nb for _ in range(nb)]
    for iz in range(nz):
        for iy in range(ny):
            for ix in range(nx):
                c = [M[r][0] * ix + M[r][1] * iy + M[r][2] * iz + M[r][3] for r in range(3)]
                n = (mx, my, mz)
                if any(not (-0.5 <= c[r] < n[r] - 0.5) for r in range(3)):
                    continue
                if interp == 0:
                    j = [int(math.floor(c[r] + 0.5)) for r in range(3)]
                    v = float(moving[j[2], j[1], j[0]])
                else:
                    v = 0.0
                    g = [math.floor(c[r]) for r in range(3)]
                    f = [c[r] - g[r] for r in range(3)]
                    for dz in (0, 1):
                        for dy in (0, 1):
                            for dx in (0, 1):
                                w = ((f[0] if dx else 1 - f[0]) * (f[1] if dy else 1 - f[1])
                                     * (f[2] if dz else 1 - f[2]))
                                x = min(max(g[0] + dx, 0), mx - 1)
                                y = min(max(g[1] + dy, 0), my - 1)
                                z = min(max(g[2] + dz, 0), mz - 1)
                                v += w * float(moving[z, y, x])
                a = min(max(int(math.floor(float(fixed[iz, iy, ix]) * nb)), 0), nb - 1)
                b = min(max(int(math.floor(v * nb)), 0), nb - 1)
                h[a][b] += 1
    return np.array(h, dtype=np.uint32)


@pytest.mark.parametrize("interp", [0, 1])
def test_p10_brute_force_4cubed(interp):
    rng = np.random.default_rng(42)
    fixed = (rng.integers(0, 64, (4, 4, 4)) / 64).astype(np.float32)
    moving = (rng.integers(0, 64, (4, 4, 4)) / 64).astype(np.float32)
    mats = [IDENT,
            np.array([[1, 0, 0, 0.25], [0, 1, 0, -0.5], [0, 0, 1, 0.75]]),
            np.array([[0.75, 0.25, 0, 0.5], [-0.25, 1, 0.125, 0.25], [0, 0.25, 0.5, 1.0]]),
            np.array([[0, 1, 0, 0.0], [0, 0, 1, 0.25], [1, 0, 0, 0.5]]),   # axis permutation
            np.array([[-1, 0, 0, 3.0], [0, 1, 0, 0.0], [0, 0, 1.25, -0.5]])]
    for M in mats:
        ref = brute_force_hist(fixed, moving, np.asarray(M, dtype=np.float64), 8, interp)
        h, nv = orc.joint_hist(fixed, moving, np.asarray(M, dtype=np.float32), 8, 0, 1, 0, 1, interp)
        assert np.array_equal(h, ref), M
        assert nv == ref.sum()


# ---------------------------------------------------------------- CANON-1 and family generators
def test_canon1_identity_is_exact_and_matches_physical_composition():
    fd, fs, md, ms = (260, 311, 260), (0.7, 0.7, 0.7), (182, 218, 182), (1.0, 1.0, 1.0)
    Tid = np.concatenate([np.eye(3), np.zeros((3, 1))], axis=1)
    M = orc.index_affine(Tid, fd, fs, fd, fs)
    assert np.array_equal(M, IDENT)  # identity self-pair samples exactly on voxel centres
    rng = np.random.default_rng(1)
    for _ in range(20):
        A = np.eye(3) + rng.uniform(-0.3, 0.3, (3, 3))
        t = rng.uniform(-20, 20, 3)
        M = orc.index_affine(np.concatenate([A, t[:, None]], axis=1), fd, fs, md, ms).astype(np.float64)
        i = rng.uniform(0, 259, (3, 50))
        x = np.array(fs)[:, None] * (i - (np.array(fd)[:, None] - 1) / 2)      # fixed physical
        y = A @ x + t[:, None]                                                 # moving physical
        c = y / np.array(ms)[:, None] + (np.array(md)[:, None] - 1) / 2        # moving index
        assert np.max(np.abs(M[:, :3] @ i + M[:, 3:4] - c)) < 2e-4             # fp32 rounding of M only


def test_family_generators_against_scipy():
    p = (11.0, -23.0, 37.0)
    R = orc.family_matrix(orc.FAMILY_ROTATION_EULER_DEG, p)
    ref = Rotation.from_euler("xyz", p, degrees=True).as_matrix()  # extrinsic xyz = Rz Ry Rx
    assert np.allclose(R[:, :3], ref, atol=1e-14) and np.all(R[:, 3] == 0)
    assert np.allclose(R[:, :3], ph.euler_deg_matrix(p)[:, :3], atol=1e-14)
    v = np.array([0.3, -0.2, 0.5])
    Rv = orc.family_matrix(orc.FAMILY_ROTATION_VERSOR, v)
    ref = Rotation.from_quat([v[0], v[1], v[2], math.sqrt(1 - v @ v)]).as_matrix()
    assert np.allclose(Rv[:, :3], ref, atol=1e-14)
    # outside the unit ball -> mapped to its surface: a half-turn about v/|v|
    Rs = orc.family_matrix(orc.FAMILY_ROTATION_VERSOR, 3 * v)
    u = v / np.linalg.norm(v)
    assert np.allclose(Rs[:, :3], 2 * np.outer(u, u) - np.eye(3), atol=1e-12)
    assert np.array_equal(orc.family_matrix(orc.FAMILY_TRANSLATION, (1, 2, 3)),
                          np.array([[1, 0, 0, 1], [0, 1, 0, 2], [0, 0, 1, 3.0]]))
    assert np.array_equal(orc.family_matrix(orc.FAMILY_SCALE, (1.1, 0.9, 1.0))[:, :3], np.diag([1.1, 0.9, 1.0]))
    assert np.allclose(orc.family_matrix(orc.FAMILY_SCALE_LOG, (0.1, -0.1, 0))[:, :3],
                       np.diag(np.exp([0.1, -0.1, 0])), atol=1e-15)


# ---------------------------------------------------------------- P11: the map peaks at the truth
def test_p11_c1_map_peaks_at_ground_truth_and_layout():
    cfg = ph.config_c1()
    r = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, 0, 1, 0, 1,
                   cfg.family, cfg.lo, cfg.hi, cfg.n, q=cfg.q)
    m = r["map"]
    assert m.shape == (3, 5, 5, 5)
    k2, k1, k0 = np.unravel_index(r["argmax"][0], m.shape[1:])
    p = [cfg.lo[d] + k * (cfg.hi[d] - cfg.lo[d]) / (cfg.n[d] - 1) for d, k in enumerate((k0, k1, k2))]
    assert max(abs(p[d] - cfg.truth[d]) for d in range(3)) <= 1.0  # within one grid step (Chebyshev)
    for ch in range(3):
        assert r["argmax"][ch] == int(np.argmax(m[ch].ravel()))
    # a map voxel equals a direct evaluation of that transform (p0 fastest)
    T = orc.family_matrix(0, (1.0, -2.0, 0.0))
    M = orc.index_affine(T, (32, 32, 32), cfg.fixed_spacing, (32, 32, 32), cfg.moving_spacing)
    h, _ = orc.joint_hist(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, 1)
    assert m[:, 2, 0, 3] == pytest.approx(orc.entropies(h, cfg.q), abs=1e-14)
    # self-pair: the gold standard is the centre of the map
    r = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.fixed, cfg.fixed_spacing, 64, 0, 1, 0, 1,
                   0, (-2, -2, -2), (2, 2, 2), (5, 5, 5))
    assert r["argmax"][0] == 62


# ---------------------------------------------------------------- P12: fp32 vs fp64 geometry (report)
def test_p12_f64_geometry_differs_only_slightly():
    cfg = ph.config_c1()
    T = np.concatenate([ph.euler_deg_matrix((3, -2, 1))[:, :3], np.array([[0.3], [-0.7], [0.2]])], axis=1)
    M32 = orc.index_affine(T, (32,) * 3, cfg.fixed_spacing, (32,) * 3, cfg.moving_spacing)
    h32, _ = orc.joint_hist(cfg.fixed, cfg.moving, M32, 64, 0, 1, 0, 1, 1)
    h64, _ = orc.joint_hist(cfg.fixed, cfg.moving, M32.astype(np.float64), 64, 0, 1, 0, 1, 1, f64_coords=True)
    moved = np.abs(h32.astype(np.int64) - h64.astype(np.int64)).sum() / 2
    assert moved <= 1e-3 * cfg.fixed.size
    assert abs(orc.entropies(h32)[0] - orc.entropies(h64)[0]) < 1e-3


def test_eval_batch_matches_single_calls():
    cfg = ph.config_c1()
    rng = np.random.default_rng(8)
    Ms = np.stack([rand_affine(rng, (32, 32, 32), 0.05) for _ in range(5)])
    r = orc.eval_batch(cfg.fixed, cfg.moving, Ms, 64, 0, 1, 0, 1, 1, q=[0.5], want_hist=True)
    for k in range(5):
        h, nv = orc.joint_hist(cfg.fixed, cfg.moving, Ms[k], 64, 0, 1, 0, 1, 1)
        assert np.array_equal(r["hist"][k], h) and r["nvalid"][k] == nv
        assert np.array_equal(r["mi"][k], orc.entropies(h, [0.5]))


def test_map_range_helper_equals_orc_map():
    """oracle.mi_map_range (grid formula + family generator + CANON-1 per node, in Python around the C++
    calls) over the whole node range reproduces orc_map bit for bit on a grid with a non-representable step,
    and a sub-box is the corresponding slice."""
    cfg = ph.config_c1(grid_n=4)
    lo, hi = (-1.0, -0.7, 0.1), (1.0, 1.3, 0.9)
    args = (cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, 0, 1, 0, 1, cfg.family, lo, hi, cfg.n)
    full = orc.mi_map(*args, q=(0.5,))["map"]
    assert np.array_equal(orc.mi_map_range(*args, (0, 0, 0), cfg.n, q=(0.5,)), full)
    assert np.array_equal(orc.mi_map_range(*args, (1, 0, 2), (3, 4, 4), q=(0.5,)), full[:, 2:4, 0:4, 1:3])


def test_expected_bank_load_of_independent_uniform_lanes():
    """Roofline arithmetic, not oracle arithmetic: a warp-wide shared-memory update takes as many passes as the
    fullest of the 32 banks holds distinct addresses.  For 32 lanes with independent uniform bins that is 3.53 on
    average (the denominator of the headline roofline fraction); an arithmetic progression of
    bins across the lanes -- what one linear congruential generator per thread, seeded linearly in the thread
    index, produces -- is spread more evenly (about 2.7)."""
    rng = np.random.default_rng(7)
    x = rng.integers(0, 1 << 16, size=(20000, 32))
    load = np.array([np.bincount(r & 31, minlength=32).max() for r in x])
    assert abs(load.mean() - 3.53) < 0.03
    lane = np.arange(32, dtype=np.uint64)
    loads = []
    for _ in range(4000):
        a, d = (int(v) for v in rng.integers(0, 1 << 32, size=2))
        s = (np.uint64(a) + lane * np.uint64(d | 1)) & np.uint64(0xFFFFFFFF)
        loads.append(np.bincount(((s >> np.uint64(10)) & np.uint64(31)).astype(np.int64), minlength=32).max())
    assert 2.4 < np.mean(loads) < 3.0, np.mean(loads)
