"""Pins of the oracle's partial-volume interpolation (reading A21; Maes et al., the paper's ref. [5],
PAPER.md:228; "the effects of interpolation") against what the mathematics fixes -- none of
them re-calls the oracle's own formula:

  PV1  every sample adds exactly 2^15 units: sum(h) = nvalid * 2^15; for an all-valid transform the row sums
       are the fixed-bin histogram times 2^15 whatever the transform
  PV2  integer shifts: all weight on one neighbour -> h_pv = 2^15 * h_nearest = 2^15 * h_trilinear
  PV3  worked 2x2x2 example by hand: c = (.5,.5,.5) -> eight weights of 16^3 = 4096; c = (.25,0,0) ->
       24*32*32 = 24576 on v000 and 8*32*32 = 8192 on v100
  PV4  brute force on 4^3 volumes with independent Python loops (own floor / fraction / clamp code)
  PV5  a shift of j + 1/4 voxel along x: h_pv = 24*1024 * H(shift j) + 8*1024 * H(shift j+1), the two
       integer-shift histograms built with numpy slicing and bincount
  PV6  the uint64 entropy routine is scale-free: entropies(2^15 * h) = entropies(h) of the pinned uint32 routine
  PV7  rounding of the fraction to 1/32: ties go up (f = 1/64 -> u = 1), f just below -> u = 0
"""
import math

import numpy as np
import pytest

import oracle as orc
from paper_1909_10690_b200 import phantoms as ph

UNITS = 1 << 15


def ident_index(shift=(0.0, 0.0, 0.0)):
    """Index-space [I | shift] (float32): c = i + shift."""
    M = np.zeros((3, 4), dtype=np.float32)
    M[0, 0] = M[1, 1] = M[2, 2] = 1.0
    M[:, 3] = shift
    return M


def bins_of(v, nb, lo=0.0, hi=1.0):
    """Independent CANON-5 in numpy float32."""
    scale = np.float32(np.float64(nb) / (np.float64(np.float32(hi)) - np.float64(np.float32(lo))))
    t = (v.astype(np.float32) - np.float32(lo)) * scale
    return np.clip(np.floor(t), 0, nb - 1).astype(np.int64)


def test_pv1_units_per_sample_and_fixed_marginal():
    fixed = ph.random_volume((9, 7, 5), 1)
    moving = ph.random_volume((20, 18, 16), 2)
    rng = np.random.default_rng(0)
    for _ in range(5):
        A = np.eye(3) + rng.uniform(-0.15, 0.15, (3, 3))
        T = np.concatenate([A, rng.uniform(-1, 1, 3)[:, None]], axis=1)
        M = orc.index_affine(T, (9, 7, 5), (1, 1, 1), (20, 18, 16), (1, 1, 1))
        h, nv = orc.joint_hist_pv(fixed, moving, M, 16, 0, 1, 0, 1)
        assert nv == fixed.size                                   # the moving volume covers every sample
        assert int(h.sum()) == nv * UNITS
        assert np.array_equal(h.sum(axis=1), np.bincount(bins_of(fixed, 16).ravel(), minlength=16) * UNITS)
    # partial overlap: still 2^15 per valid sample
    M = orc.index_affine(np.concatenate([np.eye(3), [[2.3], [-1.1], [0.4]]], axis=1), (9, 7, 5), (1, 1, 1), (6, 6, 6), (1, 1, 1))
    h, nv = orc.joint_hist_pv(fixed, ph.random_volume((6, 6, 6), 3), M, 16, 0, 1, 0, 1)
    assert 0 < nv < fixed.size and int(h.sum()) == nv * UNITS


def test_pv2_integer_shifts_equal_nearest_and_trilinear():
    cfg = ph.get_config("C1")
    for shift in [(0, 0, 0), (1, -2, 0), (-3, 4, 5), (31, 0, 0), (40, 0, 0)]:
        M = ident_index(shift)
        h, nv = orc.joint_hist_pv(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1)
        for interp in (0, 1):
            h2, nv2 = orc.joint_hist(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, interp)
            assert nv == nv2 and np.array_equal(h, h2.astype(np.uint64) * UNITS)


def test_pv3_worked_2x2x2_example():
    # one fixed voxel (bin 0 of 8); eight moving voxels, voxel (x,y,z) has value (x + 2y + 4z + 0.5)/8 -> bin x+2y+4z
    fixed = np.zeros((1, 1, 1), dtype=np.float32)
    moving = ((np.arange(8).reshape(2, 2, 2) + 0.5) / 8).astype(np.float32)      # [z][y][x]
    h, nv = orc.joint_hist_pv(fixed, moving, ident_index((0.5, 0.5, 0.5)), 8, 0, 1, 0, 1)
    assert nv == 1 and np.array_equal(h[0], np.full(8, 4096, dtype=np.uint64)) and h[1:].sum() == 0
    h, nv = orc.joint_hist_pv(fixed, moving, ident_index((0.25, 0.0, 0.0)), 8, 0, 1, 0, 1)
    want = np.zeros(8, dtype=np.uint64)
    want[0], want[1] = 24 * 32 * 32, 8 * 32 * 32                                   # 0.75 on v000, 0.25 on v100
    assert nv == 1 and np.array_equal(h[0], want)
    # in the half-voxel border the clamped neighbour is the edge voxel itself: c_x = -0.25 -> all weight on v000
    h, nv = orc.joint_hist_pv(fixed, moving, ident_index((-0.25, 0.0, 0.0)), 8, 0, 1, 0, 1)
    assert nv == 1 and h[0, 0] == UNITS
    # through CANON-1: a physical shift of (-0.25, -0.5, -0.5) mm on a 1 mm grid puts the sample at c = (.25, 0, 0)
    T = np.concatenate([np.eye(3), [[-0.25], [-0.5], [-0.5]]], axis=1)
    M = orc.index_affine(T, (1, 1, 1), (1, 1, 1), (2, 2, 2), (1, 1, 1))
    assert np.array_equal(M, ident_index((0.25, 0.0, 0.0)))
    r = orc.eval_batch(fixed, moving, M[None], 8, 0, 1, 0, 1, orc.INTERP_PARTIAL_VOLUME, want_hist=True)
    assert np.array_equal(r["hist"][0][0], want) and r["nvalid"][0] == 1


def test_pv4_brute_force_4cubed():
    """Matrix entries with 8 fractional bits and indices < 4: every product and sum of CANON-2 is exact, so the
    brute force can form the coordinates in plain double arithmetic and must get the fused fp32 result."""
    rng = np.random.default_rng(5)
    fixed = ph.random_volume((4, 4, 4), 11)
    moving = ph.random_volume((4, 4, 4), 12)
    for trial in range(6):
        A = np.eye(3) + rng.integers(-40, 41, (3, 3)) / 256.0
        t = rng.integers(-300, 301, 3) / 256.0
        M = np.concatenate([A, t[:, None]], axis=1).astype(np.float32)
        want, nv_want = brute_force_pv_exact(fixed, moving, M, 8)
        got, nv = orc.joint_hist_pv(fixed, moving, M, 8, 0, 1, 0, 1)
        assert nv == nv_want and nv > 0 and np.array_equal(got, want), trial


def brute_force_pv_exact(fixed, moving, M, nb):
    """Independent Python loops; coordinates in double (exact here: entries have 8 fractional bits, indices < 4)."""
    nzf, nyf, nxf = fixed.shape
    nzm, nym, nxm = moving.shape
    dims = (nxm, nym, nzm)
    h = np.zeros((nb, nb), dtype=np.uint64)
    nv = 0
    Md = M.astype(np.float64)
    for iz in range(nzf):
        for iy in range(nyf):
            for ix in range(nxf):
                c = [Md[k, 0] * ix + Md[k, 1] * iy + Md[k, 2] * iz + Md[k, 3] for k in range(3)]
                if not all(-0.5 <= c[k] < dims[k] - 0.5 for k in range(3)):
                    continue
                lo_hi, wts = [], []
                for k in range(3):
                    g = math.floor(c[k])
                    u = int(math.floor((c[k] - g) * 32.0 + 0.5))
                    lo_hi.append((max(g, 0), min(g + 1, dims[k] - 1)))
                    wts.append((32 - u, u))
                a = int(bins_of(np.array([fixed[iz, iy, ix]]), nb)[0])
                for dz in range(2):
                    for dy in range(2):
                        for dx in range(2):
                            w = wts[0][dx] * wts[1][dy] * wts[2][dz]
                            if w:
                                v = moving[lo_hi[2][dz], lo_hi[1][dy], lo_hi[0][dx]]
                                h[a, int(bins_of(np.array([v]), nb)[0])] += np.uint64(w)
                nv += 1
    return h, nv


def test_pv5_quarter_voxel_shift_is_a_mix_of_two_integer_shifts():
    nb = 32
    fixed = ph.random_volume((6, 5, 4), 21)                       # (nz, ny, nx) = (4, 5, 6)
    moving = ph.random_volume((12, 9, 8), 22)
    fa = bins_of(fixed, nb).ravel()
    mb = bins_of(moving, nb)
    for j in (0, 2, 5):
        h, nv = orc.joint_hist_pv(fixed, moving, ident_index((j + 0.25, 1.0, 2.0)), nb, 0, 1, 0, 1)
        assert nv == fixed.size
        parts = []
        for jj in (j, j + 1):                                    # moving voxel of fixed (ix,iy,iz) is (ix+jj, iy+1, iz+2)
            sub = mb[2:2 + 4, 1:1 + 5, jj:jj + 6].ravel()
            parts.append(np.bincount(fa * nb + sub, minlength=nb * nb).reshape(nb, nb).astype(np.uint64))
        assert np.array_equal(h, np.uint64(24 * 1024) * parts[0] + np.uint64(8 * 1024) * parts[1])


def test_pv6_uint64_entropies_are_scale_free():
    rng = np.random.default_rng(7)
    h = rng.integers(0, 50, (16, 16)).astype(np.uint32)
    h[3] = 0
    q = (0.5, 1.0, 2.0)
    for form in (0, 1):
        a, da = orc.entropies(h, q, form, detail=True)
        b, db = orc.entropies(h.astype(np.uint64) * np.uint64(UNITS), q, form, detail=True)
        assert np.max(np.abs(a - b)) <= 1e-12 and np.max(np.abs(da - db)) <= 1e-12
    assert np.all(orc.entropies(np.zeros((4, 4), dtype=np.uint64), q) == 0.0)
    # and the whole path: MI of a PV evaluation at an integer shift equals the nearest-neighbour MI
    cfg = ph.get_config("C1")
    M = ident_index((1, -2, 0))[None]
    pv = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, orc.INTERP_PARTIAL_VOLUME, q=q)
    nn = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, 0, q=q)
    assert np.max(np.abs(pv["mi"] - nn["mi"])) <= 1e-12 and np.array_equal(pv["nvalid"], nn["nvalid"])


def test_pv7_fraction_rounding_ties_go_up():
    fixed = np.zeros((1, 1, 1), dtype=np.float32)
    moving = np.array([[[0.25, 0.75]]], dtype=np.float32)        # two voxels along x: bins 0 and 1 of 2
    for cx, u in [(1.0 / 64, 1), (1.0 / 64 - 2.0 ** -20, 0), (0.5, 16), (1 - 1.0 / 64, 32), (1 - 1.0 / 64 - 2.0 ** -20, 31)]:
        h, nv = orc.joint_hist_pv(fixed, moving, ident_index((cx, 0.0, 0.0)), 2, 0, 1, 0, 1)
        assert nv == 1 and h[0, 1] == u * 1024 and h[0, 0] == (32 - u) * 1024, (cx, u)


def test_pv_map_peaks_near_the_truth_and_is_smoother_than_nearest():
    """P11 for the PV map: the C1 half-step map peaks within one grid step of the truth (1.5,-2,0.5); between
    two integer shifts the PV value moves in steps no larger than the nearest-neighbour jump."""
    cfg = ph.config_c1(grid_n=9)
    r = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, 0, 1, 0, 1, cfg.family,
                   cfg.lo, cfg.hi, cfg.n, q=(), interp=orc.INTERP_PARTIAL_VOLUME)
    k2, k1, k0 = np.unravel_index(int(r["argmax"][0]), r["map"].shape[1:])
    p = [cfg.lo[d] + k * 0.5 for d, k in enumerate((k0, k1, k2))]
    assert max(abs(p[d] - cfg.truth[d]) for d in range(3)) <= 1.0
