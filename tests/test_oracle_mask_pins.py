"""Pins of the oracle's fixed-voxel mask (reading A19: the sampled subset of PAPER.md:212's random-sampling
question is an input): additivity over a partition, the all-ones and all-zeros masks, brute force."""
import numpy as np

import oracle as orc
from paper_1909_10690_b200 import phantoms as ph


def _setup():
    cfg = ph.get_config("C1")
    T = np.stack([orc.family_matrix(0, (1.5, -2, 0.5)), orc.family_matrix(1, (3, -2, 5)), orc.family_matrix(3, (1.1, 0.9, 1.05))])
    M = orc.physical_to_index(T, (32,) * 3, cfg.fixed_spacing, (32,) * 3, cfg.moving_spacing)
    mask = ph.keyed_uniform(77, np.arange(cfg.fixed.size, dtype=np.uint64)).reshape(cfg.fixed.shape) < 0.3
    return cfg, M, mask


def test_mask_histograms_add_up_over_a_partition():
    cfg, M, mask = _setup()
    for interp in (0, 1):
        full = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, interp, want_hist=True)
        a = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, interp, want_hist=True, mask=mask)
        b = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, interp, want_hist=True, mask=~mask)
        assert np.array_equal(a["hist"] + b["hist"], full["hist"])
        assert np.array_equal(a["nvalid"] + b["nvalid"], full["nvalid"])
        assert np.all(a["nvalid"] < 0.4 * full["nvalid"]) and np.all(a["nvalid"] > 0.2 * full["nvalid"])
        ones = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, interp, q=(0.5,), want_hist=True, mask=np.ones_like(mask))
        ref = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, interp, q=(0.5,), want_hist=True)
        assert np.array_equal(ones["hist"], ref["hist"]) and np.array_equal(ones["mi"], ref["mi"])
        none = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, interp, q=(2.0,), mask=np.zeros_like(mask))
        assert np.all(none["nvalid"] == 0) and np.all(none["mi"] == 0.0)


def test_masked_histogram_equals_numpy_bincount_of_the_selected_voxels():
    cfg, M, mask = _setup()
    for interp in (0, 1):
        val, valid = orc.resample(cfg.fixed.shape[::-1], cfg.moving, M[1], interp)
        sel = (valid != 0) & mask
        a = orc.prebin(cfg.fixed, 64, 0, 1)[sel]
        b = orc.prebin(val, 64, 0, 1)[sel]
        want = np.bincount(a * 64 + b, minlength=64 * 64).reshape(64, 64)
        got = orc.eval_batch(cfg.fixed, cfg.moving, M[1:2], 64, 0, 1, 0, 1, interp, want_hist=True, mask=mask)
        assert np.array_equal(got["hist"][0], want) and got["nvalid"][0] == sel.sum()


def test_masked_map_equals_masked_batch():
    cfg, _, mask = _setup()
    r = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, 64, 0, 1, 0, 1, 0, (-1, -1, -1), (1, 1, 1),
                   (3, 2, 3), q=(0.5,), mask=mask)
    T = np.stack([orc.family_matrix(0, (k0 - 1.0, -1.0 + 2.0 * k1, k2 - 1.0)) for k2 in range(3) for k1 in range(2) for k0 in range(3)])
    M = orc.physical_to_index(T, (32,) * 3, cfg.fixed_spacing, (32,) * 3, cfg.moving_spacing)
    b = orc.eval_batch(cfg.fixed, cfg.moving, M, 64, 0, 1, 0, 1, 1, q=(0.5,), mask=mask)
    assert np.array_equal(r["map"].reshape(2, -1).T, b["mi"])
    full = orc.mi_map(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, 64, 0, 1, 0, 1, 0, (-1, -1, -1), (1, 1, 1),
                      (3, 2, 3), q=(0.5,))
    assert not np.array_equal(full["map"], r["map"])
