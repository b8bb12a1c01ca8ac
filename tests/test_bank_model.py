"""The shared-memory bank model behind the headline roofline, checked on the CPU.

A warp-wide `red.shared.add.u32` takes as many passes ("wavefronts") of the shared-memory crossbar as the fullest
of the 32 four-byte banks holds DISTINCT addresses; lanes on one address are merged by the hardware.  ncu confirms
the model on the probe kernel (profiles/r2c_ncu.md: 3.530 wavefronts per update for independent uniform bins --
the expected maximum load of 32 balls in 32 bins -- 1.000 for lane-distinct banks) and on zhist_kernel (2.95 on the
C5 data).  This test applies the model to the z kernel's own lane-to-column mapping on a reduced-resolution C5 pair
(numpy / scipy only; neither the oracle nor the CUDA library is involved) and pins what DESIGN.md section 10 states:
real data costs less than independent uniform bins (same-address merges), and neither the row pad nor a
permutation of the columns moves the figure by more than a few per cent.
"""
import numpy as np
import pytest
from scipy.ndimage import map_coordinates

from paper_1909_10690_b200 import phantoms as ph

NB = 256
ROWS_DUMP = 192          # columns outside the moving volume count into a dump row


def wavefronts(addr):
    """addr: (R, 32) word addresses of R warp-wide updates -> mean over R of max_bank #distinct addresses."""
    a = np.sort(addr, axis=1)
    first = np.ones_like(a, dtype=bool)
    first[:, 1:] = a[:, 1:] != a[:, :-1]
    bank = np.where(first, a % 32, 32)
    cnt = np.zeros((a.shape[0], 33), np.int32)
    np.add.at(cnt, (np.repeat(np.arange(a.shape[0]), 32), bank.ravel()), 1)
    return float(cnt[:, :32].max(axis=1).mean())


@pytest.fixture(scope="module")
def c5_cells():
    cfg = ph.get_config("C5", res=0.5, grid_n=3)
    F, Mv = cfg.fixed, cfg.moving
    nz, ny, nx = F.shape
    fb = np.clip(np.floor(F * NB), 0, NB - 1).astype(np.int64)
    cnt = np.bincount(fb.ravel(), minlength=NB)
    rank = np.empty(NB, np.int64)
    rank[np.argsort(-cnt, kind="stable")] = np.arange(NB)          # rows are ranked by population (DESIGN 5.1)
    fa = rank[fb]
    fs, ms = cfg.fixed_spacing[0], cfg.moving_spacing[0]

    def c(n_f, n_m, t):
        return (fs * (np.arange(n_f) - (n_f - 1) / 2) + t) / ms + (n_m - 1) / 2
    zs = np.arange(10, nz - 10, 9)
    Z, Y, X = np.meshgrid(c(nz, Mv.shape[0], 1.0)[zs], c(ny, Mv.shape[1], -4.5), c(nx, Mv.shape[2], 3.0), indexing="ij")
    b = np.clip(np.floor(map_coordinates(Mv, [Z, Y, X], order=1, mode="nearest") * NB), 0, NB - 1).astype(np.int64)
    ok = ((Z >= -0.5) & (Z < Mv.shape[0] - 0.5) & (Y >= -0.5) & (Y < Mv.shape[1] - 0.5) & (X >= -0.5) & (X < Mv.shape[2] - 0.5))
    ncol = ny * nx
    colpitch = (ncol + 255) // 256 * 256
    A = np.full((len(zs), colpitch), ROWS_DUMP, np.int64)
    B = np.zeros((len(zs), colpitch), np.int64)
    A[:, :ncol] = np.where(ok, fa[zs], ROWS_DUMP).reshape(len(zs), -1)
    B[:, :ncol] = b.reshape(len(zs), -1)
    # zhist_kernel: thread = 8 columns (two groups of 4 adjacent ones, 128 apart), update k of a warp takes column k
    # of each lane: col = wcol + 4 lane + (k & 3) + 128 (k >> 2), wcol = (tile 1024 + warp 32) 8
    lanes = np.array([w * 256 + np.arange(32) * 4 + (k & 3) + 128 * (k >> 2) for w in range(colpitch // 256) for k in range(8)])
    return A, B, lanes


def cost(A, B, lanes, pad, perm=None):
    if perm is not None:
        A, B = A[:, perm], B[:, perm]
    addr = (A[:, lanes] * (NB + pad) + B[:, lanes]).reshape(-1, 32)
    return wavefronts(addr)


def test_real_data_costs_less_than_independent_uniform_bins(c5_cells):
    A, B, lanes = c5_cells
    rng = np.random.default_rng(3)
    uniform = wavefronts(rng.integers(0, NB * (NB + 9), size=(20000, 32)))
    assert abs(uniform - 3.53) < 0.05                      # the roofline's denominator (ncu: 3.530)
    real = cost(A, B, lanes, 9)
    assert 2.6 < real < 3.2, real                          # ncu on the full-size C5 map: 2.95
    assert real < uniform - 0.3


def test_no_row_pad_and_no_column_order_changes_the_cost_much(c5_cells):
    A, B, lanes = c5_cells
    base = cost(A, B, lanes, 9)
    pads = {pad: cost(A, B, lanes, pad) for pad in (3, 5, 7, 11, 13, 17, 41)}
    assert max(abs(v - base) for v in pads.values()) < 0.12 * base, pads
    assert cost(A, B, lanes, 32) > base + 0.3              # an even pad of 32 puts one column of all rows on one bank
    rng = np.random.default_rng(4)
    rand = cost(A, B, lanes, 9, rng.permutation(A.shape[1]))
    by_tissue = cost(A, B, lanes, 9, np.argsort((A > 16).mean(axis=0), kind="stable"))
    assert rand > base - 0.05                              # scattering the columns does not help
    assert by_tissue > 0.88 * base, (by_tissue, base)      # grouping them by tissue share: a few per cent at most
