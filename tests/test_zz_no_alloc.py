"""mi_eval_noalloc against the existing path (mi_create + mi_eval_batch), through the C ABI.

mi_eval_noalloc is the entry point for callers that must not let this library allocate device memory:
processes in which another allocator owns the whole GPU (here: torch's caching allocator hands out every
buffer the call touches), or loops that cannot afford the device-wide synchronisation of cudaMalloc.  Its
histogram scratch is one static 256 KB device array that every call reuses, so the things worth checking
are exactly the ones a shared, never-freed array can get wrong:

  * the result equals the existing path's -- histogram and nvalid bit for bit, MI within the tolerance
    the parity tests use (1e-4 nats) -- for both interpolators, with 64 bins (histogram entirely in shared
    memory) and 256 bins (upper rows counted straight into the static array);
  * calls in a row do not see each other's leftovers: transform A, then B (fewer valid samples, so stale
    cells would show), then A again, all on one stream as the header asks;
  * sizes beyond the array are refused with MI_ERR_UNSUPPORTED and a message, not truncated;
  * free device memory does not move across calls once the first call has done its per-device set-up.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_1909_10690_b200 import phantoms as ph

pytestmark = pytest.mark.gpu

MI_TOL = 1e-4   # nats, the bar of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def mi():
    from paper_1909_10690_b200 import build
    build.build()
    from paper_1909_10690_b200 import binding
    return binding


def physical(rot_deg, shift, scale=(1.0, 1.0, 1.0)):
    A = ph.euler_deg_matrix(rot_deg)[:, :3] @ np.diag(scale)
    return np.concatenate([A, np.asarray(shift, dtype=np.float64)[:, None]], axis=1)


def pairs():
    c1 = ph.get_config("C1")
    yield "C1 32^3, 64 bins", c1.fixed, c1.moving, c1.fixed_spacing, c1.moving_spacing, 64
    c3 = ph.config_c3(res=0.25, grid_n=3)
    # different dims and spacings on the two sides; 256 bins -> rows 200..255 bypass shared memory
    moving = np.ascontiguousarray(c3.moving[3:, :, 5:])
    yield "C3/4 cropped, 256 bins", c3.fixed, moving, c3.fixed_spacing, (2.9, 2.8, 3.0), 256


def test_noalloc_equals_existing_path_on_calls_in_a_row(mi):
    import torch
    q = (0.5, 2.0)
    for name, fixed, moving, fs, ms, nb in pairs():
        extent = np.asarray(fixed.shape[::-1]) * np.asarray(fs)
        TA = physical((3.0, -2.0, 1.5), 0.02 * extent)
        TB = physical((-6.0, 4.0, 9.0), (0.35 * extent[0], -0.2 * extent[1], 0.1 * extent[2]), (1.05, 0.95, 1.0))
        seq = [TA, TB, TA]
        d_fixed, d_moving = torch.from_numpy(fixed).cuda(), torch.from_numpy(moving).cuda()
        # everything the call writes is allocated here, by the caller's allocator, before the calls
        d_mi = torch.empty(1 + len(q), dtype=torch.float64, device="cuda")
        d_hist = torch.empty((nb, nb), dtype=torch.int32, device="cuda")
        d_nv = torch.empty(1, dtype=torch.int64, device="cuda")
        with mi.mi_create(fixed, moving, fs, ms, nb, device=0) as ctx:
            for interp in (mi.MI_INTERP_NEAREST, mi.MI_INTERP_TRILINEAR):
                ref_mi, ref_hist, ref_nv = mi.mi_eval_batch(ctx, np.stack(seq), q, interp, hist_out=True, nvalid_out=True)
                assert ref_nv[1] < ref_nv[0], "the second transform should leave part of the overlap empty"
                free_after_first = None
                for k, T in enumerate(seq):
                    d_hist.fill_(-1)
                    mi.mi_eval_noalloc(d_fixed, d_moving, fs, ms, nb, T, q, interp, 0, d_mi, d_hist, d_nv)
                    torch.cuda.synchronize()
                    got_hist = d_hist.cpu().numpy().view(np.uint32)
                    assert np.array_equal(got_hist, ref_hist[k]), (name, interp, k)
                    assert int(d_nv.item()) == int(ref_nv[k]) == int(got_hist.sum(dtype=np.int64))
                    err = float(np.max(np.abs(d_mi.cpu().numpy() - ref_mi[k])))
                    assert err <= MI_TOL, (name, interp, k, err)
                    free = torch.cuda.mem_get_info(0)[0]
                    if free_after_first is None:
                        free_after_first = free      # the first call may load the module / do the set-up
                    else:
                        assert free == free_after_first, "a later call changed the free device memory"


def test_noalloc_pseudo_additive_and_no_optional_outputs(mi):
    import torch
    c1 = ph.get_config("C1")
    T = physical((1.0, 2.0, -3.0), (1.0, -0.5, 0.25))
    q = (0.7, 1.0, 1.5)
    d_fixed, d_moving = torch.from_numpy(c1.fixed).cuda(), torch.from_numpy(c1.moving).cuda()
    d_mi = torch.empty(1 + len(q), dtype=torch.float64, device="cuda")
    with mi.mi_create(c1.fixed, c1.moving, c1.fixed_spacing, c1.moving_spacing, c1.nbins, device=0) as ctx:
        mi.mi_set_tsallis_form(ctx, mi.MI_TSALLIS_PSEUDO_ADDITIVE)
        ref, _, _ = mi.mi_eval_batch(ctx, T[None], q, mi.MI_INTERP_TRILINEAR)
    for _ in range(2):
        d_mi.fill_(float("nan"))
        mi.mi_eval_noalloc(d_fixed, d_moving, c1.fixed_spacing, c1.moving_spacing, c1.nbins, T, q,
                           mi.MI_INTERP_TRILINEAR, mi.MI_TSALLIS_PSEUDO_ADDITIVE, d_mi)
        torch.cuda.synchronize()
        got = d_mi.cpu().numpy()
        assert np.max(np.abs(got - ref[0])) <= MI_TOL
        assert got[2] == got[0], "q == 1 returns the Shannon value"


def test_noalloc_refuses_sizes_beyond_the_static_array(mi):
    import torch
    c1 = ph.get_config("C1")
    d_fixed, d_moving = torch.from_numpy(c1.fixed).cuda(), torch.from_numpy(c1.moving).cuda()
    d_mi = torch.full((16,), 7.0, dtype=torch.float64, device="cuda")
    T = physical((0, 0, 0), (0, 0, 0))
    with pytest.raises(mi.MIError) as e:
        mi.mi_eval_noalloc(d_fixed, d_moving, c1.fixed_spacing, c1.moving_spacing, 257, T, (), mi_out=d_mi)
    assert e.value.status == mi.MI_ERR_UNSUPPORTED and "256" in str(e.value)
    with pytest.raises(mi.MIError) as e:
        mi.mi_eval_noalloc(d_fixed, d_moving, c1.fixed_spacing, c1.moving_spacing, 64, T, (1.5,) * 9, mi_out=d_mi)
    assert e.value.status == mi.MI_ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert bool((d_mi == 7.0).all()), "a refused call must not write its outputs"
