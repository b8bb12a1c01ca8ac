"""Host-side checks of the C-ABI boundary that need no GPU: the library loads, exports what
include/mi.h declares, validates arguments, refuses to compute without a device (no CPU fallback),
and its host step a2 (CANON-1, family generators) equals the oracle's bit for bit."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1909_10690_b200 import build
    build.build()
    from paper_1909_10690_b200 import binding
    return binding


def _has_gpu():
    import torch
    return torch.cuda.is_available()


def test_library_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "mi.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(mi_[a-z_0-9]+)\s*\(", header))
    assert {"mi_create", "mi_eval_batch", "mi_map", "mi_destroy", "mi_last_error"} <= declared
    dll = ctypes.CDLL(lib.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(dll, name), name
    assert declared == set(lib.EXPORTS)
    assert "sm_100a" in lib.mi_version()


def test_binding_never_imports_the_oracle():
    for fn in ("binding.py", "__init__.py", "build.py", "phantoms.py"):
        src = open(os.path.join(ROOT, "paper_1909_10690_b200", fn)).read()
        assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), fn
    for fn in os.listdir(os.path.join(ROOT, "paper_1909_10690_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_1909_10690_b200", "csrc", fn)).read(), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp")):
            assert "paper_1909_10690_b200" not in open(os.path.join(ROOT, "oracle", fn)).read().replace(
                "paper_1909_10690_b200/csrc", ""), fn


def test_library_reads_no_environment_variable():
    """Kernel selection is a function of the C-ABI arguments and mi_set_option only."""
    for fn in os.listdir(os.path.join(ROOT, "paper_1909_10690_b200", "csrc")):
        assert "getenv" not in open(os.path.join(ROOT, "paper_1909_10690_b200", "csrc", fn)).read(), fn
    assert "environ" not in open(os.path.join(ROOT, "paper_1909_10690_b200", "binding.py")).read()


def test_index_affine_bit_for_bit_against_oracle(lib):
    rng = np.random.default_rng(0)
    geoms = [((260, 311, 260), (0.7, 0.7, 0.7), (182, 218, 182), (1.0, 1.0, 1.0)),
             ((32, 32, 32), (1.0, 1.0, 1.0), (32, 32, 32), (1.0, 1.0, 1.0)),
             ((37, 21, 13), (0.9, 1.3, 2.1), (19, 44, 30), (1.7, 0.6, 1.1))]
    for fd, fs, md, ms in geoms:
        for _ in range(200):
            A = np.eye(3) + rng.uniform(-0.5, 0.5, (3, 3))
            t = rng.uniform(-30, 30, 3)
            T = np.concatenate([A, t[:, None]], axis=1)
            a = lib.mi_index_affine(T, fd, fs, md, ms)
            b = orc.index_affine(T, fd, fs, md, ms)
            assert a.tobytes() == b.tobytes()
    Tid = np.concatenate([np.eye(3), np.zeros((3, 1))], axis=1)
    assert np.array_equal(lib.mi_index_affine(Tid, (260, 311, 260), (0.7,) * 3, (260, 311, 260), (0.7,) * 3),
                          np.eye(3, 4, dtype=np.float32))


def test_family_matrix_equals_oracle(lib):
    rng = np.random.default_rng(1)
    for fam in range(5):
        for _ in range(50):
            p = rng.uniform(-1.5, 1.5, 3) * (20 if fam in (0, 1) else 1)
            a = lib.mi_family_matrix(fam, p)
            b = orc.family_matrix(fam, p)
            assert np.array_equal(a, b), (fam, p)
    with pytest.raises(lib.MIError):
        lib.mi_family_matrix(9, (0, 0, 0))
    with pytest.raises(lib.MIError):
        lib.mi_family_matrix(0, (np.nan, 0, 0))


def test_compose_matrix_bit_for_bit_against_oracle(lib):
    from oracle import multimetric as mm
    rng = np.random.default_rng(4)
    for _ in range(50):
        p = np.concatenate([rng.uniform(-20, 20, 3), rng.uniform(-40, 40, 3), rng.uniform(0.5, 1.5, 3)])
        assert np.array_equal(lib.mi_compose_matrix(p), mm.compose_matrix(p))
    with pytest.raises(lib.MIError):
        lib.mi_compose_matrix([0, 0, 0, 0, np.nan, 0, 1, 1, 1])


def test_seed_from_map_equals_oracle(lib):
    from oracle import multimetric as mm
    lo, hi, n = (-0.3, -0.2, -0.25), (0.3, 0.25, 0.2), (5, 4, 3)
    for fam in range(5):
        for index in range(0, 60, 7):
            a, b = lib.mi_seed_from_map(fam, lo, hi, n, index), mm.seed_from_map(fam, lo, hi, n, index)
            # exp / asin / atan2 come from two maths libraries (libm, numpy's SIMD loops): an ulp, not a bit pattern
            assert np.array_equal(a, b) if fam not in (2, 4) else np.max(np.abs(a - b)) <= 1e-12, (fam, index)
    for bad in (-1, 60):
        with pytest.raises(lib.MIError):
            lib.mi_seed_from_map(0, lo, hi, n, bad)


def test_create_validates_arguments(lib):
    v = np.zeros((4, 4, 4), dtype=np.float32)
    sp = (1.0, 1.0, 1.0)
    cases = [dict(nbins=1), dict(fixed_spacing=(0.0, 1, 1)), dict(moving_spacing=(1, np.inf, 1)),
             dict(fixed_lo=1.0, fixed_hi=1.0), dict(moving_lo=2.0, moving_hi=1.0),
             dict(fixed_dims=(0, 4, 4))]
    for kw in cases:
        args = dict(fixed=v, moving=v, fixed_spacing=sp, moving_spacing=sp, nbins=16)
        args.update(kw)
        with pytest.raises(lib.MIError) as ei:
            lib.mi_create(**args)
        assert ei.value.status == lib.MI_ERR_INVALID_ARG, kw
    with pytest.raises(lib.MIError) as ei:
        lib.mi_create(v, v, sp, sp, 4097)
    assert ei.value.status == lib.MI_ERR_UNSUPPORTED


def test_no_cpu_fallback_without_a_device(lib):
    if _has_gpu():
        pytest.skip("a CUDA device is present")
    v = np.zeros((4, 4, 4), dtype=np.float32)
    with pytest.raises(lib.MIError) as ei:
        lib.mi_create(v, v, (1, 1, 1), (1, 1, 1), 16)
    assert ei.value.status == lib.MI_ERR_CUDA
    assert lib.mi_last_error(None) != ""
    with pytest.raises(lib.MIError) as ei:
        lib.mi_probe_shared_atomic_rate(0, 64, 0, 16)
    assert ei.value.status == lib.MI_ERR_CUDA
