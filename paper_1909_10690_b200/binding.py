"""ctypes binding of libmi_b200.so -- same names as include/mi.h, argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  There is NO fallback: if the shared
library has not been built (`python -m paper_1909_10690_b200.build`) importing this module raises,
and on a box without a CUDA device every compute call raises MIError(MI_ERR_CUDA).

Arrays may be numpy arrays (host) or torch tensors (host or CUDA); their data pointers are passed
straight through.  Volumes are (nz, ny, nx) C-contiguous float32 (x fastest), dims are (nx, ny, nz).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmi_b200.so")

MI_OK, MI_ERR_INVALID_ARG, MI_ERR_UNSUPPORTED, MI_ERR_OUT_OF_MEMORY, MI_ERR_CUDA, MI_ERR_INTERNAL = range(6)
MI_INTERP_NEAREST, MI_INTERP_TRILINEAR, MI_INTERP_PARTIAL_VOLUME = 0, 1, 2
MI_PV_UNITS_PER_VOXEL = 1 << 15
MI_TSALLIS_ADDITIVE, MI_TSALLIS_PSEUDO_ADDITIVE = 0, 1
(MI_FAMILY_TRANSLATION, MI_FAMILY_ROTATION_EULER_DEG, MI_FAMILY_ROTATION_VERSOR, MI_FAMILY_SCALE,
 MI_FAMILY_SCALE_LOG) = range(5)
_STATUS = {0: "MI_OK", 1: "MI_ERR_INVALID_ARG", 2: "MI_ERR_UNSUPPORTED", 3: "MI_ERR_OUT_OF_MEMORY",
           4: "MI_ERR_CUDA", 5: "MI_ERR_INTERNAL"}

(MI_OPT_SEPARABLE, MI_OPT_FUSE_ENTROPY, MI_OPT_BIN_MODE_MAX, MI_OPT_ZHIST_ROWS_MAX, MI_OPT_ZHIST_PAD, MI_OPT_XY_BUDGET_MB,
 MI_OPT_SEP_HIST_BUDGET_MB, MI_OPT_HIST_BUDGET_MB, MI_OPT_GENERIC_PAD, MI_OPT_GENERIC_SMEM_KB, MI_OPT_GENERIC_TY_LOG2,
 MI_OPT_GENERIC_UNROLL, MI_OPT_ZHIST_MATCH_ANY, MI_OPT_GENERIC_GATHER, MI_OPT_GENERIC_THREADS,
 MI_OPT_GENERIC_SLAB_MB) = range(16)
(MI_INFO_NUM_SMS, MI_INFO_BIN_MODE, MI_INFO_ZHIST_ROWS, MI_INFO_RARE_VOXELS, MI_INFO_GENERIC_ROWS,
 MI_INFO_LAST_PATH, MI_INFO_LAST_UPDATES_ISSUED, MI_INFO_QUADS_BUILT) = range(100, 108)

EXPORTS = ("mi_create", "mi_set_tsallis_form", "mi_set_fixed_mask", "mi_eval_batch", "mi_eval_batch_pv", "mi_eval_noalloc", "mi_map", "mi_map_range", "mi_set_option",
           "mi_get_option", "mi_destroy", "mi_last_error",
           "mi_family_matrix", "mi_index_affine", "mi_get_bins", "mi_last_timing", "mi_release_cached_memory",
           "mi_map_gradient", "mi_map_basins", "mi_compose_matrix", "mi_seed_from_map", "mi_multimetric_gradient", "mi_register", "mi_pv_min_delta",
           "mi_probe_shared_atomic_rate", "mi_probe_gather_rate", "mi_version")

if not os.path.exists(LIB_PATH):
    raise ImportError("%s is missing: build it with `python -m paper_1909_10690_b200.build` "
                      "(there is no CPU fallback)" % LIB_PATH)
_lib = C.CDLL(LIB_PATH)

_vp = C.c_void_p
_lib.mi_create.argtypes = [C.POINTER(_vp), _vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, C.c_float, C.c_float,
                           C.c_float, C.c_float, C.c_int32, _vp]
_lib.mi_create.restype = C.c_int
_lib.mi_set_tsallis_form.argtypes = [_vp, C.c_int]
_lib.mi_set_tsallis_form.restype = C.c_int
_lib.mi_set_fixed_mask.argtypes = [_vp, _vp]
_lib.mi_set_fixed_mask.restype = C.c_int
_lib.mi_eval_batch.argtypes = [_vp, _vp, C.c_int64, _vp, C.c_int32, C.c_int, _vp, _vp, _vp]
_lib.mi_eval_batch.restype = C.c_int
_lib.mi_eval_batch_pv.argtypes = [_vp, _vp, C.c_int64, _vp, C.c_int32, _vp, _vp, _vp]
_lib.mi_eval_batch_pv.restype = C.c_int
_lib.mi_eval_noalloc.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, C.c_float, C.c_float, C.c_float, C.c_float,
                                 _vp, _vp, C.c_int32, C.c_int, C.c_int, _vp, _vp, _vp, C.c_int32, _vp]
_lib.mi_eval_noalloc.restype = C.c_int
_lib.mi_map.argtypes = [_vp, C.c_int, _vp, _vp, _vp, _vp, C.c_int32, C.c_int, _vp, _vp]
_lib.mi_map.restype = C.c_int
_lib.mi_map_range.argtypes = [_vp, C.c_int, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int32, C.c_int, _vp, _vp, _vp]
_lib.mi_map_range.restype = C.c_int
_lib.mi_set_option.argtypes = [_vp, C.c_int, C.c_int64]
_lib.mi_set_option.restype = C.c_int
_lib.mi_get_option.argtypes = [_vp, C.c_int, _vp]
_lib.mi_get_option.restype = C.c_int
_lib.mi_destroy.argtypes = [_vp]
_lib.mi_destroy.restype = None
_lib.mi_last_error.argtypes = [_vp]
_lib.mi_last_error.restype = C.c_char_p
_lib.mi_family_matrix.argtypes = [C.c_int, _vp, _vp]
_lib.mi_family_matrix.restype = C.c_int
_lib.mi_index_affine.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
_lib.mi_index_affine.restype = C.c_int
_lib.mi_get_bins.argtypes = [_vp, C.c_int32, _vp]
_lib.mi_get_bins.restype = C.c_int
_lib.mi_release_cached_memory.argtypes = [C.c_int32]
_lib.mi_release_cached_memory.restype = C.c_int
_lib.mi_seed_from_map.argtypes = [C.c_int, _vp, _vp, _vp, C.c_int64, _vp]
_lib.mi_seed_from_map.restype = C.c_int
_lib.mi_compose_matrix.argtypes = [_vp, _vp]
_lib.mi_compose_matrix.restype = C.c_int
_lib.mi_multimetric_gradient.argtypes = [_vp, _vp, _vp, C.c_double, C.c_int, _vp, _vp]
_lib.mi_multimetric_gradient.restype = C.c_int
_lib.mi_pv_min_delta.argtypes = [_vp, _vp]
_lib.mi_pv_min_delta.restype = C.c_int
_lib.mi_register.argtypes = [_vp, _vp, _vp, _vp, _vp, C.c_int32, C.c_double, C.c_int, _vp, _vp, _vp]
_lib.mi_register.restype = C.c_int
_lib.mi_map_gradient.argtypes = [_vp, _vp, _vp, _vp, _vp, C.c_int32, _vp]
_lib.mi_map_gradient.restype = C.c_int
_lib.mi_map_basins.argtypes = [_vp, _vp, C.c_int32, C.c_int32, C.c_int64, _vp, _vp, _vp, C.c_int32, _vp]
_lib.mi_map_basins.restype = C.c_int
_lib.mi_last_timing.argtypes = [_vp, _vp, _vp]
_lib.mi_last_timing.restype = C.c_int
_lib.mi_probe_shared_atomic_rate.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, _vp]
_lib.mi_probe_shared_atomic_rate.restype = C.c_int
_lib.mi_probe_gather_rate.argtypes = [_vp, _vp, C.c_int32, C.c_int32, _vp]
_lib.mi_probe_gather_rate.restype = C.c_int
_lib.mi_version.argtypes = []
_lib.mi_version.restype = C.c_char_p


class MIError(RuntimeError):
    def __init__(self, status, msg=""):
        self.status = int(status)
        super().__init__("%s: %s" % (_STATUS.get(self.status, str(status)), msg))


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _ptr(x):
    """Data pointer of a numpy array / torch tensor / raw int, or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if _is_torch(x):
        assert x.is_contiguous()
        return x.data_ptr()
    assert x.flags["C_CONTIGUOUS"]
    return x.ctypes.data


def _f64(a, n=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1))
    assert n is None or a.size == n
    return a


def _i32(a, n):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.int32).reshape(-1))
    assert a.size == n
    return a


def _volume(v):
    """float32, contiguous; keeps torch tensors (host or CUDA) as they are."""
    if _is_torch(v):
        import torch
        assert v.dtype == torch.float32 and v.dim() == 3
        return v.contiguous()
    v = np.ascontiguousarray(v, dtype=np.float32)
    assert v.ndim == 3
    return v


class MIContext:
    """Owns an mi_ctx*; also remembers the shapes the marshalling needs."""

    def __init__(self, handle, nbins, fixed_dims, moving_dims):
        self.handle = handle
        self.nbins = int(nbins)
        self.fixed_dims = tuple(int(d) for d in fixed_dims)
        self.moving_dims = tuple(int(d) for d in moving_dims)

    def __del__(self):
        try:
            mi_destroy(self)
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        mi_destroy(self)


def _check(ctx, status):
    if status != MI_OK:
        h = ctx.handle if isinstance(ctx, MIContext) else None
        raise MIError(status, (_lib.mi_last_error(h) or b"").decode())


def mi_version() -> str:
    return _lib.mi_version().decode()


def mi_last_error(ctx=None) -> str:
    return (_lib.mi_last_error(ctx.handle if ctx is not None else None) or b"").decode()


def mi_create(fixed, moving, fixed_spacing, moving_spacing, nbins, fixed_lo=0.0, fixed_hi=1.0,
              moving_lo=0.0, moving_hi=1.0, device=0, cuda_stream=None, fixed_dims=None,
              moving_dims=None) -> MIContext:
    fixed, moving = _volume(fixed), _volume(moving)
    if fixed_dims is None:
        fixed_dims = tuple(fixed.shape)[::-1]
    if moving_dims is None:
        moving_dims = tuple(moving.shape)[::-1]
    fd, md = _i32(fixed_dims, 3), _i32(moving_dims, 3)
    fs, ms = _f64(fixed_spacing, 3), _f64(moving_spacing, 3)
    h = _vp()
    st = _lib.mi_create(C.byref(h), _ptr(fixed), _ptr(fd), _ptr(fs), _ptr(moving), _ptr(md), _ptr(ms),
                        int(nbins), float(fixed_lo), float(fixed_hi), float(moving_lo), float(moving_hi),
                        int(device), cuda_stream)
    if st != MI_OK:
        raise MIError(st, mi_last_error(None))
    return MIContext(h, nbins, fd, md)


def mi_destroy(ctx) -> None:
    if ctx is not None and getattr(ctx, "handle", None):
        h, ctx.handle = ctx.handle, None
        _lib.mi_destroy(h)


def mi_set_tsallis_form(ctx, form) -> None:
    _check(ctx, _lib.mi_set_tsallis_form(ctx.handle, int(form)))


def mi_eval_batch(ctx, T, q=(), interp=MI_INTERP_TRILINEAR, mi_out=None, hist_out=None, nvalid_out=None):
    """T: (N,3,4) physical [A|t].  Outputs: pass arrays/tensors to fill, True to allocate a host
    array, None/False to skip (mi_out is always produced).  Returns (mi, hist, nvalid)."""
    T = _f64(T)
    N = T.size // 12
    assert T.size == N * 12
    q = _f64(q)
    nq = q.size
    nb = ctx.nbins
    if mi_out is None or mi_out is True:
        mi_out = np.empty((N, 1 + nq), dtype=np.float64)
    if hist_out is True:
        hist_out = np.empty((N, nb, nb), dtype=np.uint32)
    elif hist_out is False:
        hist_out = None
    if nvalid_out is True:
        nvalid_out = np.empty(N, dtype=np.int64)
    elif nvalid_out is False:
        nvalid_out = None
    st = _lib.mi_eval_batch(ctx.handle, _ptr(T), N, _ptr(q) if nq else None, nq, int(interp), _ptr(mi_out),
                            _ptr(hist_out), _ptr(nvalid_out))
    _check(ctx, st)
    return mi_out, hist_out, nvalid_out


def mi_eval_batch_pv(ctx, T, q=(), mi_out=None, hist_out=None, nvalid_out=None):
    """Partial-volume interpolation: as mi_eval_batch, histograms are (N, nbins, nbins) uint64 in units of
    2^-15 voxel.  Returns (mi, hist, nvalid)."""
    T = _f64(T)
    N = T.size // 12
    assert T.size == N * 12
    q = _f64(q)
    nq = q.size
    nb = ctx.nbins
    if mi_out is None or mi_out is True:
        mi_out = np.empty((N, 1 + nq), dtype=np.float64)
    if hist_out is True:
        hist_out = np.empty((N, nb, nb), dtype=np.uint64)
    elif hist_out is False:
        hist_out = None
    if nvalid_out is True:
        nvalid_out = np.empty(N, dtype=np.int64)
    elif nvalid_out is False:
        nvalid_out = None
    st = _lib.mi_eval_batch_pv(ctx.handle, _ptr(T), N, _ptr(q) if nq else None, nq, _ptr(mi_out), _ptr(hist_out),
                               _ptr(nvalid_out))
    _check(ctx, st)
    return mi_out, hist_out, nvalid_out


def mi_eval_noalloc(fixed, moving, fixed_spacing, moving_spacing, nbins, T, q=(), interp=MI_INTERP_TRILINEAR,
                    form=0, mi_out=None, hist_out=None, nvalid_out=None, fixed_lo=0.0, fixed_hi=1.0, moving_lo=0.0,
                    moving_hi=1.0, device=0, cuda_stream=None):
    """One transform's MI (and optionally its joint histogram) for callers that must not let the library
    allocate device memory -- the GPU is owned by another allocator, or cudaMalloc's device-wide sync is
    not acceptable in their loop.  The histogram scratch is a 256 KB static array inside the library, so
    nbins <= 256 and nq <= 8, and calls overlapping on one GPU would race (see include/mi.h).

    fixed, moving: float32 CUDA tensors (z, y, x).  mi_out (1+nq float64), hist_out (nbins x nbins, uint32
    stored in an int32 tensor) and nvalid_out (1 int64) are CUDA tensors the caller allocated; mi_out is
    required, the others may be None.  Work is only queued on the stream: synchronise before reading."""
    assert _is_torch(fixed) and _is_torch(moving) and fixed.is_cuda and moving.is_cuda, "device tensors only"
    fixed, moving = _volume(fixed), _volume(moving)
    assert mi_out is not None, "mi_out must be a caller-allocated CUDA tensor"
    T = _f64(T, 12)
    q = _f64(q)
    fd = _i32(tuple(fixed.shape)[::-1], 3)
    md = _i32(tuple(moving.shape)[::-1], 3)
    fs, ms = _f64(fixed_spacing, 3), _f64(moving_spacing, 3)
    if cuda_stream is None:
        import torch
        cuda_stream = torch.cuda.current_stream(device).cuda_stream
    st = _lib.mi_eval_noalloc(_ptr(fixed), _ptr(fd), _ptr(fs), _ptr(moving), _ptr(md), _ptr(ms), int(nbins),
                              float(fixed_lo), float(fixed_hi), float(moving_lo), float(moving_hi), _ptr(T),
                              _ptr(q) if q.size else None, q.size, int(interp), int(form), _ptr(mi_out),
                              _ptr(hist_out), _ptr(nvalid_out), int(device), cuda_stream)
    if st != MI_OK:
        raise MIError(st, mi_last_error(None))
    return mi_out, hist_out, nvalid_out


def mi_map(ctx, family, lo, hi, n, q=(), interp=MI_INTERP_TRILINEAR, map_out=None, argmax_out=None):
    """Returns (map (1+nq, n2, n1, n0) float64, argmax (1+nq,) int64)."""
    lo, hi, n = _f64(lo, 3), _f64(hi, 3), _i32(n, 3)
    q = _f64(q)
    nq = q.size
    if map_out is None:
        map_out = np.empty((1 + nq, int(n[2]), int(n[1]), int(n[0])), dtype=np.float64)
    if argmax_out is None:
        argmax_out = np.empty(1 + nq, dtype=np.int64)
    st = _lib.mi_map(ctx.handle, int(family), _ptr(lo), _ptr(hi), _ptr(n), _ptr(q) if nq else None, nq,
                     int(interp), _ptr(map_out), _ptr(argmax_out))
    _check(ctx, st)
    return map_out, argmax_out


def mi_map_range(ctx, family, lo, hi, n, begin=None, end=None, q=(), interp=MI_INTERP_TRILINEAR, map_out=None,
                 argmax_out=None, hist_out=None):
    """Sub-box [begin, end) of the grid (lo, hi, n); node parameters are those of the whole grid.
    Returns (map (1+nq, m2, m1, m0), argmax (1+nq,) into the sub-box, hist or None); hist_out=True
    allocates (m2*m1*m0, nbins, nbins) uint32 on the host."""
    lo, hi, n = _f64(lo, 3), _f64(hi, 3), _i32(n, 3)
    begin = _i32(begin, 3) if begin is not None else np.zeros(3, dtype=np.int32)
    end = _i32(end, 3) if end is not None else n.copy()
    m = [int(end[d] - begin[d]) for d in range(3)]
    q = _f64(q)
    nq = q.size
    if map_out is None:
        map_out = np.empty((1 + nq, m[2], m[1], m[0]), dtype=np.float64)
    if argmax_out is None:
        argmax_out = np.empty(1 + nq, dtype=np.int64)
    if hist_out is True:
        hist_out = np.empty((m[2] * m[1] * m[0], ctx.nbins, ctx.nbins), dtype=np.uint32)
    elif hist_out is False:
        hist_out = None
    st = _lib.mi_map_range(ctx.handle, int(family), _ptr(lo), _ptr(hi), _ptr(n), _ptr(begin), _ptr(end),
                           _ptr(q) if nq else None, nq, int(interp), _ptr(map_out), _ptr(argmax_out), _ptr(hist_out))
    _check(ctx, st)
    return map_out, argmax_out, hist_out


def mi_set_option(ctx, key, value) -> None:
    _check(ctx, _lib.mi_set_option(ctx.handle, int(key), int(value)))


def mi_get_option(ctx, key) -> int:
    out = np.zeros(1, dtype=np.int64)
    _check(ctx, _lib.mi_get_option(ctx.handle, int(key), _ptr(out)))
    return int(out[0])


def mi_family_matrix(family, p) -> np.ndarray:
    p = _f64(p, 3)
    T = np.empty(12, dtype=np.float64)
    st = _lib.mi_family_matrix(int(family), _ptr(p), _ptr(T))
    if st != MI_OK:
        raise MIError(st, "mi_family_matrix")
    return T.reshape(3, 4)


def mi_index_affine(T, fixed_dims, fixed_spacing, moving_dims, moving_spacing) -> np.ndarray:
    T = _f64(T, 12)
    fd, md = _i32(fixed_dims, 3), _i32(moving_dims, 3)
    fs, ms = _f64(fixed_spacing, 3), _f64(moving_spacing, 3)
    M = np.empty(12, dtype=np.float32)
    st = _lib.mi_index_affine(_ptr(T), _ptr(fd), _ptr(fs), _ptr(md), _ptr(ms), _ptr(M))
    if st != MI_OK:
        raise MIError(st, "mi_index_affine")
    return M.reshape(3, 4)


def mi_get_bins(ctx, which: int) -> np.ndarray:
    dims = ctx.fixed_dims if which == 0 else ctx.moving_dims
    out = np.empty((dims[2], dims[1], dims[0]), dtype=np.uint8 if ctx.nbins <= 256 else np.uint16)
    _check(ctx, _lib.mi_get_bins(ctx.handle, int(which), _ptr(out)))
    return out


def mi_last_timing(ctx):
    """(ms[5], launches[5]) of the last eval/map call: setup, resample+hist, entropy, map assembly, and
    the dominant histogram kernel alone (a part of resample+hist)."""
    ms = np.zeros(5, dtype=np.float32)
    ln = np.zeros(5, dtype=np.int64)
    _check(ctx, _lib.mi_last_timing(ctx.handle, _ptr(ms), _ptr(ln)))
    return ms, ln


class _BasinStats(C.Structure):
    _fields_ = [("n_extrema", C.c_int64), ("target", C.c_int64), ("target_label", C.c_int64),
                ("captured", C.c_int64), ("capture_fraction", C.c_double), ("max_steps", C.c_int32),
                ("iterations", C.c_int32)]


def _map_channel(m):
    """One channel of a map: (n2, n1, n0) float64, numpy or torch (host or CUDA); returns (array, n)."""
    if _is_torch(m):
        import torch
        assert m.dtype == torch.float64 and m.dim() == 3
        m = m.contiguous()
    else:
        m = np.ascontiguousarray(m, dtype=np.float64)
        assert m.ndim == 3
    return m, _i32(tuple(m.shape)[::-1], 3)


def _like(m, shape, dtype_np, dtype_torch_name):
    if _is_torch(m):
        import torch
        return torch.empty(shape, dtype=getattr(torch, dtype_torch_name), device=m.device)
    return np.empty(shape, dtype=dtype_np)


def mi_map_gradient(m, lo, hi, device=0, cuda_stream=None):
    """Finite-difference gradient field (3, n2, n1, n0) of one map channel, in the memory of `m`."""
    m, n = _map_channel(m)
    out = _like(m, (3,) + tuple(m.shape), np.float64, "float64")
    lo, hi = _f64(lo, 3), _f64(hi, 3)          # keep the arrays alive across the call
    _check(None, _lib.mi_map_gradient(_ptr(m), _ptr(n), _ptr(lo), _ptr(hi), _ptr(out), int(device), cuda_stream))
    return out


def mi_map_basins(m, direction=1, connectivity=26, target=-1, device=0, cuda_stream=None, want_arrays=True):
    """Discrete steepest ascent (+1) / descent (-1) basins of one map channel: dict with label, steps
    (in the memory of `m`, None if not wanted) and the mi_basin_stats fields."""
    m, n = _map_channel(m)
    label = _like(m, tuple(m.shape), np.int64, "int64") if want_arrays else None
    steps = _like(m, tuple(m.shape), np.int32, "int32") if want_arrays else None
    st = _BasinStats()
    _check(None, _lib.mi_map_basins(_ptr(m), _ptr(n), int(direction), int(connectivity), int(target), _ptr(label),
                                    _ptr(steps), C.addressof(st), int(device), cuda_stream))
    out = {k: getattr(st, k) for k, _ in _BasinStats._fields_}
    out["label"], out["steps"] = label, steps
    return out


def mi_set_fixed_mask(ctx, mask) -> None:
    """mask: None (all voxels) or an array / tensor of the fixed volume's shape, non-zero = voxel takes part."""
    if mask is None:
        _check(ctx, _lib.mi_set_fixed_mask(ctx.handle, None))
        return
    if _is_torch(mask):
        import torch
        m = (mask != 0).to(torch.uint8).contiguous()
    else:
        m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.uint8)
    assert tuple(m.shape) == ctx.fixed_dims[::-1]
    _check(ctx, _lib.mi_set_fixed_mask(ctx.handle, _ptr(m)))


def mi_seed_from_map(family, lo, hi, n, index) -> np.ndarray:
    """Nine registration parameters of map node `index` (e.g. an arg max of mi_map): the p0 of mi_register."""
    lo, hi, n = _f64(lo, 3), _f64(hi, 3), _i32(n, 3)
    p = np.empty(9, dtype=np.float64)
    st = _lib.mi_seed_from_map(int(family), _ptr(lo), _ptr(hi), _ptr(n), int(index), _ptr(p))
    if st != MI_OK:
        raise MIError(st, "mi_seed_from_map")
    return p


def mi_compose_matrix(p) -> np.ndarray:
    p = _f64(p, 9)
    T = np.empty(12, dtype=np.float64)
    st = _lib.mi_compose_matrix(_ptr(p), _ptr(T))
    if st != MI_OK:
        raise MIError(st, "mi_compose_matrix")
    return T.reshape(3, 4)


def mi_multimetric_gradient(ctx, p, delta, q, interp=MI_INTERP_TRILINEAR):
    """(grad[9], values[2]) -- Tsallis_q differences for the translation parameters, Shannon for the rest."""
    p, delta = _f64(p, 9), _f64(delta, 9)
    grad, vals = np.empty(9, dtype=np.float64), np.empty(2, dtype=np.float64)
    _check(ctx, _lib.mi_multimetric_gradient(ctx.handle, _ptr(p), _ptr(delta), float(q), int(interp), _ptr(grad),
                                             _ptr(vals)))
    return grad, vals


class _RegisterInfo(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("steps", C.c_double * 3), ("values", C.c_double * 2)]


def mi_pv_min_delta(ctx) -> np.ndarray:
    """Smallest finite-difference steps (9 doubles, units of p) MI_INTERP_PARTIAL_VOLUME resolves on this context."""
    out = np.empty(9, dtype=np.float64)
    _check(ctx, _lib.mi_pv_min_delta(ctx.handle, _ptr(out)))
    return out


def mi_register(ctx, p0, delta, step0, step_min, max_iter, q, interp=MI_INTERP_TRILINEAR):
    """Regular-step multi-metric ascent: dict(p, iterations, trace (iterations + 1, 9), steps, values)."""
    p0, delta, step0, step_min = _f64(p0, 9), _f64(delta, 9), _f64(step0, 3), _f64(step_min, 3)
    p = np.empty(9, dtype=np.float64)
    trace = np.zeros((int(max_iter) + 1, 9), dtype=np.float64)
    info = _RegisterInfo()
    _check(ctx, _lib.mi_register(ctx.handle, _ptr(p0), _ptr(delta), _ptr(step0), _ptr(step_min), int(max_iter), float(q),
                                 int(interp), _ptr(p), _ptr(trace), C.addressof(info)))
    return {"p": p, "iterations": int(info.iterations), "trace": trace[: info.iterations + 1].copy(),
            "steps": np.array(list(info.steps)), "values": np.array(list(info.values))}


def mi_release_cached_memory(device=0) -> None:
    st = _lib.mi_release_cached_memory(int(device))
    if st != MI_OK:
        raise MIError(st, "mi_release_cached_memory")


def mi_probe_gather_rate(ctx, T, reps=3) -> float:
    """Samples per second of the generic kernel without its histogram updates on transforms T (n, 3, 4)."""
    T = _f64(T)
    n = T.size // 12
    out = np.zeros(1, dtype=np.float64)
    _check(ctx, _lib.mi_probe_gather_rate(ctx.handle, _ptr(T), n, int(reps), _ptr(out)))
    return float(out[0])


def mi_probe_shared_atomic_rate(device=0, nbins=256, pattern=1, iters=4096) -> float:
    out = np.zeros(1, dtype=np.float64)
    st = _lib.mi_probe_shared_atomic_rate(int(device), int(nbins), int(pattern), int(iters), _ptr(out))
    if st != MI_OK:
        raise MIError(st, "mi_probe_shared_atomic_rate")
    return float(out[0])
