"""CPU oracle for the exhaustive MI map -- TEST INFRASTRUCTURE, not product code.

Thin ctypes wrapper around `oracle/mi_oracle.cpp` (built on demand by `oracle/build.py`).  Only
`tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this package; the CUDA library and its Python binding never do (and this package never
imports them).  All arithmetic lives in the C++ file; this module only marshals numpy arrays.

Array conventions: volumes are C-contiguous float32 numpy arrays of shape (nz, ny, nx) -- x fastest
-- and "dims" are always (nx, ny, nz), as in SURVEY.md section 8(b).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = None

INTERP_NEAREST = 0
INTERP_TRILINEAR = 1
INTERP_PARTIAL_VOLUME = 2
PV_UNITS_PER_VOXEL = 1 << 15      # reading A21: per-axis weights in 1/32 voxel, a sample adds 32^3 units
TSALLIS_ADDITIVE = 0
TSALLIS_PSEUDO_ADDITIVE = 1
FAMILY_TRANSLATION = 0
FAMILY_ROTATION_EULER_DEG = 1
FAMILY_ROTATION_VERSOR = 2
FAMILY_SCALE = 3
FAMILY_SCALE_LOG = 4

_f32p = C.POINTER(C.c_float)
_f64p = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)
_i64p = C.POINTER(C.c_int64)
_u32p = C.POINTER(C.c_uint32)
_u64p = C.POINTER(C.c_uint64)
_u8p = C.POINTER(C.c_uint8)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_index_affine.argtypes = [_f64p, _i32p, _f64p, _i32p, _f64p, _f32p]
        L.orc_index_affine.restype = None
        L.orc_family_matrix.argtypes = [C.c_int, _f64p, _f64p]
        L.orc_family_matrix.restype = C.c_int
        L.orc_prebin.argtypes = [_f32p, C.c_int64, C.c_int, C.c_float, C.c_float, _i32p]
        L.orc_prebin.restype = None
        L.orc_resample.argtypes = [_i32p, _f32p, _i32p, _f32p, C.c_int, _f32p, _u8p]
        L.orc_resample.restype = None
        hist_args = [_f32p, _i32p, _f32p, _i32p, None, C.c_int, C.c_float, C.c_float, C.c_float,
                     C.c_float, C.c_int, _u32p]
        L.orc_joint_hist.argtypes = hist_args[:4] + [_f32p] + hist_args[5:]
        L.orc_joint_hist.restype = C.c_int64
        L.orc_joint_hist_f64.argtypes = hist_args[:4] + [_f64p] + hist_args[5:]
        L.orc_joint_hist_f64.restype = C.c_int64
        L.orc_entropies.argtypes = [_u32p, C.c_int, _f64p, C.c_int, C.c_int, _f64p, _f64p]
        L.orc_entropies.restype = None
        L.orc_eval_batch.argtypes = [_f32p, _i32p, _f32p, _i32p, _f32p, C.c_int64, C.c_int,
                                     C.c_float, C.c_float, C.c_float, C.c_float, C.c_int, _f64p,
                                     C.c_int, C.c_int, _f64p, _u32p, _i64p]
        L.orc_eval_batch.restype = C.c_int
        L.orc_map.argtypes = [_f32p, _i32p, _f64p, _f32p, _i32p, _f64p, C.c_int, C.c_float,
                              C.c_float, C.c_float, C.c_float, C.c_int, _f64p, _f64p, _i32p, _f64p,
                              C.c_int, C.c_int, C.c_int, _f64p, _i64p]
        L.orc_map.restype = C.c_int
        L.orc_eval_batch_masked.argtypes = [_f32p, _i32p, _f32p, _i32p, _f32p, C.c_int64, C.c_int,
                                            C.c_float, C.c_float, C.c_float, C.c_float, C.c_int, _f64p,
                                            C.c_int, C.c_int, _u8p, _f64p, _u32p, _i64p]
        L.orc_eval_batch_masked.restype = C.c_int
        L.orc_map_masked.argtypes = [_f32p, _i32p, _f64p, _f32p, _i32p, _f64p, C.c_int, C.c_float,
                                     C.c_float, C.c_float, C.c_float, C.c_int, _f64p, _f64p, _i32p, _f64p,
                                     C.c_int, C.c_int, C.c_int, _u8p, _f64p, _i64p]
        L.orc_map_masked.restype = C.c_int
        L.orc_entropies_u64.argtypes = [_u64p, C.c_int, _f64p, C.c_int, C.c_int, _f64p, _f64p]
        L.orc_entropies_u64.restype = None
        L.orc_joint_hist_pv.argtypes = [_f32p, _i32p, _f32p, _i32p, _f32p, C.c_int, C.c_float, C.c_float, C.c_float,
                                        C.c_float, _u8p, _u64p]
        L.orc_joint_hist_pv.restype = C.c_int64
        L.orc_eval_batch_pv.argtypes = [_f32p, _i32p, _f32p, _i32p, _f32p, C.c_int64, C.c_int, C.c_float, C.c_float,
                                        C.c_float, C.c_float, _f64p, C.c_int, C.c_int, _u8p, _f64p, _u64p, _i64p]
        L.orc_eval_batch_pv.restype = C.c_int
        L.orc_max_threads.argtypes = []
        L.orc_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def _vol(v):
    v = np.ascontiguousarray(v, dtype=np.float32)
    assert v.ndim == 3
    return v


def _dims(v):
    nz, ny, nx = v.shape
    return np.array([nx, ny, nz], dtype=np.int32)


def _q(q):
    q = np.ascontiguousarray(np.atleast_1d(np.asarray(q if q is not None else [], dtype=np.float64)))
    return q, int(q.size)


def max_threads() -> int:
    return int(lib().orc_max_threads())


def index_affine(T, fixed_dims, fixed_spacing, moving_dims, moving_spacing) -> np.ndarray:
    """CANON-1: physical 3x4 [A|t] (double) -> index-space 3x4 [M|m0] (float32)."""
    T = np.ascontiguousarray(T, dtype=np.float64).reshape(12)
    fd = np.ascontiguousarray(fixed_dims, dtype=np.int32)
    md = np.ascontiguousarray(moving_dims, dtype=np.int32)
    fs = np.ascontiguousarray(fixed_spacing, dtype=np.float64)
    ms = np.ascontiguousarray(moving_spacing, dtype=np.float64)
    out = np.empty(12, dtype=np.float32)
    lib().orc_index_affine(_p(T, _f64p), _p(fd, _i32p), _p(fs, _f64p), _p(md, _i32p), _p(ms, _f64p),
                           _p(out, _f32p))
    return out.reshape(3, 4)


def family_matrix(family: int, p) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float64).reshape(3)
    T = np.empty(12, dtype=np.float64)
    rc = lib().orc_family_matrix(int(family), _p(p, _f64p), _p(T, _f64p))
    if rc != 0:
        raise ValueError("unknown family %r" % (family,))
    return T.reshape(3, 4)


def prebin(vol, nb: int, lo: float, hi: float) -> np.ndarray:
    v = np.ascontiguousarray(vol, dtype=np.float32)
    out = np.empty(v.size, dtype=np.int32)
    lib().orc_prebin(_p(v.reshape(-1), _f32p), v.size, int(nb), float(lo), float(hi), _p(out, _i32p))
    return out.reshape(v.shape)


def resample(fixed_dims, moving, M, interp: int):
    """value, valid = v(T(x)) on the fixed grid; shapes (nz, ny, nx) of the fixed volume."""
    mv = _vol(moving)
    fd = np.ascontiguousarray(fixed_dims, dtype=np.int32)
    md = _dims(mv)
    M = np.ascontiguousarray(M, dtype=np.float32).reshape(12)
    shape = (int(fd[2]), int(fd[1]), int(fd[0]))
    value = np.empty(shape, dtype=np.float32)
    valid = np.empty(shape, dtype=np.uint8)
    lib().orc_resample(_p(fd, _i32p), _p(mv, _f32p), _p(md, _i32p), _p(M, _f32p), int(interp),
                       _p(value, _f32p), _p(valid, _u8p))
    return value, valid.astype(bool)


def joint_hist(fixed, moving, M, nb, flo, fhi, mlo, mhi, interp, f64_coords: bool = False):
    """hist (nb, nb) uint32 [row = fixed bin, col = moving bin], nvalid."""
    fx, mv = _vol(fixed), _vol(moving)
    fd, md = _dims(fx), _dims(mv)
    hist = np.empty((nb, nb), dtype=np.uint32)
    if f64_coords:
        M = np.ascontiguousarray(M, dtype=np.float64).reshape(12)
        nv = lib().orc_joint_hist_f64(_p(fx, _f32p), _p(fd, _i32p), _p(mv, _f32p), _p(md, _i32p),
                                      _p(M, _f64p), int(nb), flo, fhi, mlo, mhi, int(interp),
                                      _p(hist, _u32p))
    else:
        M = np.ascontiguousarray(M, dtype=np.float32).reshape(12)
        nv = lib().orc_joint_hist(_p(fx, _f32p), _p(fd, _i32p), _p(mv, _f32p), _p(md, _i32p),
                                  _p(M, _f32p), int(nb), flo, fhi, mlo, mhi, int(interp),
                                  _p(hist, _u32p))
    return hist, int(nv)


def entropies(hist, q=None, form: int = TSALLIS_ADDITIVE, detail: bool = False):
    """[Shannon I, I_q...] (and [H(A), H(B), H(A,B)] if detail) from a joint histogram (uint32 counts, or
    uint64 partial-volume weight units when the array's dtype is uint64)."""
    wide = np.asarray(hist).dtype == np.uint64
    h = np.ascontiguousarray(hist, dtype=np.uint64 if wide else np.uint32)
    nb = h.shape[0]
    assert h.shape == (nb, nb)
    qa, nq = _q(q)
    out = np.empty(1 + nq, dtype=np.float64)
    det = np.empty(3, dtype=np.float64)
    if wide:
        lib().orc_entropies_u64(_p(h, _u64p), nb, _p(qa, _f64p), nq, int(form), _p(out, _f64p), _p(det, _f64p))
    else:
        lib().orc_entropies(_p(h, _u32p), nb, _p(qa, _f64p), nq, int(form), _p(out, _f64p), _p(det, _f64p))
    return (out, det) if detail else out


def joint_hist_pv(fixed, moving, M, nb, flo, fhi, mlo, mhi, mask=None):
    """Partial-volume joint histogram (reading A21): (nb, nb) uint64 in units of 2^-15 voxel, nvalid."""
    fx, mv = _vol(fixed), _vol(moving)
    fd, md = _dims(fx), _dims(mv)
    M = np.ascontiguousarray(M, dtype=np.float32).reshape(12)
    hist = np.empty((nb, nb), dtype=np.uint64)
    mk = _mask(mask, fx)
    nv = lib().orc_joint_hist_pv(_p(fx, _f32p), _p(fd, _i32p), _p(mv, _f32p), _p(md, _i32p), _p(M, _f32p), int(nb),
                                 flo, fhi, mlo, mhi, _p(mk.reshape(-1), _u8p) if mk is not None else None,
                                 _p(hist, _u64p))
    return hist, int(nv)


def _mask(mask, fx):
    """uint8 mask of the fixed volume's shape (non-zero = the voxel takes part), or None."""
    if mask is None:
        return None
    m = np.ascontiguousarray(np.asarray(mask) != 0, dtype=np.uint8)
    assert m.shape == fx.shape
    return m


def eval_batch(fixed, moving, M, nb, flo, fhi, mlo, mhi, interp, q=None, form=TSALLIS_ADDITIVE,
               want_hist: bool = False, mask=None):
    """M: (N, 3, 4) float32 index-space transforms -> dict(mi (N,1+nq), nvalid (N,), hist?, threads).
    mask: optional subset of the fixed voxels that takes part (reading A19)."""
    fx, mv = _vol(fixed), _vol(moving)
    fd, md = _dims(fx), _dims(mv)
    M = np.ascontiguousarray(M, dtype=np.float32).reshape(-1, 12)
    N = M.shape[0]
    qa, nq = _q(q)
    mi = np.empty((N, 1 + nq), dtype=np.float64)
    nvalid = np.empty(N, dtype=np.int64)
    mk = _mask(mask, fx)
    if int(interp) == INTERP_PARTIAL_VOLUME:      # uint64 histograms in units of 2^-15 voxel
        hist = np.empty((N, nb, nb), dtype=np.uint64) if want_hist else None
        threads = lib().orc_eval_batch_pv(_p(fx, _f32p), _p(fd, _i32p), _p(mv, _f32p), _p(md, _i32p), _p(M, _f32p), N,
                                          int(nb), flo, fhi, mlo, mhi, _p(qa, _f64p), nq, int(form),
                                          _p(mk.reshape(-1), _u8p) if mk is not None else None, _p(mi, _f64p),
                                          _p(hist, _u64p) if want_hist else None, _p(nvalid, _i64p))
        return {"mi": mi, "nvalid": nvalid, "hist": hist, "threads": int(threads)}
    hist = np.empty((N, nb, nb), dtype=np.uint32) if want_hist else None
    threads = lib().orc_eval_batch_masked(_p(fx, _f32p), _p(fd, _i32p), _p(mv, _f32p), _p(md, _i32p),
                                          _p(M, _f32p), N, int(nb), flo, fhi, mlo, mhi, int(interp),
                                          _p(qa, _f64p), nq, int(form),
                                          _p(mk.reshape(-1), _u8p) if mk is not None else None, _p(mi, _f64p),
                                          _p(hist, _u32p) if want_hist else None, _p(nvalid, _i64p))
    return {"mi": mi, "nvalid": nvalid, "hist": hist, "threads": int(threads)}


def physical_to_index(T, fixed_dims, fixed_spacing, moving_dims, moving_spacing) -> np.ndarray:
    """(N,3,4) physical transforms -> (N,3,4) float32 index-space transforms (CANON-1 per row)."""
    T = np.ascontiguousarray(T, dtype=np.float64).reshape(-1, 3, 4)
    return np.stack([index_affine(t, fixed_dims, fixed_spacing, moving_dims, moving_spacing) for t in T])


def mi_map(fixed, fixed_spacing, moving, moving_spacing, nb, flo, fhi, mlo, mhi, family, lo, hi, n,
           q=None, form=TSALLIS_ADDITIVE, interp=INTERP_TRILINEAR, mask=None):
    """Exhaustive map: dict(map (1+nq, n2, n1, n0), argmax (1+nq,), threads)."""
    fx, mv = _vol(fixed), _vol(moving)
    fd, md = _dims(fx), _dims(mv)
    fs = np.ascontiguousarray(fixed_spacing, dtype=np.float64)
    ms = np.ascontiguousarray(moving_spacing, dtype=np.float64)
    lo = np.ascontiguousarray(lo, dtype=np.float64)
    hi = np.ascontiguousarray(hi, dtype=np.float64)
    n = np.ascontiguousarray(n, dtype=np.int32)
    qa, nq = _q(q)
    out = np.empty((1 + nq, int(n[2]), int(n[1]), int(n[0])), dtype=np.float64)
    am = np.empty(1 + nq, dtype=np.int64)
    mk = _mask(mask, fx)
    threads = lib().orc_map_masked(_p(fx, _f32p), _p(fd, _i32p), _p(fs, _f64p), _p(mv, _f32p), _p(md, _i32p),
                                   _p(ms, _f64p), int(nb), flo, fhi, mlo, mhi, int(family), _p(lo, _f64p),
                                   _p(hi, _f64p), _p(n, _i32p), _p(qa, _f64p), nq, int(form), int(interp),
                                   _p(mk.reshape(-1), _u8p) if mk is not None else None,
                                   _p(out, _f64p), _p(am, _i64p))
    return {"map": out, "argmax": am, "threads": int(threads)}


def grid_nodes_index_affines(fixed_dims, fixed_spacing, moving_dims, moving_spacing, family, lo, hi, n, nodes):
    """Index-space transforms (len(nodes), 3, 4) float32 of grid nodes (k0, k1, k2) of the map grid
    (lo, hi, n): parameter k on axis d is lo[d] + k (hi[d]-lo[d])/(n[d]-1) in double (include/mi.h), then the
    family generator and CANON-1 -- the same composition orc_map does for every node."""
    T = []
    for node in nodes:
        p = [float(lo[d]) if int(n[d]) == 1 else float(lo[d]) + float(node[d]) * (float(hi[d]) - float(lo[d])) / float(int(n[d]) - 1)
             for d in range(3)]
        T.append(family_matrix(family, p))
    return physical_to_index(np.stack(T), fixed_dims, fixed_spacing, moving_dims, moving_spacing)


def mi_map_range(fixed, fixed_spacing, moving, moving_spacing, nb, flo, fhi, mlo, mhi, family, lo, hi, n, begin, end,
                 q=None, form=TSALLIS_ADDITIVE, interp=INTERP_TRILINEAR, mask=None):
    """The nodes begin[d] <= k_d < end[d] of the exhaustive map over the grid (lo, hi, n):
    map (1+nq, m2, m1, m0) with p0 fastest -- each node evaluated by orc_eval_batch."""
    fx, mv = _vol(fixed), _vol(moving)
    nodes = [(k0, k1, k2) for k2 in range(begin[2], end[2]) for k1 in range(begin[1], end[1])
             for k0 in range(begin[0], end[0])]
    M = grid_nodes_index_affines(_dims(fx), fixed_spacing, _dims(mv), moving_spacing, family, lo, hi, n, nodes)
    r = eval_batch(fx, mv, M, nb, flo, fhi, mlo, mhi, interp, q=q, form=form, mask=mask)
    m = [end[d] - begin[d] for d in range(3)]
    return np.ascontiguousarray(r["mi"].T).reshape(r["mi"].shape[1], m[2], m[1], m[0])
