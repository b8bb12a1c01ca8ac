"""Seeded synthetic phantoms standing in for the HCP volumes the paper measured on.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle's tests: it
generates inputs and holds none of the method's arithmetic (no resampling, no binning, no
histogram, no entropy).  It depends on numpy only.

Recipe:
    analytic label function P(physical mm point) -> per-modality intensity table -> x smooth bias
    -> + Gaussian noise -> clamp [0, 1] -> float32.
"moving = fixed transformed by G" means moving(y) = P(G^-1 y), so a map over the family that G
belongs to should peak at T = G.  Noise is position-keyed (splitmix64 of seed and linear voxel
index -> two uniforms -> Box-Muller), so it does not depend on traversal order or chunking.
Volumes are C-contiguous float32 arrays of shape (nz, ny, nx); physical frames are volume-centred
with axes = index axes: voxel i sits at spacing * (i - (n-1)/2).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from functools import lru_cache

import numpy as np

_U64 = np.uint64


def splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output per uint64 input (vectorised, wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = x.astype(_U64) + _U64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)
        return z ^ (z >> _U64(31))


def keyed_uniform(seed: int, idx: np.ndarray, stream: int = 0) -> np.ndarray:
    """U(0,1) float64 keyed by (seed, stream, idx); never exactly 0."""
    with np.errstate(over="ignore"):
        key = splitmix64(np.asarray([(seed * 2 + stream) & 0xFFFFFFFFFFFFFFFF], dtype=_U64))[0]
        bits = splitmix64(idx.astype(_U64) ^ key)
    return ((bits >> _U64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def keyed_normal(seed: int, idx: np.ndarray) -> np.ndarray:
    """N(0,1) float64 keyed by (seed, idx) via Box-Muller."""
    u1 = keyed_uniform(seed, idx, 0)
    u2 = keyed_uniform(seed, idx, 1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


@dataclass(frozen=True)
class Ellipsoid:
    centre: tuple  # mm
    semi: tuple    # mm
    label: int


@dataclass
class Phantom:
    """A label function: background label 0, ellipsoids painted in order (later wins)."""
    ellipsoids: list = field(default_factory=list)

    def labels(self, X, Y, Z) -> np.ndarray:
        lab = np.zeros(np.broadcast(X, Y, Z).shape, dtype=np.int16)
        for e in self.ellipsoids:
            d = (((X - e.centre[0]) / e.semi[0]) ** 2 + ((Y - e.centre[1]) / e.semi[1]) ** 2
                 + ((Z - e.centre[2]) / e.semi[2]) ** 2)
            lab[d <= 1.0] = e.label
        return lab


def render(phantom: Phantom, table, dims, spacing, Ginv=None, sigma=0.0, noise_seed=0,
           bias_amp=0.0, chunk=16) -> np.ndarray:
    """Sample `phantom` on a (nx, ny, nz) grid with `spacing` mm.

    Ginv: 3x4 [A|t] mapping a point y of THIS image's physical frame to the phantom's frame
    (P(G^-1 y)); None = identity.  table: label -> intensity.  Bias is evaluated in this image's
    own frame on coordinates normalised to [-1, 1].
    """
    nx, ny, nz = (int(d) for d in dims)
    sx, sy, sz = (float(s) for s in spacing)
    table = np.asarray(table, dtype=np.float64)
    out = np.empty((nz, ny, nx), dtype=np.float32)
    x = (np.arange(nx, dtype=np.float64) - (nx - 1) / 2.0) * sx
    y = (np.arange(ny, dtype=np.float64) - (ny - 1) / 2.0) * sy
    hx, hy, hz = max(nx * sx / 2.0, 1e-9), max(ny * sy / 2.0, 1e-9), max(nz * sz / 2.0, 1e-9)
    G = None if Ginv is None else np.asarray(Ginv, dtype=np.float64).reshape(3, 4)
    for z0 in range(0, nz, chunk):
        z1 = min(nz, z0 + chunk)
        z = (np.arange(z0, z1, dtype=np.float64) - (nz - 1) / 2.0) * sz
        Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
        if G is None:
            PX, PY, PZ = X, Y, Z
        else:
            PX = G[0, 0] * X + G[0, 1] * Y + G[0, 2] * Z + G[0, 3]
            PY = G[1, 0] * X + G[1, 1] * Y + G[1, 2] * Z + G[1, 3]
            PZ = G[2, 0] * X + G[2, 1] * Y + G[2, 2] * Z + G[2, 3]
        val = table[phantom.labels(PX, PY, PZ)]
        if bias_amp:
            val = val * (1.0 + bias_amp * np.cos(np.pi * (X / hx) / 2 + 0.5)
                         * np.cos(np.pi * (Y / hy) / 2 - 0.3) * np.cos(np.pi * (Z / hz) / 2 + 0.2))
        if sigma:
            lin = (np.arange(z0, z1, dtype=np.int64)[:, None, None] * ny
                   + np.arange(ny, dtype=np.int64)[None, :, None]) * nx + np.arange(nx, dtype=np.int64)
            val = val + sigma * keyed_normal(noise_seed, lin.astype(_U64))
        out[z0:z1] = np.clip(val, 0.0, 1.0).astype(np.float32)
    return out


def invert_affine(T) -> np.ndarray:
    T = np.asarray(T, dtype=np.float64).reshape(3, 4)
    Ai = np.linalg.inv(T[:, :3])
    return np.concatenate([Ai, (-Ai @ T[:, 3])[:, None]], axis=1)


def euler_deg_matrix(p) -> np.ndarray:
    """R = Rz(p2) Ry(p1) Rx(p0), degrees, as a 3x4 [R|0] (input-side helper for the rotated pair)."""
    ax, ay, az = np.deg2rad(np.asarray(p, dtype=np.float64))
    Rx = np.array([[1, 0, 0], [0, np.cos(ax), -np.sin(ax)], [0, np.sin(ax), np.cos(ax)]])
    Ry = np.array([[np.cos(ay), 0, np.sin(ay)], [0, 1, 0], [-np.sin(ay), 0, np.cos(ay)]])
    Rz = np.array([[np.cos(az), -np.sin(az), 0], [np.sin(az), np.cos(az), 0], [0, 0, 1]])
    return np.concatenate([Rz @ Ry @ Rx, np.zeros((3, 1))], axis=1)


# ----------------------------------------------------------------------------------------------
# The five BASELINE.json configs (C1..C5) and small variants for fast tests.
# ----------------------------------------------------------------------------------------------

@dataclass
class Config:
    name: str
    fixed: np.ndarray
    moving: np.ndarray
    fixed_spacing: tuple
    moving_spacing: tuple
    nbins: int
    family: int            # mi_family enum value (0 translation, 1 Euler deg, 2 versor, 3 scale, 4 log scale)
    lo: tuple
    hi: tuple
    n: tuple
    q: tuple
    truth: tuple           # ground-truth parameters G
    ranges: tuple = (0.0, 1.0, 0.0, 1.0)  # fixed_lo, fixed_hi, moving_lo, moving_hi

    @property
    def n_transforms(self) -> int:
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])

    @property
    def evaluations(self) -> int:
        return int(self.fixed.size) * self.n_transforms


def _translation(d):
    return np.concatenate([np.eye(3), np.asarray(d, dtype=np.float64)[:, None]], axis=1)


def c1_phantom() -> Phantom:
    return Phantom([Ellipsoid((0, 0, 0), (13, 11, 12), 1), Ellipsoid((0, 0, 0), (9, 7.5, 8.5), 2),
                    Ellipsoid((0, 0, 0), (5, 4, 4.5), 3)])


def config_c1(grid_n=5, seed=101) -> Config:
    """C1: 32^3, 64 bins, translation grid over +-2 voxels; truth (1.5,-2,0.5)."""
    dims, sp = (32, 32, 32), (1.0, 1.0, 1.0)
    table = [0.0, 0.2, 0.5, 0.8]
    d = (1.5, -2.0, 0.5)
    P = c1_phantom()
    fixed = render(P, table, dims, sp, None, 0.02, seed)
    moving = render(P, table, dims, sp, invert_affine(_translation(d)), 0.02, seed + 1)
    return Config("C1", fixed, moving, sp, sp, 64, 0, (-2, -2, -2), (2, 2, 2), (grid_n,) * 3,
                  (0.5, 2.0), d)


def config_c2(size=128, grid_n=21, half_range=10.0, seed=202) -> Config:
    """C2: size^3 (128), 128 bins, 6 random ellipsoid tissue classes, translation grid."""
    rng = np.random.default_rng(seed)
    scale = size / 128.0
    ell = []
    table = [0.0]
    for k in range(6):
        c = rng.uniform(-30, 30, 3) * scale
        s = rng.uniform(12, 45, 3) * scale
        ell.append(Ellipsoid(tuple(c), tuple(s), k + 1))
        table.append(float(rng.uniform(0, 1)))
    d = tuple(float(v) for v in rng.uniform(-1, 1, 3))
    dims, sp = (size,) * 3, (1.0, 1.0, 1.0)
    P = Phantom(ell)
    fixed = render(P, table, dims, sp, None, 0.03, seed)
    moving = render(P, table, dims, sp, invert_affine(_translation(d)), 0.03, seed + 1)
    r = half_range
    return Config("C2", fixed, moving, sp, sp, 128, 0, (-r,) * 3, (r,) * 3, (grid_n,) * 3, (0.5,), d)


# labels of the head phantom
BG, SKULL, CSF, GM, WM = 0, 1, 2, 3, 4
T1_TABLE = [0.0, 0.10, 0.15, 0.55, 0.80]
T2_TABLE = [0.0, 0.05, 0.90, 0.50, 0.30]


def head_phantom(seed=303, scale=1.0) -> Phantom:
    """Skull/CSF/GM/WM ellipsoid shells plus 24 seeded interior ellipsoids (16 GM, 8 CSF)."""
    rng = np.random.default_rng(seed)
    s = scale
    ell = [Ellipsoid((0, 0, 0), (75 * s, 95 * s, 85 * s), SKULL),
           Ellipsoid((0, 0, 0), (70 * s, 90 * s, 80 * s), CSF),
           Ellipsoid((0, 0, 0), (66 * s, 86 * s, 76 * s), GM),
           Ellipsoid((0, 0, 0), (58 * s, 78 * s, 68 * s), WM)]
    for k in range(24):
        c = rng.uniform(-1, 1, 3) * np.array([40, 55, 45]) * s
        a = rng.uniform(5, 16, 3) * s
        ell.append(Ellipsoid(tuple(c), tuple(a), GM if k < 16 else CSF))
    return Phantom(ell)


def _head_dims(scale):
    """Full size at scale 1; reduced-resolution variants keep the physical field of view."""
    return tuple(max(4, int(round(d * scale))) for d in (260, 311, 260))


def config_c3(res=1.0, grid_n=15, seed=303) -> Config:
    """C3: head phantom (res=1 -> 260x311x260 @0.7 mm), moving rotated (4,-3,2) deg, Euler grid."""
    dims = _head_dims(res)
    sp = (0.7 / res,) * 3
    P = head_phantom(seed)
    G = euler_deg_matrix((4.0, -3.0, 2.0))
    fixed = render(P, T1_TABLE, dims, sp, None, 0.02, seed, bias_amp=0.1)
    moving = render(P, T1_TABLE, dims, sp, invert_affine(G), 0.02, seed + 1, bias_amp=0.1)
    return Config("C3", fixed, moving, sp, sp, 256, 1, (-7, -7, -7), (7, 7, 7), (grid_n,) * 3, (),
                  (4.0, -3.0, 2.0))


def config_c4(res=1.0, grid_n=11, seed=303) -> Config:
    """C4: head phantom, moving scaled (1.05,0.97,1.02), scale grid over [0.9,1.1], five q values."""
    dims = _head_dims(res)
    sp = (0.7 / res,) * 3
    P = head_phantom(seed)
    G = np.concatenate([np.diag([1.05, 0.97, 1.02]), np.zeros((3, 1))], axis=1)
    fixed = render(P, T1_TABLE, dims, sp, None, 0.02, seed, bias_amp=0.1)
    moving = render(P, T1_TABLE, dims, sp, invert_affine(G), 0.02, seed + 1, bias_amp=0.1)
    return Config("C4", fixed, moving, sp, sp, 256, 3, (0.9,) * 3, (1.1,) * 3, (grid_n,) * 3,
                  (0.2, 0.5, 0.8, 1.5, 2.0), (1.05, 0.97, 1.02))


def config_c5(res=1.0, grid_n=41, seed=303) -> Config:
    """C5 (headline): T1-like fixed 260x311x260 @0.7 mm, T2-like moving 182x218x182 @1.0 mm shifted
    (3.2,-4.7,1.1) mm; 256 bins; translation grid 41^3 over +-10 mm."""
    fdims = _head_dims(res)
    mdims = tuple(max(4, int(round(d * res))) for d in (182, 218, 182))
    fsp, msp = (0.7 / res,) * 3, (1.0 / res,) * 3
    P = head_phantom(seed)
    d = (3.2, -4.7, 1.1)
    fixed = render(P, T1_TABLE, fdims, fsp, None, 0.02, seed, bias_amp=0.1)
    moving = render(P, T2_TABLE, mdims, msp, invert_affine(_translation(d)), 0.03, seed + 1,
                    bias_amp=0.1)
    return Config("C5", fixed, moving, fsp, msp, 256, 0, (-10,) * 3, (10,) * 3, (grid_n,) * 3, (), d)


def config_c5all(res=1.0, grid_n=41, seed=303, salt=0.02) -> Config:
    """C5 with EVERY fixed bin populated, as real MR data at 256 bins is (the label phantom leaves the bins
    between its tissue means empty, so at most 192 of 256 fixed bins hold voxels): a seeded 2 % of the fixed
    voxels are replaced by uniform values in [0, 1].  The z kernel's shared histogram holds 209 rows at 256
    bins, so the rarest fixed bins take the rare-voxel kernel, the histograms are written to global memory and a
    separate entropy launch follows -- the path real data takes.  Stress input for bench.py --config C5ALL."""
    c = config_c5(res, grid_n, seed)
    idx = np.arange(c.fixed.size, dtype=_U64)
    pick = keyed_uniform(seed + 7, idx, 0) < salt
    vals = keyed_uniform(seed + 7, idx, 1).astype(np.float32)
    fixed = c.fixed.copy().reshape(-1)
    fixed[pick] = vals[pick]
    return Config("C5ALL", fixed.reshape(c.fixed.shape), c.moving, c.fixed_spacing, c.moving_spacing, c.nbins, c.family,
                  c.lo, c.hi, c.n, c.q, c.truth)


def config_paper51(res=1.0, grid_n=51, seed=303) -> Config:
    """Paper-shaped context run (not one of BASELINE.json's configs): the paper maps "the same image on
    both fixed and moving" and gives 51 positions over +-25 mm per axis as its example
    of a translation map: the T1-like head phantom against itself, 51^3 translations,
    Shannon + Tsallis q = 0.5, 2.0 (the orders of Figs. 4-5)."""
    dims = _head_dims(res)
    sp = (0.7 / res,) * 3
    fixed = render(head_phantom(seed), T1_TABLE, dims, sp, None, 0.02, seed, bias_amp=0.1)
    return Config("PAPER51", fixed, fixed, sp, sp, 256, 0, (-25,) * 3, (25,) * 3, (grid_n,) * 3, (0.5, 2.0),
                  (0.0, 0.0, 0.0))


def config_paperrot(res=1.0, grid_n=15, seed=303) -> Config:
    """The paper's rotation parameter space (section 3.2): the versor ball -- p = axis * sin(theta/2),
    "all points outside the sphere with radius = 1 are mapped to the sphere surface" -- so the map covers the
    cube [-1, 1]^3 and every rotation up to 180 degrees.  Same image on both sides; an odd grid
    puts the gold standard (0, 0, 0) on a node.  Shannon + Tsallis q = 0.5, 1.1 (Fig. 9's best order), 2.0."""
    dims = _head_dims(res)
    sp = (0.7 / res,) * 3
    fixed = render(head_phantom(seed), T1_TABLE, dims, sp, None, 0.02, seed, bias_amp=0.1)
    return Config("PAPERROT", fixed, fixed, sp, sp, 256, 2, (-1.0,) * 3, (1.0,) * 3, (grid_n,) * 3, (0.5, 1.1, 2.0),
                  (0.0, 0.0, 0.0))


def config_paperscale(res=1.0, grid_n=15, seed=303, half_range=0.5) -> Config:
    """The paper's scale parameter space (section 3.3): zero-centred parameters, "parameters
    greater than zero" = a moving image scaled bigger -- family SCALE_LOG, factor = exp(p).  The paper prints no
    range; +-0.5 (factors 0.61 .. 1.65) is this repository's choice.  Same image on both sides; Shannon +
    Tsallis q = 0.5, 2.0 (one order on each side of 1, Fig. 14)."""
    dims = _head_dims(res)
    sp = (0.7 / res,) * 3
    fixed = render(head_phantom(seed), T1_TABLE, dims, sp, None, 0.02, seed, bias_amp=0.1)
    return Config("PAPERSCALE", fixed, fixed, sp, sp, 256, 4, (-half_range,) * 3, (half_range,) * 3, (grid_n,) * 3,
                  (0.5, 2.0), (0.0, 0.0, 0.0))


@lru_cache(maxsize=8)
def get_config(name: str, **kw) -> Config:
    """Cached access: get_config('C5'), get_config('C3', res=0.25, grid_n=5) ..."""
    return {"C1": config_c1, "C2": config_c2, "C3": config_c3, "C4": config_c4,
            "C5": config_c5, "C5ALL": config_c5all, "PAPER51": config_paper51, "PAPERROT": config_paperrot,
            "PAPERSCALE": config_paperscale}[name](**kw)


def ramp_volume(dims, coeffs) -> np.ndarray:
    """moving(i,j,k) = alpha*i + beta*j + gamma*k + delta (pin P6 input)."""
    nx, ny, nz = dims
    a, b, g, d = coeffs
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return (a * i + b * j + g * k + d).astype(np.float32)


def random_volume(dims, seed, lo=0.0, hi=1.0) -> np.ndarray:
    nx, ny, nz = dims
    u = keyed_uniform(seed, np.arange(nx * ny * nz, dtype=_U64))
    return (lo + (hi - lo) * u).astype(np.float32).reshape(nz, ny, nx)
