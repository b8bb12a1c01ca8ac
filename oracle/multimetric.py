"""CPU oracle for the multi-metric finite-difference gradient -- TEST INFRASTRUCTURE, not product code
(same rules as oracle/__init__.py).

The paper's strategy (section 4): "we can use the same histogram to produce the
Shannon and Tsallis results [so] the reasonable strategy is to use multiple algorithms in the
gradient descent.  In this way we can use the Tsallis in the translation gradients and Shannon in
the rotation and scale gradients".  The paper gives no parameterisation of the combined transform
and no difference rule; the readings taken (A18):

* nine parameters p = (tx, ty, tz [mm], ax, ay, az [deg], sx, sy, sz [factors]); the transform is
  y = R(a) S(s) x + t with R = Rz Ry Rx (the map family ROTATION_EULER_DEG), S = diag(s) (family
  SCALE), both about the volume centre (the physical origin, CANON-1), translation last;
* component k of the gradient is the central difference (F_k(p + d_k e_k) - F_k(p - d_k e_k)) / (2 d_k)
  with F_k = the Tsallis MI of order q for the three translation parameters and the Shannon MI for
  the six rotation and scale parameters; all 2*9 + 1 transforms are evaluated from one joint
  histogram each, which yields both metrics (the "same histogram" of PAPER.md:199);
* d_k <= 0 skips component k (gradient 0).

`register` (reading A20) is the loop of Fig. 1 around that gradient; its step rule is this build's --
the paper prints none -- so against the paper it is "parity unpinned"; it is pinned on its own rule and
against the exhaustive map's maximum.

Pins (tests/test_oracle_multimetric_pins.py): the composition against scipy's rotations and the map
families; every gradient component against the central difference of an exhaustive map of the same
family computed by oracle.mi_map + map_analysis.map_gradient (channel, sign, step and parameter
order); the values at p.
"""
from __future__ import annotations

import numpy as np

import oracle as _orc

N_PARAMS = 9
TRANSLATION_PARAMS = (0, 1, 2)          # use the Tsallis channel
SHANNON_PARAMS = (3, 4, 5, 6, 7, 8)     # rotation and scale: use the Shannon channel


def compose_matrix(p) -> np.ndarray:
    """Physical 3x4 [A|t] of the nine parameters: A = R(ax,ay,az) diag(sx,sy,sz), t = (tx,ty,tz)."""
    p = np.asarray(p, dtype=np.float64).reshape(N_PARAMS)
    R = _orc.family_matrix(_orc.FAMILY_ROTATION_EULER_DEG, p[3:6])[:, :3]
    A = R * p[6:9][None, :]              # column j scaled by s_j: one product per entry
    return np.concatenate([A, p[0:3][:, None]], axis=1)


def multimetric_gradient(fixed, fixed_spacing, moving, moving_spacing, nbins, ranges, p, delta, q,
                         interp=_orc.INTERP_TRILINEAR, form=_orc.TSALLIS_ADDITIVE):
    """Returns (grad[9], values[2] = (Shannon, Tsallis_q) at p)."""
    p = np.asarray(p, dtype=np.float64).reshape(N_PARAMS)
    delta = np.asarray(delta, dtype=np.float64).reshape(N_PARAMS)
    Ts = [compose_matrix(p)]
    for k in range(N_PARAMS):
        for sgn in (+1.0, -1.0):
            pk = p.copy()
            pk[k] = p[k] + sgn * delta[k]
            Ts.append(compose_matrix(pk))
    T = np.stack(Ts)
    fd, md = fixed.shape[::-1], moving.shape[::-1]
    M = _orc.physical_to_index(T, fd, fixed_spacing, md, moving_spacing)
    vals = _orc.eval_batch(fixed, moving, M, nbins, *ranges, interp, q=(float(q),), form=form)["mi"]
    grad = np.zeros(N_PARAMS)
    for k in range(N_PARAMS):
        if delta[k] <= 0:
            continue
        ch = 1 if k in TRANSLATION_PARAMS else 0
        grad[k] = (vals[1 + 2 * k, ch] - vals[2 + 2 * k, ch]) / (2.0 * delta[k])
    return grad, vals[0].copy()


def seed_from_map(family, lo, hi, n, index) -> np.ndarray:
    """Hand-off from an exhaustive map to `register` (reading A22; "exhaustive search over all the parameters"
    as the robust start, then the multi-metric gradient of PAPER.md:199, 210): the nine parameters
    of the map node with linear index `index` (p0 fastest) on the grid (lo, hi, n) of `family`, identity in the
    other groups.  Node k of axis d is lo + k (hi - lo)/(n - 1) as everywhere.  Translation / Euler / scale
    nodes are copied; log-scale nodes become factors exp(p); a versor node becomes the Euler angles of its
    rotation matrix R = Rz Ry Rx: ay = -asin(R20), ax = atan2(R21, R22), az = atan2(R10, R00)."""
    n = [int(v) for v in n]
    k = (index % n[0], (index // n[0]) % n[1], index // (n[0] * n[1]))
    node = [float(lo[d]) if n[d] == 1 else float(lo[d]) + float(k[d]) * (float(hi[d]) - float(lo[d])) / float(n[d] - 1)
            for d in range(3)]
    p = np.array([0, 0, 0, 0, 0, 0, 1, 1, 1], dtype=np.float64)
    if family == _orc.FAMILY_TRANSLATION:
        p[0:3] = node
    elif family == _orc.FAMILY_ROTATION_EULER_DEG:
        p[3:6] = node
    elif family == _orc.FAMILY_SCALE:
        p[6:9] = node
    elif family == _orc.FAMILY_SCALE_LOG:
        p[6:9] = np.exp(np.asarray(node))
    elif family == _orc.FAMILY_ROTATION_VERSOR:
        R = _orc.family_matrix(family, node)[:, :3]
        p[4] = np.degrees(np.arcsin(min(1.0, max(-1.0, -R[2, 0]))))
        p[3] = np.degrees(np.arctan2(R[2, 1], R[2, 2]))
        p[5] = np.degrees(np.arctan2(R[1, 0], R[0, 0]))
    else:
        raise ValueError("unknown family %r" % (family,))
    return p


GROUPS = ((0, 1, 2), (3, 4, 5), (6, 7, 8))      # translation [mm], rotation [deg], scale [factor]


def register(fixed, fixed_spacing, moving, moving_spacing, nbins, ranges, p0, delta, step0, step_min, max_iter, q,
             interp=_orc.INTERP_TRILINEAR, form=_orc.TSALLIS_ADDITIVE):
    """The loop of the paper's Fig. 1 (Transform -> Metric -> Optimizer) driven by the
    multi-metric gradient of section 4.  The paper names "gradient descent" and the multi-metric strategy
    but prints no step rule; the rule taken (A20) is regular-step gradient ASCENT (+MI is
    maximised, reading A2) applied to each parameter group with its own step length:

        g = multimetric_gradient(p)                      (Tsallis for translations, Shannon otherwise)
        for each group G with step L_G >= step_min[G]:
            d = g_G / |g_G|                              (skipped when |g_G| == 0)
            if d . d_prev_G < 0:  L_G = L_G / 2          (the direction turned back: halve the step)
            if L_G >= step_min[G]:  p_G = p_G + L_G * d
        stop when no group moved, or after max_iter iterations.

    Returns dict(p (9,), iterations, trace (iterations + 1, 9) of the visited p, steps (3,) final step lengths,
    values (2,) = (Shannon, Tsallis) at the last gradient evaluation)."""
    p = np.asarray(p0, dtype=np.float64).reshape(N_PARAMS).copy()
    delta = np.asarray(delta, dtype=np.float64).reshape(N_PARAMS)
    L = np.asarray(step0, dtype=np.float64).reshape(3).copy()
    Lmin = np.asarray(step_min, dtype=np.float64).reshape(3)
    prev = [None, None, None]
    trace = [p.copy()]
    vals = np.zeros(2)
    it = 0
    while it < int(max_iter):
        g, vals = multimetric_gradient(fixed, fixed_spacing, moving, moving_spacing, nbins, ranges, p, delta, q,
                                       interp=interp, form=form)
        moved = False
        for gi, idx in enumerate(GROUPS):
            if not (L[gi] >= Lmin[gi] and L[gi] > 0):
                continue
            gg = g[list(idx)]
            norm = float(np.sqrt(gg[0] * gg[0] + gg[1] * gg[1] + gg[2] * gg[2]))
            if norm == 0.0:
                continue
            d = gg / norm
            if prev[gi] is not None and (d[0] * prev[gi][0] + d[1] * prev[gi][1] + d[2] * prev[gi][2]) < 0.0:
                L[gi] = L[gi] / 2.0
            prev[gi] = d
            if L[gi] >= Lmin[gi]:
                p[list(idx)] = p[list(idx)] + L[gi] * d
                moved = True
        it += 1
        trace.append(p.copy())
        if not moved:
            break
    return {"p": p, "iterations": it, "trace": np.stack(trace), "steps": L, "values": vals}
