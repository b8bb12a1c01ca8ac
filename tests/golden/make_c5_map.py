"""Writes tests/golden/c5_map_oracle.npy: the oracle's full C5 map (41^3 = 68 921 translations, Shannon MI,
trilinear, 256 bins) -- SURVEY.md 8(d) "--full runs all 68 921 for the argmax check"; north_star: "the map's
argmax identical" (the map of PAPER.md:57, 71; eq. 3).

Calls only `oracle/` (and the seeded input generator `paper_1909_10690_b200.phantoms`, which holds none of the
method's arithmetic).  About 1.45e12 evaluations: 30-60 minutes on 8-16 host cores, so the map is computed one p2
slab at a time and the slabs done so far are kept in <out>.partial.npz -- an interrupted run resumes.

    python tests/golden/make_c5_map.py [--out tests/golden/c5_map_oracle.npy]

The file holds float64 [n2][n1][n0] (p0 fastest), the layout of mi_map's channel 0.
tests/test_gpu_parity.py::test_c5_full_map_against_the_stored_oracle_map compares all 68 921 values and the arg max.
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "tests", "golden", "c5_map_oracle.npy"))
    ap.add_argument("--slabs", default=None, help="LO:HI -- only p2 slabs LO <= k2 < HI, highest first (to split the "
                                                  "work over two machines); the partial file is kept")
    ap.add_argument("--merge", action="append", default=[], help="another run's .partial.npz: its finished slabs are copied")
    args = ap.parse_args()
    import oracle as orc
    from paper_1909_10690_b200 import phantoms as ph

    cfg = ph.get_config("C5")
    n0, n1, n2 = (int(v) for v in cfg.n)
    part = args.out + ".partial.npz"
    out = np.full((n2, n1, n0), np.nan)
    if os.path.exists(part):
        out = np.load(part)["map"]
    for other in args.merge:
        o = np.load(other)["map"]
        fill = np.isnan(out).any(axis=(1, 2)) & ~np.isnan(o).any(axis=(1, 2))
        out[fill] = o[fill]
        print("merged %d slabs from %s" % (int(fill.sum()), other), flush=True)
    order = range(n2)
    if args.slabs:
        a, b = (int(v) for v in args.slabs.split(":"))
        order = range(min(b, n2) - 1, max(a, 0) - 1, -1)
    t0 = time.time()
    for k2 in order:
        if not np.isnan(out[k2]).any():
            continue
        m = orc.mi_map_range(cfg.fixed, cfg.fixed_spacing, cfg.moving, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                             cfg.family, cfg.lo, cfg.hi, cfg.n, (0, 0, k2), (n0, n1, k2 + 1), q=(),
                             interp=orc.INTERP_TRILINEAR)
        out[k2] = m[0, 0]
        np.savez(part + ".tmp.npz", map=out)
        os.replace(part + ".tmp.npz", part)
        print("slab %d/%d done, %.0f s" % (k2 + 1, n2, time.time() - t0), flush=True)
    if np.isnan(out).any():
        np.savez(part + ".tmp.npz", map=out)
        os.replace(part + ".tmp.npz", part)
        print("%d of %d slabs done; partial kept in %s" % (int((~np.isnan(out).any(axis=(1, 2))).sum()), n2, part))
        return
    np.save(args.out, out)
    if os.path.exists(part):
        os.remove(part)
    print("wrote %s: arg max %d, max %.12f" % (args.out, int(np.argmax(out)), float(out.max())))


if __name__ == "__main__":
    main()
