#!/usr/bin/env python
"""Writes scenegen/calibration.json: the scale multipliers that bring the synthetic C4 / C5 scenes to
the workload statistics BASELINE.json asks for:

  C4  "mean per-pixel depth complexity of about 60"  -> oracle's mean covering count per pixel
      (pairs with rho^2 <= c^2, counter `cover`) averaged over the 16 views = 60 +- 5
  C5  "tiles average about 300 splats"               -> oracle's E / tiles = 300 +- 15

Calls only oracle/ and scenegen/ (never the CUDA path).  Bisection on log(scale_mult); the measured
statistic is monotone in the multiplier.  Run:  python oracle/calibrate_scenes.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import scenegen  # noqa: E402
from scenegen import scenes  # noqa: E402

OUT = os.path.join(ROOT, "scenegen", "calibration.json")


def stat_c4(mult):
    sc = scenes.room_scene(4, 2_000_000, n_patches=400, patch_lo=0.2, patch_hi=1.0, scale_mult=mult,
                           patch_area_boost=4.0)
    cams = scenes._path_cameras(scenegen.SplitMix(1004), 16, 1200, 680, 600.0, circle=True)
    cfg = oracle.make_cfg()
    cover = [oracle.render(sc, oracle.make_cam(c), cfg)["counters"]["cover"] / (c.width * c.height) for c in cams]
    return float(np.mean(cover)), [round(float(x), 2) for x in cover]


def stat_c5(mult):
    sc = scenes.room_scene(5, 5_000_000, scale_mult=mult, active_frac=0.2)
    cam = scenes._room_camera(scenegen.SplitMix(1005), 640, 480, 525.0)
    cfg = oracle.make_cfg()
    b = oracle.binning(sc, oracle.make_cam(cam), cfg)
    return b["E"] / b["ranges"].shape[0], None


def bisect(stat, target, tol, lo=0.2, hi=1.0, iters=12):
    trace = []
    for _ in range(iters):
        mid = float(np.sqrt(lo * hi))
        v, detail = stat(mid)
        trace.append((mid, v))
        print(f"  scale_mult {mid:.5f} -> {v:.2f}", flush=True)
        if abs(v - target) <= tol:
            return mid, v, detail, trace
        if v > target:
            hi = mid
        else:
            lo = mid
    raise RuntimeError("calibration did not converge: %r" % trace)


def main():
    cal = {}
    print("C4: mean covering count per pixel -> 60 +- 2 (bar +- 5)")
    m, v, detail, _ = bisect(stat_c4, 60.0, 2.0)
    cal["C4"] = dict(scale_mult=round(m, 6), n_patches=400, patch_area_boost=4.0, mean_cover_per_pixel=round(v, 3),
                     cover_per_view=detail)
    print("C5: mean entries per tile -> 300 +- 5 (bar +- 15)")
    m, v, _, _ = bisect(stat_c5, 300.0, 5.0)
    cal["C5"] = dict(scale_mult=round(m, 6), mean_entries_per_tile=round(v, 3))
    cal["written_by"] = "oracle/calibrate_scenes.py"
    with open(OUT, "w") as fh:
        json.dump(cal, fh, indent=1)
        fh.write("\n")
    print("wrote", OUT)


if __name__ == "__main__":
    main()
