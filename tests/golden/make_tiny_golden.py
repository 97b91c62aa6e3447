"""Writes tests/golden/tiny_seed0.txt: digest of the Tiny workload (BASELINE.json configs[0]: seed 0,
1 world, 4 agents + 12 quads, 32x32, 90 deg, t_max 100) as rendered by the CPU ORACLE ONLY
(oracle/gp_oracle.c through oracle/__init__.py).  Nothing here touches the CUDA path.

The paper prints no pixel value for this path, so this is not a paper fixture: it is a
regression digest of the pinned oracle, regenerated only when a change to the oracle's arithmetic is
justified against DESIGN.md (the commit message must say so).

    python tests/golden/make_tiny_golden.py
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import gp_scenes as gs  # noqa: E402
import oracle  # noqa: E402


def digest_lines():
    cfg = gs.config("tiny")
    agents, quads = gs.gen_world_prims(cfg)
    prims = np.concatenate([agents, quads], axis=1)[0]
    par = oracle.make_params(cam_height=cfg.cam_height, t_max=cfg.t_max, fov_rad=float(np.float32(cfg.fov_rad)))
    lines = ["# view class_counts(sky,ground,marking,vehicle) depth_sum_f64 sha256(cls|inst|depth|rgb)"]
    for a in range(cfg.agents):
        r = oracle.render_view(prims, a, cfg.H, cfg.W, par)
        h = hashlib.sha256()
        for k in ("cls", "inst", "depth", "rgb"):
            h.update(np.ascontiguousarray(r[k]).tobytes())
        counts = np.bincount(r["cls"].ravel(), minlength=4)
        lines.append("%d %d,%d,%d,%d %.9f %s" % (a, *counts, float(r["depth"].astype(np.float64).sum()), h.hexdigest()))
    return lines


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_seed0.txt")
    with open(out, "w") as f:
        f.write("\n".join(digest_lines()) + "\n")
    print(open(out).read())
