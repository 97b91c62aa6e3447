import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a B200 (run with -m gpu on the GPU box)")


import gp_scenes as gs  # noqa: E402


def pytest_sessionfinish(session, exitstatus):
    """-m gpu runs: the summed parity counts (pixels compared, excluded tie pixels, how many of those matched anyway,
    mismatches) go to gpurun_out/parity_report.json, from which profiles/r02_parity.md is written."""
    try:
        import json
        import parity_util
        if parity_util.REPORT:
            out = os.path.join(ROOT, "gpurun_out")
            os.makedirs(out, exist_ok=True)
            with open(os.path.join(out, "parity_report.json"), "w") as f:
                json.dump({"exitstatus": int(exitstatus), "report": parity_util.REPORT}, f, indent=1, sort_keys=True)
    except Exception:       # noqa: BLE001 - reporting must never fail a test run
        pass


def make_prim(cx, cy, cz, hx, hy, hz, cos_yaw=1.0, sin_yaw=0.0, cls=3, inst=0, shape=0):
    p = np.zeros((), dtype=gs.PRIM_DTYPE)
    p["cx"], p["cy"], p["cz"] = cx, cy, cz
    p["hx"], p["hy"], p["hz"] = hx, hy, hz
    p["cos_yaw"], p["sin_yaw"] = cos_yaw, sin_yaw
    p["cls"], p["inst"], p["shape"] = cls, inst, shape
    return p


def make_sphere(cx, cy, cz, r, cls=7, inst=0):
    return make_prim(cx, cy, cz, r, r, r, 1.0, 0.0, cls=cls, inst=inst, shape=gs.SHAPE_SPHERE)


def ego_at_origin(cos_yaw=1.0, sin_yaw=0.0, half_len=2.0):
    """Vehicle whose front-centre (the camera foot point) is exactly the world origin."""
    return make_prim(-half_len * cos_yaw, -half_len * sin_yaw, 0.75, half_len, 0.9, 0.75,
                     cos_yaw, sin_yaw, cls=3, inst=0)


def stack(*prims):
    out = np.zeros(len(prims), dtype=gs.PRIM_DTYPE)
    for i, p in enumerate(prims):
        out[i] = p
    return out


@pytest.fixture(scope="session")
def tiny_world():
    cfg = gs.config("tiny")
    a, q = gs.gen_world_prims(cfg)
    return cfg, np.concatenate([a, q], axis=1)
