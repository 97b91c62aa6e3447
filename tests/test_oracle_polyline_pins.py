"""Pins of the oracle's polyline -> strip expansion (contract C1p).  CPU only."""
import math

import numpy as np

import gp_scenes as gs
import oracle
from conftest import ego_at_origin, make_prim, stack


def quads_of(points, **kw):
    return oracle.polyline_quads(np.asarray(points, np.float32), dtype=gs.PRIM_DTYPE, **kw)


def test_axis_aligned_and_345_segments():
    q = quads_of([[[1, 2], [5, 2], [5, 10]], [[0, 0], [3, 4], [3, 4]]], half_width=0.1, z=0.02, cls=2, inst0=70)
    assert len(q) == 4
    # (1,2)->(5,2): centre (3,2), half length 2, heading +x, all exact
    assert (q[0]["cx"], q[0]["cy"], q[0]["hx"], q[0]["cos_yaw"], q[0]["sin_yaw"]) == (3.0, 2.0, 2.0, 1.0, 0.0)
    # (5,2)->(5,10): heading +y
    assert (q[1]["cx"], q[1]["cy"], q[1]["hx"], q[1]["cos_yaw"], q[1]["sin_yaw"]) == (5.0, 6.0, 4.0, 0.0, 1.0)
    # (0,0)->(3,4): the 3-4-5 triangle
    assert q[2]["hx"] == 2.5 and abs(q[2]["cos_yaw"] - 0.6) < 1e-7 and abs(q[2]["sin_yaw"] - 0.8) < 1e-7
    assert (q[2]["cx"], q[2]["cy"]) == (1.5, 2.0)
    # repeated vertex: zero-length quad with the default heading
    assert (q[3]["hx"], q[3]["cos_yaw"], q[3]["sin_yaw"]) == (0.0, 1.0, 0.0) and (q[3]["cx"], q[3]["cy"]) == (3.0, 4.0)
    assert (q["hy"] == np.float32(0.1)).all() and (q["hz"] == 0).all() and (q["cz"] == np.float32(0.02)).all()
    assert q["inst"].tolist() == [70, 71, 72, 73] and (q["cls"] == 2).all() and (q["shape"] == 0).all()


def test_strips_tile_the_polyline():
    cfg = gs.SceneConfig("lanes", 9, 2, 4, 0, 120.0, 32, 32)
    pts = gs.gen_lane_polylines(cfg, n_lines=6, pts_per_line=9)
    assert pts.shape == (2, 6, 9, 2)
    for w in range(2):
        q = quads_of(pts[w]).reshape(6, 8)
        p64 = pts[w].astype(np.float64)
        seg = np.hypot(*(p64[:, 1:] - p64[:, :-1]).transpose(2, 0, 1))          # library hypot, fp64
        assert np.allclose(2.0 * q["hx"], seg, rtol=1e-6)
        # each quad's two ends are the segment's vertices; unit heading
        for sign, vert in ((-1, p64[:, :-1]), (1, p64[:, 1:])):
            ex = q["cx"] + sign * q["hx"] * q["cos_yaw"]; ey = q["cy"] + sign * q["hx"] * q["sin_yaw"]
            assert np.allclose(ex, vert[..., 0], atol=2e-5) and np.allclose(ey, vert[..., 1], atol=2e-5)
        assert np.allclose(np.hypot(q["cos_yaw"], q["sin_yaw"]), 1.0, atol=3e-7)
        assert np.allclose(seg, 5.0, atol=1e-4)                                  # generator: 5 m steps


def test_polyline_strip_renders_like_the_equivalent_quad():
    # a straight lane marking along the optical axis built from 4 collinear 5 m segments renders exactly
    # like one 20 m quad (CF5) except for the instance ids
    line = [[[5, 0], [10, 0], [15, 0], [20, 0], [25, 0]]]
    strips = quads_of(line, half_width=1.0, inst0=10)
    one = make_prim(15, 0, 0.01, 10, 1.0, 0, cls=2, inst=10)
    a = oracle.render_view(stack(ego_at_origin(), *strips), 0, 64, 64)
    b = oracle.render_view(stack(ego_at_origin(), one), 0, 64, 64)
    assert np.array_equal(a["cls"], b["cls"]) and np.array_equal(a["depth"], b["depth"]) and np.array_equal(a["rgb"], b["rgb"])
    # every marking pixel carries the id of the segment its depth falls into (segment k spans x in [5+5k, 10+5k])
    m = a["cls"] == 2
    assert m.sum() > 50
    seg = np.floor((a["depth"][m].astype(np.float64) - 5.0) / 5.0).astype(int)
    assert (a["inst"][m] == 10 + seg).all()
    assert {10, 11, 13} <= set(np.unique(a["inst"][m]).tolist())
