"""Pins of the oracle's sphere primitive (contract C5s; "traffic lights use spheres").

Expectations come from elementary geometry (silhouette circle, nearest point, tangent depth), from
symmetry, and from the fp64 renderer, which intersects spheres by closest approach + half chord rather
than by the quadratic the fp32 contract uses.  CPU only.
"""
import math

import numpy as np
import pytest

import gp_scenes as gs
import oracle
from conftest import ego_at_origin, make_prim, make_sphere, stack

LIGHT = gs.CLASS_LIGHT


def grid(H, W, th=1.0):
    s = ((np.arange(W) + 0.5) * 2.0 / W - 1.0) * th
    v = (1.0 - (np.arange(H) + 0.5) * 2.0 / H) * th * H / W
    return np.meshgrid(s, v)          # S[i, j], V[i, j]


@pytest.mark.parametrize("D,r", [(10.0, 0.5), (6.0, 1.0), (40.0, 2.0)])
def test_sphere_on_the_optical_axis(D, r):
    # Sphere centred on the optical axis (camera height), D ahead.  A ray with image coordinates (s, v) has
    # direction (1, s, v); its distance from the centre is D sqrt(s^2+v^2) / sqrt(1+s^2+v^2), so the
    # silhouette is the disc (s^2 + v^2)(D^2 - r^2) <= r^2.  The central ray (odd image) hits at depth D - r;
    # every hit has planar depth in [D - r, D - r^2/D] (nearest point .. tangent circle).
    H = W = 65
    r_ = oracle.render_view(stack(ego_at_origin(), make_sphere(D, 0, 1.6, r, inst=9)), 0, H, W)
    S, V = grid(H, W)
    q = (S * S + V * V) * (D * D - r * r)
    inside, outside = q <= r * r * (1 - 1e-4), q >= r * r * (1 + 1e-4)
    hit = r_["cls"] == LIGHT
    assert hit[inside].all() and not hit[outside].any() and inside.sum() >= 5
    assert r_["depth"][H // 2, W // 2] == np.float32(D - r)
    assert (r_["depth"][hit] >= np.float32(D - r)).all()
    assert (r_["depth"][hit] <= (D - r * r / D) * (1 + 1e-5)).all()
    assert (r_["inst"][hit] == 9).all()
    # emissive: palette colour unshaded
    for ch in range(3):
        assert (r_["rgb"][ch][hit] == gs.DEFAULT_PALETTE[LIGHT][ch]).all()
    # depth grows with distance from the image centre (nearer point of the sphere faces the camera)
    row = r_["depth"][H // 2]
    cols = np.nonzero(hit[H // 2])[0]
    right = row[cols[cols >= W // 2]]
    assert (np.diff(right) >= 0).all()


def test_sphere_depth_matches_point_on_sphere():
    # every hit pixel's point o + t d lies on the sphere (|p - c| = r to fp32 accuracy) and is the near one
    c = np.array([14.0, 3.0, 4.0]); r = 1.5
    H, W = 60, 80
    out = oracle.render_view(stack(ego_at_origin(), make_sphere(*c, r, inst=1)), 0, H, W)
    S, V = grid(H, W)
    hit = out["cls"] == LIGHT
    assert hit.sum() > 30
    t = out["depth"].astype(np.float64)
    # camera at (0,0,1.6) heading +x: right = -y, up = +z
    P = np.stack([t, -S * t, 1.6 + V * t], axis=-1)
    dist = np.linalg.norm(P - c, axis=-1)
    assert np.allclose(dist[hit], r, atol=2e-4)
    d = np.stack([np.ones_like(S), -S, V], axis=-1)
    assert (((P - c) * d).sum(-1)[hit] <= 1e-4).all()        # front side: outward normal faces the camera


def test_sphere_occlusion_order_and_range():
    ego = ego_at_origin()
    box = make_prim(8, 0, 1.6, .5, 3, 3, inst=1)             # a wall 7.5 m ahead
    lamp_front = make_sphere(5, 0, 1.6, 0.5, inst=2)
    lamp_behind = make_sphere(12, 0, 1.6, 0.5, inst=3)
    far = make_sphere(150, 0, 1.6, 5.0, inst=4)              # beyond t_max = 100
    behind_cam = make_sphere(-5, 0, 1.6, 0.5, inst=5)
    inside = make_sphere(0.1, 0, 1.6, 1.0, inst=6)           # camera inside: skipped (U3)
    r = oracle.render_view(stack(ego, box, lamp_front, lamp_behind, far, behind_cam, inside), 0, 33, 33)
    ids = set(np.unique(r["inst"]).tolist())
    assert 2 in ids and 1 in ids and not ({3, 4, 5, 6} & ids)
    assert r["inst"][16, 16] == 2 and r["depth"][16, 16] == np.float32(4.5)


def test_sphere_ignores_yaw_and_half_extent_fields():
    a = make_sphere(9, 1, 2.0, 0.7, inst=1)
    b = a.copy(); b["cos_yaw"], b["sin_yaw"], b["hy"], b["hz"] = 0.6, 0.8, 5.0, 0.0
    ra = oracle.render_view(stack(ego_at_origin(), a), 0, 40, 40)
    rb = oracle.render_view(stack(ego_at_origin(), b), 0, 40, 40)
    for k in ("cls", "inst", "depth", "rgb"):
        assert np.array_equal(ra[k], rb[k])
    assert (ra["cls"] == LIGHT).sum() > 4


@pytest.mark.parametrize("seed", range(4))
def test_spheres_fp32_quadratic_vs_fp64_closest_approach(seed):
    rng = np.random.default_rng(900 + seed)
    psi = rng.uniform(-math.pi, math.pi)
    prims = [make_prim(0, 0, .75, 2.2, 1.0, .75, math.cos(psi), math.sin(psi), inst=0)]
    for i in range(10):
        ang, dist = rng.uniform(-math.pi, math.pi), rng.uniform(4, 40)
        prims.append(make_sphere(dist * math.cos(ang), dist * math.sin(ang), rng.uniform(0.5, 6), rng.uniform(0.15, 1.5), inst=20 + i))
    for i in range(6):
        ang, dist = rng.uniform(-math.pi, math.pi), rng.uniform(6, 40)
        y = rng.uniform(-math.pi, math.pi)
        prims.append(make_prim(dist * math.cos(ang), dist * math.sin(ang), .75, 2.2, 1.0, .75, math.cos(y), math.sin(y), inst=40 + i))
    prims = stack(*prims)
    bad = tot = 0
    for _ in range(4):
        d = rng.uniform(-math.pi, math.pi)
        cam = (math.cos(d), math.sin(d), rng.uniform(-1, 1))
        p = math.radians(rng.uniform(-8, 8))
        a = oracle.render_view(prims, 0, 50, 58, cp=np.float32(math.cos(p)), sp=np.float32(math.sin(p)), cam=cam)
        b = oracle.shadow_view(prims, 0, 50, 58, cp=np.float32(math.cos(p)), sp=np.float32(math.sin(p)), cam=cam)
        same = a["win"] == b["win"]
        tie = (b["t2"] - b["depth"]) <= 1e-5
        bad += int((~same & ~tie).sum()); tot += same.size
        ok = same & (a["win"] != -2)
        assert np.allclose(a["depth"][ok], b["depth"][ok], rtol=1e-5, atol=2e-5)
    sph = np.isin(a["inst"], np.arange(20, 30))
    assert bad <= 3, (bad, tot)


def test_far_plane_on_a_sphere_is_inclusive():
    # A sphere of radius 2 centred 12 m ahead at camera height: every surface point has x >= 10, and planar depth IS x, so
    # the one ray that enters at exactly 10.0 is the central one (33 x 33: pixel (16, 16) has s = v = 0; A = 1, B = -12,
    # t_ca = 12, half chord 2 -> t_n = 10 exactly in fp32).  t_max = 10 keeps that single pixel (C5s: t_n <= t_max,
    # inclusive), t_max = 9.99 removes the sphere altogether.  With t_max = 10.5 the drawn part is the cap x <= 10.5,
    # checked against the fp64 quadratic per pixel.
    world = stack(ego_at_origin(), make_sphere(12, 0, 1.6, 2.0, inst=4))
    on = oracle.render_view(world, 0, 33, 33, params=oracle.make_params(t_max=10.0))
    assert (on["inst"] == 4).sum() == 1 and on["inst"][16, 16] == 4 and on["depth"][16, 16] == np.float32(10.0)
    off = oracle.render_view(world, 0, 33, 33, params=oracle.make_params(t_max=9.99))
    assert not (off["inst"] == 4).any() and off["cls"][16, 16] == 0 and off["depth"][16, 16] == 0.0
    H = W = 65
    cap = oracle.render_view(world, 0, H, W, params=oracle.make_params(t_max=10.5))
    i, j = np.mgrid[0:H, 0:W].astype(np.float64)
    s = (j + 0.5) * 2.0 / W - 1.0
    v = 1.0 - (i + 0.5) * 2.0 / H
    d = np.stack([np.ones_like(s), -s, v], axis=-1)                    # camera at (0, 0, 1.6) heading +x: right = -y
    e = np.array([-12.0, 0.0, 0.0])
    A = (d * d).sum(-1); B = (d * e).sum(-1); C = 144.0 - 4.0
    disc = B * B - A * C
    with np.errstate(invalid="ignore"):
        t = np.where(disc >= 0, (-B - np.sqrt(np.where(disc >= 0, disc, 0.0))) / A, np.inf)
    sure_in = t <= 10.5 - 1e-4
    sure_out = t >= 10.5 + 1e-4
    got = cap["inst"] == 4
    assert sure_in.sum() > 20 and got[sure_in].all() and not got[sure_out].any()
    assert (cap["depth"][got] <= np.float32(10.5)).all()
    whole = oracle.render_view(world, 0, H, W)
    assert ((whole["inst"] == 4) & ~got).sum() > 20                     # the rim of the disc lies beyond 10.5 m: cut away
