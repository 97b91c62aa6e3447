"""Pins of the oracle's camera rig (contract C2: yaw offset + mount point; SURVEY.md §8(f) NEXT-2,
PAPER.md:317/:319/:434-435 "4 cameras (front, front-left, front-right, rear)").

None of these re-types the oracle's heading composition: each compares a rig camera with a plain
front camera (already pinned by CF1-CF6) of a differently posed ego whose camera coincides, with
closed-form depths, or with the fp64 shadow renderer.  CPU only.
"""
import math

import numpy as np
import pytest

import gp_scenes as gs
import oracle
from conftest import ego_at_origin, make_prim, stack

VEH = 3


def scene_around_origin(seed, n=10, extent=30.0):
    """A few boxes and quads around the origin (none closer than 3 m to it)."""
    rng = np.random.default_rng(seed)
    prims = []
    for i in range(n):
        while True:
            x, y = rng.uniform(-extent, extent, 2)
            if math.hypot(x, y) > 6.0:
                break
        psi = rng.uniform(-math.pi, math.pi)
        if i % 3 == 2:
            prims.append(make_prim(x, y, 0.01, rng.uniform(1.5, 8), 0.075, 0.0, math.cos(psi), math.sin(psi), cls=2, inst=10 + i))
        else:
            prims.append(make_prim(x, y, 0.75, rng.uniform(2, 2.5), rng.uniform(.9, 1.05), 0.75, math.cos(psi), math.sin(psi), inst=10 + i))
    return prims


EXACT_TURNS = {          # yaw offsets whose cos / sin are exact in fp32, and the equivalent ego heading
    "rear": ((-1.0, 0.0), (-1.0, 0.0)),
    "left90": ((0.0, 1.0), (0.0, 1.0)),
    "right90": ((0.0, -1.0), (0.0, -1.0)),
}


@pytest.mark.parametrize("name", sorted(EXACT_TURNS))
def test_rig_camera_equals_front_camera_of_a_turned_ego(name):
    # Ego heading +x with its front-centre at the origin.  A rig camera turned by 180 / +-90 degrees and
    # mounted at the front-centre sees exactly what the FRONT camera of an ego heading that way sees
    # when that ego's front-centre is also the origin (the ego box itself is never drawn).  All the
    # numbers involved are exact in fp32, so the images must agree bit for bit.
    (cd, sd), (ck2, sk2) = EXACT_TURNS[name]
    others = scene_around_origin(3)
    a = oracle.render_view(stack(ego_at_origin(1.0, 0.0), *others), 0, 40, 48, cam=(cd, sd, 1.0))
    b = oracle.render_view(stack(ego_at_origin(ck2, sk2), *others), 0, 40, 48)
    for k in ("cls", "inst", "depth", "rgb", "t2"):
        assert np.array_equal(a[k], b[k]), k
    assert (a["cls"] >= 2).sum() > 20            # the scene is actually visible


def test_rig_default_camera_is_the_front_camera():
    prims = stack(ego_at_origin(0.6, 0.8), *scene_around_origin(5))
    a = oracle.render_view(prims, 0, 33, 36, cp=math.cos(0.05), sp=math.sin(0.05))
    b = oracle.render_view(prims, 0, 33, 36, cp=math.cos(0.05), sp=math.sin(0.05), cam=(1.0, 0.0, 1.0))
    for k in ("cls", "inst", "depth", "rgb"):
        assert np.array_equal(a[k], b[k])


@pytest.mark.parametrize("mount,depth", [(1.0, 8.0), (0.0, 10.0), (-1.0, 12.0), (0.5, 9.0)])
def test_mount_point_shifts_the_camera_along_the_ego_axis(mount, depth):
    # Ego centred on the origin, half length 2; a box whose near face is the plane x = 10.  The camera
    # sits at x = 2 * mount, so the planar depth of the face is 10 - 2 * mount, exactly.
    ego = make_prim(0, 0, .75, 2, .9, .75, inst=0)
    box = make_prim(12, 0, .75, 2, .9, .75, inst=1)
    r = oracle.render_view(stack(ego, box), 0, 32, 32, cam=(1.0, 0.0, mount))
    hit = r["cls"] == VEH
    assert hit.any() and (r["depth"][hit] == np.float32(depth)).all()
    # lateral extent: |s| * depth <= 0.9
    s = ((np.arange(32) + 0.5) * 2 / 32 - 1.0)
    cols = np.nonzero(np.abs(s) * depth <= 0.9)[0]
    assert sorted(set(np.nonzero(hit)[1].tolist())) == cols.tolist()


@pytest.mark.parametrize("deg", [60.0, -60.0, 35.0, 123.0])
def test_box_straight_ahead_of_a_turned_camera(deg):
    # A box 4 x 1.8 x 1.5 m facing the turned camera squarely, its near face 10 m along the camera's
    # axis: the face pixels are rows 16-18 x columns 15-16 at planar depth 10 (CF1 through the rig).
    d = math.radians(deg)
    ux, uy = math.cos(d), math.sin(d)
    box = make_prim(12 * ux, 12 * uy, .75, 2, .9, .75, ux, uy, inst=1)
    r = oracle.render_view(stack(ego_at_origin(), box), 0, 32, 32, cam=(ux, uy, 1.0))
    hit = np.zeros((32, 32), bool)
    hit[16:19, 15:17] = True
    assert ((r["cls"] == VEH) == hit).all()
    assert np.allclose(r["depth"][hit], 10.0, rtol=2e-6)


def test_left_is_positive_yaw_offset():
    # A box 10 m ahead and 10 m to the LEFT (+y) of the camera is on the optical axis of a camera turned
    # +45 degrees, and outside the 90-degree view of one turned -45 degrees.
    c = math.sqrt(0.5)
    box = make_prim(10, 10, .75, 1, 1, .75, c, c, inst=1)
    left = oracle.render_view(stack(ego_at_origin(), box), 0, 32, 32, cam=(c, c, 1.0))
    right = oracle.render_view(stack(ego_at_origin(), box), 0, 32, 32, cam=(c, -c, 1.0))
    cols = np.nonzero((left["cls"] == VEH).any(axis=0))[0]
    assert cols.min() >= 13 and cols.max() <= 18 and 15 in cols and 16 in cols
    assert not (right["cls"] == VEH).any()


@pytest.mark.parametrize("seed", range(4))
def test_rig_fp32_contract_vs_fp64_face_enumeration(seed):
    # random rigs (yaw offset, mount), pitched, odd sizes: the fp32 slab renderer and the fp64 face
    # enumeration pick the same winner except on fp-sensitive pixels; depth within 1e-5.
    rng = np.random.default_rng(100 + seed)
    psi = rng.uniform(-math.pi, math.pi)
    ego = make_prim(rng.uniform(-3, 3), rng.uniform(-3, 3), .75, 2.3, 1.0, .75, math.cos(psi), math.sin(psi), inst=0)
    prims = stack(ego, *scene_around_origin(200 + seed, n=14, extent=25.0))
    par = oracle.make_params(fov_rad=np.float32(math.radians(rng.uniform(70, 110))))
    bad = tot = 0
    for _ in range(3):
        d = rng.uniform(-math.pi, math.pi)
        cam = (np.float32(math.cos(d)), np.float32(math.sin(d)), np.float32(rng.uniform(-1, 1)))
        p = math.radians(rng.uniform(-6, 6))
        H, W = 45, 52
        a = oracle.render_view(prims, 0, H, W, par, cp=np.float32(math.cos(p)), sp=np.float32(math.sin(p)), cam=cam)
        b = oracle.shadow_view(prims, 0, H, W, par, cp=np.float32(math.cos(p)), sp=np.float32(math.sin(p)), cam=cam)
        same = a["win"] == b["win"]
        tie = (b["t2"] - b["depth"]) <= 1e-5
        bad += int((~same & ~tie).sum()); tot += same.size
        ok = same & (a["win"] != -2)
        assert np.allclose(a["depth"][ok], b["depth"][ok], rtol=1e-5, atol=1e-5)
        assert (a["win"] >= 0).sum() > 10
    assert bad <= 2, (bad, tot)
