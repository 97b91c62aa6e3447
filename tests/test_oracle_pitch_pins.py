"""Pins of the oracle's PITCHED camera basis (contract C2: f = (cp ck, cp sk, sp), r = (sk, -ck, 0),
u = (-sp ck, -sp sk, cp); reading U6: pitch positive = nose up).

Every expectation here is elementary geometry written in fp64 from the ANGLES (never from the oracle's
own f / r / u), involves primitives under pitch != 0, and does not go through the fp64 shadow renderer —
which shares the C2 convention, so a mistake common to both renderers (a flipped sign on u's horizontal
part, a dropped cos p on f) would otherwise pass every test.  CPU only.
"""
import math

import numpy as np
import pytest

import gp_scenes as gs
import oracle
from conftest import ego_at_origin, make_prim, make_sphere, stack

SKY, GROUND, VEH, LIGHT = 0, 1, 3, gs.CLASS_LIGHT
PITCHES = [-30.0, -5.0, 5.0, 30.0, 85.0]
YAWS = [0.0, 37.0, -120.0]


def basis(yaw_deg, pitch_deg):
    """Right-handed camera frame from the two angles, fp64: f forward (nose up for p > 0), r to the camera's
    right, u = r x f up.  Built by rotating the level frame about the right axis, not from the contract."""
    y, p = math.radians(yaw_deg), math.radians(pitch_deg)
    f0 = np.array([math.cos(y), math.sin(y), 0.0])
    r = np.array([math.sin(y), -math.cos(y), 0.0])
    z = np.array([0.0, 0.0, 1.0])
    f = math.cos(p) * f0 + math.sin(p) * z          # level forward tipped towards +z
    u = np.cross(r, f)
    assert abs(f @ r) < 1e-15 and abs(np.linalg.norm(u) - 1) < 1e-15 and u[2] >= 0
    return f, r, u


def pitch_cs(pitch_deg):
    p = math.radians(pitch_deg)
    return np.float32(math.cos(p)), np.float32(math.sin(p))


def grid(H, W, th=1.0):
    s = ((np.arange(W) + 0.5) * 2.0 / W - 1.0) * th
    v = (1.0 - (np.arange(H) + 0.5) * 2.0 / H) * th * H / W
    return np.meshgrid(s, v)          # S[i, j], V[i, j]


def high_camera(**kw):
    # camera 100 m up with a 40 m far plane: the ground's planar depth is 100 / -(sp + v cp) >= 50 m for every
    # pitch and row used here (|sp + v cp| <= sqrt(2)), so it is never drawn
    return oracle.make_params(cam_height=CAM_H, t_max=40.0, **kw)


CAM_H = 100.0
O = np.array([0.0, 0.0, CAM_H])       # camera origin of ego_at_origin() under high_camera()


# ------------------------------------------------------------ (a) a target on the optical axis
@pytest.mark.parametrize("pitch", PITCHES)
@pytest.mark.parametrize("yaw", YAWS)
def test_sphere_on_the_pitched_axis_is_at_the_image_centre(yaw, pitch):
    # centre c = o + D f: the silhouette is the disc (s^2 + v^2)(D^2 - rho^2) <= rho^2 about the image centre
    # and the central ray meets the sphere at planar depth D - rho (|f| = 1).
    D, rho, H, W = 12.0, 1.0, 65, 65
    f, _, _ = basis(yaw, pitch)
    c = O + D * f
    y = math.radians(yaw)
    world = stack(ego_at_origin(math.cos(y), math.sin(y)), make_sphere(*c, rho, inst=5))
    cp, sp = pitch_cs(pitch)
    out = oracle.render_view(world, 0, H, W, high_camera(), cp=cp, sp=sp)
    S, V = grid(H, W)
    q = (S * S + V * V) * (D * D - rho * rho)
    inside, outside = q <= rho * rho * (1 - 2e-3), q >= rho * rho * (1 + 2e-3)
    hit = out["cls"] == LIGHT
    assert inside.sum() >= 5 and hit[inside].all() and not hit[outside].any()
    assert (out["cls"][~hit] == SKY).all()
    assert abs(out["depth"][H // 2, W // 2] - (D - rho)) <= 1e-5 * (D - rho)
    assert (out["depth"][hit] >= (D - rho) * (1 - 1e-5)).all()
    assert (out["depth"][hit] <= (D - rho * rho / D) * (1 + 1e-5)).all()


# ------------------------------------------------------------ (b) targets displaced along u and r
@pytest.mark.parametrize("pitch", PITCHES)
@pytest.mark.parametrize("yaw", YAWS)
@pytest.mark.parametrize("kind", ["sphere", "cube"])
def test_target_displaced_along_up_and_right_lands_on_its_row_and_column(yaw, pitch, kind):
    # A small target at o + D f + a u + b r projects to image coordinates (s, v) = (b / D, a / D): pixel
    # centroid row (1 - v / tv) H / 2 - 1/2 and column (s / th + 1) W / 2 - 1/2.  `a` fixes the sign and the
    # horizontal part of u (the row would move the wrong way / to the wrong depth otherwise), `b` the sign of r.
    D, H, W = 10.0, 129, 129
    f, r, u = basis(yaw, pitch)
    y = math.radians(yaw)
    ego = ego_at_origin(math.cos(y), math.sin(y))
    cp, sp = pitch_cs(pitch)
    for a, b in ((3.0, 0.0), (-2.0, 0.0), (0.0, 4.0), (0.0, -2.5), (2.5, -3.5)):
        c = O + D * f + a * u + b * r
        if kind == "sphere":
            tgt, cls, half = make_sphere(*c, 0.3, inst=7), LIGHT, 0.3
        else:       # a cube keeps its yaw-only orientation; its silhouette stays centred on its centre's projection
            tgt, cls, half = make_prim(*c, 0.25, 0.25, 0.25, math.cos(0.4), math.sin(0.4), cls=VEH, inst=7), VEH, 0.25
        out = oracle.render_view(stack(ego, tgt), 0, H, W, high_camera(), cp=cp, sp=sp)
        ii, jj = np.nonzero(out["cls"] == cls)
        assert len(ii) >= 9, (a, b, len(ii))
        row = (1.0 - a / D) * H / 2 - 0.5
        col = (b / D + 1.0) * W / 2 - 0.5
        assert abs(ii.mean() - row) < 0.75 and abs(jj.mean() - col) < 0.75, (a, b, ii.mean(), row, jj.mean(), col)
        # planar depth of the centre is D; the visible surface lies within the target's radius of it
        d = out["depth"][out["cls"] == cls]
        rad = half * (1.0 if kind == "sphere" else math.sqrt(3.0))
        assert (d > D - rad - 1e-3).all() and (d < D + rad).all()
        assert (out["inst"][out["cls"] == cls] == 7).all()


# ------------------------------------------------------------ (b') a wall square to the heading
@pytest.mark.parametrize("pitch", [-30.0, -5.0, 5.0, 30.0])
@pytest.mark.parametrize("yaw", YAWS)
def test_wall_ahead_depth_per_row_under_pitch(yaw, pitch):
    # A large box whose near face is the vertical plane X0 ahead of the camera along the (level) heading.  A ray
    # with image coordinates (s, v) advances cp - v sp along the heading per unit of planar depth (r has no
    # forward part), so every pixel on that face has depth X0 / (cp - v sp): constant along a row, and it is
    # on the face iff the hit height o.z + t (sp + v cp) lies in [z0, z1] and |t s| <= half width.
    X0, half_w, z0, z1, H, W = 15.0, 6.0, CAM_H - 6.0, CAM_H + 7.0, 48, 64
    y, p = math.radians(yaw), math.radians(pitch)
    ck, sk = math.cos(y), math.sin(y)
    cx, cy = (X0 + 1.0) * ck, (X0 + 1.0) * sk           # 2 m thick slab, centre 1 m behind the face
    wall = make_prim(cx, cy, 0.5 * (z0 + z1), 1.0, half_w, 0.5 * (z1 - z0), ck, sk, cls=VEH, inst=3)
    cp, sp = pitch_cs(pitch)
    out = oracle.render_view(stack(ego_at_origin(ck, sk), wall), 0, H, W, high_camera(), cp=cp, sp=sp)
    S, V = grid(H, W)
    adv = math.cos(p) - V * math.sin(p)
    t = X0 / adv
    z = CAM_H + t * (math.sin(p) + V * math.cos(p))
    m = 1e-3                                              # stay clear of the face's edges
    on = (adv > 0) & (t <= 40.0 - m) & (z >= z0 + m) & (z <= z1 - m) & (np.abs(t * S) <= half_w - m)
    off = (adv <= 0) | (t > 40.0 + m) | (z < z0 - m) | (z > z1 + m) | (np.abs(t * S) > half_w + m)
    # pixels that see the slab's top / bottom / side faces instead lie outside `on`; `off` only lists pixels whose
    # ray passes the face plane outside the face, which may still meet another face further on
    assert on.sum() > 200
    assert (out["cls"][on] == VEH).all()
    assert np.allclose(out["depth"][on], t[on], rtol=1e-5, atol=0)
    hit = out["cls"] == VEH
    assert (out["depth"][hit & off] > t[hit & off] * (1 + 1e-6)).all()    # anything seen there is behind the face plane
    # front face normal = -heading: n.L = -(0.48 ck + 0.36 sk)
    ndl = max(0.0, -(0.48 * ck + 0.36 * sk))
    s8 = min(256, int((0.25 + 0.75 * ndl) * 256.0 + 1e-9))
    exp = tuple((int(b) * s8) >> 8 for b in gs.DEFAULT_PALETTE[VEH])
    inner = on & (np.abs(t * S) <= half_w - 0.5)
    got = out["rgb"][:, inner]
    frac = np.mean([(got[ch] == exp[ch]).mean() for ch in range(3)])
    assert frac > 0.99                                     # s8 may sit on an integer boundary for one yaw: allow none in practice


# ------------------------------------------------------------ (c) pitching the camera = rotating the world
@pytest.mark.parametrize("pitch", PITCHES)
@pytest.mark.parametrize("yaw", [0.0, 37.0])
def test_pitched_view_equals_level_view_of_the_rotated_cluster(yaw, pitch):
    # Spheres stay spheres under a rotation.  Rotating the cluster about the camera's right axis through o by -p
    # (the rotation taking the pitched frame onto the level one) and looking at it with a level camera must give
    # the same image: same winners (except silhouette pixels, where fp32 rounding of the moved centres decides)
    # and the same depths to 1e-5.
    rng = np.random.default_rng(int(1000 + yaw * 10 + pitch))
    f, r, u = basis(yaw, pitch)
    f0, r0, u0 = basis(yaw, 0.0)
    R = np.outer(f0, f) + np.outer(r0, r) + np.outer(u0, u)       # maps f -> f0, r -> r0, u -> u0
    assert np.allclose(R @ R.T, np.eye(3), atol=1e-14) and np.linalg.det(R) > 0
    n = 24
    depth = rng.uniform(6.0, 30.0, n)
    a = rng.uniform(-0.8, 0.8, n) * depth
    b = rng.uniform(-0.8, 0.8, n) * depth
    rad = rng.uniform(0.3, 2.0, n)
    y = math.radians(yaw)
    ego = ego_at_origin(math.cos(y), math.sin(y))
    pit, lvl = [ego], [ego]
    for k in range(n):
        c = O + depth[k] * f + a[k] * u + b[k] * r
        c2 = O + R @ (c - O)
        pit.append(make_sphere(*c, rad[k], inst=k + 1))
        lvl.append(make_sphere(*c2, rad[k], inst=k + 1))
    H, W = 72, 96
    cp, sp = pitch_cs(pitch)
    A = oracle.render_view(stack(*pit), 0, H, W, high_camera(), cp=cp, sp=sp)
    B = oracle.render_view(stack(*lvl), 0, H, W, high_camera())
    assert (A["cls"] == LIGHT).sum() > 300
    robust = ((A["t2"].astype(np.float64) - A["depth"]) > 1e-3) & ((B["t2"].astype(np.float64) - B["depth"]) > 1e-3)
    differ = A["inst"] != B["inst"]
    assert differ.mean() < 0.01                      # silhouette pixels only
    # a silhouette pixel differs by one side seeing the sphere and the other its background
    same = ~differ
    hit = same & (A["cls"] == LIGHT)
    # fp32 centres are re-rounded after the rotation (|c| ~ 60 m -> ~4e-6 m), grazing rays amplify that
    graze = hit & robust
    assert np.allclose(A["depth"][graze], B["depth"][graze], rtol=2e-5, atol=2e-4)
    core = graze & (np.abs(A["depth"] - B["depth"]) <= 1e-5 * B["depth"])
    assert core.sum() >= 0.9 * graze.sum()


# ------------------------------------------------------------ pitch sign: nose up shows more sky
def test_positive_pitch_raises_the_horizon_row_by_tan_p():
    # level ground from a 1.6 m camera with no far plane: the horizon is the row where sp + v cp = 0, i.e.
    # v = -tan p: below the image centre for p > 0 (nose up: more sky), above it for p < 0.
    H = W = 64
    for pitch in (-20.0, -5.0, 5.0, 20.0):
        cp, sp = pitch_cs(pitch)
        out = oracle.render_view(stack(ego_at_origin()), 0, H, W, oracle.make_params(t_max=1e30), cp=cp, sp=sp)
        v = (1.0 - (np.arange(H) + 0.5) * 2.0 / H)
        exp_ground = v < -math.tan(math.radians(pitch))
        got_ground = out["cls"][:, 0] == GROUND
        clear = np.abs(v + math.tan(math.radians(pitch))) > 1e-4
        assert (got_ground == exp_ground)[clear].all()
        assert (out["cls"] == out["cls"][:, :1]).all()
