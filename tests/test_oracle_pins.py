"""Pins of the CPU oracle against what the mathematics fixes.

The paper prints no value for this path, so every expectation here is a
closed form, an invariant, a special case that reduces to a textbook routine, or a brute
force in a different formulation — none of them re-types the oracle's slab arithmetic.
CPU only.
"""
import math

import numpy as np
import pytest

import gp_scenes as gs
import oracle
from conftest import ego_at_origin, make_prim, stack

SKY, GROUND, MARK, VEH = 0, 1, 2, 3
PAL = gs.DEFAULT_PALETTE


def rows_v(H, W, th=1.0):
    i = np.arange(H, dtype=np.float64)
    return (1.0 - (i + 0.5) * 2.0 / H) * th * H / W


def cols_s(W, th=1.0):
    j = np.arange(W, dtype=np.float64)
    return ((j + 0.5) * 2.0 / W - 1.0) * th


def shade(base, ndl, ambient=0.25):
    s8 = min(256, int(math.floor((ambient + (1.0 - ambient) * ndl) * 256.0)))
    return tuple((int(b) * s8) >> 8 for b in base)


# ---------------------------------------------------------------- CF1: box straight ahead
@pytest.mark.parametrize("variant", ["yaw0", "yaw90", "heading_-x", "heading_+y"])
def test_cf1_axis_aligned_box_straight_ahead(variant):
    # Camera at (0,0,1.6); a 4 x 1.8 x 1.5 m box whose near face is the plane 10 m ahead.
    # Planar depth of every pixel on that face is exactly 10 (reading U1); the face spans
    # lateral [-0.9, 0.9] and heights [0, 1.5]: |s_j|*10 <= 0.9 -> columns 15,16;
    # 1.6 + 10 v_i in [0,1.5] -> rows 16,17,18 (32x32, 90 deg).
    if variant == "yaw0":
        ego, box, ndl = ego_at_origin(), make_prim(12, 0, .75, 2, .9, .75, 1, 0, inst=1), 0.0
    elif variant == "yaw90":       # local x along world y: swap half extents
        ego, box, ndl = ego_at_origin(), make_prim(12, 0, .75, .9, 2, .75, 0, 1, inst=1), 0.0
    elif variant == "heading_-x":  # face normal +x, light (0.48,0.36,0.8) -> n.L = 0.48
        ego, box, ndl = ego_at_origin(-1, 0), make_prim(-12, 0, .75, 2, .9, .75, 1, 0, inst=1), 0.48
    else:                          # heading +y, face normal -y -> n.L = -0.36 -> 0
        ego, box, ndl = ego_at_origin(0, 1), make_prim(0, 12, .75, .9, 2, .75, 1, 0, inst=1), 0.0
    r = oracle.render_view(stack(ego, box), 0, 32, 32)
    hit = np.zeros((32, 32), bool)
    hit[16:19, 15:17] = True
    assert ((r["cls"] == VEH) == hit).all()
    assert (r["depth"][hit] == np.float32(10.0)).all()
    assert (r["inst"][hit] == 1).all() and (r["inst"][~hit] == -1).all()
    exp = shade(PAL[VEH], ndl)
    if variant in ("yaw0", "yaw90"):
        assert exp == (10, 20, 55)
    for ch in range(3):
        assert (r["rgb"][ch][hit] == exp[ch]).all()
    # everything else: sky above the horizon, ground below
    assert (r["cls"][:16] == SKY).all()
    assert (r["cls"][16:][~hit[16:]] == GROUND).all()


def test_cf1_box_left_and_right_columns():
    # Box centre 3 m to the LEFT (+y), near face x = 10, y in [2.1, 3.9]: the near face covers
    # s = -y/10 in [-0.39,-0.21] -> columns 10,11,12 at planar depth exactly 10.  Its inner side
    # face (plane y = 2.1, x in [10,14]) is also visible: s = -2.1/x in [-0.21,-0.15] -> column 13
    # (s = -0.15625) at depth 2.1/0.15625 = 13.44.  Mirrored to the right: 19,20,21 and 18.
    for y, front, side in ((3.0, (10, 11, 12), 13), (-3.0, (19, 20, 21), 18)):
        r = oracle.render_view(stack(ego_at_origin(), make_prim(12, y, .75, 2, .9, .75, inst=1)), 0, 32, 32)
        got = sorted(set(np.nonzero(r["cls"] == VEH)[1].tolist()))
        assert tuple(got) == tuple(sorted(front + (side,)))
        for j in front:
            assert (r["depth"][16:19, j] == np.float32(10.0)).all()
        hit = r["cls"][:, side] == VEH
        assert hit.any() and np.allclose(r["depth"][hit, side], 13.44, rtol=1e-6)
        # side face normal is -y (left box) / +y (right box): n.L = -/+0.36
        exp = shade(PAL[VEH], 0.36 if y < 0 else 0.0)
        assert tuple(r["rgb"][:, 17, side]) == exp


# ---------------------------------------------------------------- CF2: ground depth per row
@pytest.mark.parametrize("H,W", [(32, 32), (64, 64), (126, 210)])
def test_cf2_ground_depth_per_row(H, W):
    r = oracle.render_view(stack(ego_at_origin()), 0, H, W)
    v = rows_v(H, W)
    for i in range(H):
        if v[i] < 0 and 1.6 / -v[i] <= 100.0 * (1 - 1e-6):
            exp = float(np.float32(1.6)) / -v[i]
            assert (r["cls"][i] == GROUND).all()
            # v_i is formed in fp32 as 1 - (i+0.5)(2/H): absolute error ~1e-7, so rows near the
            # horizon (small |v|) carry a relative depth error of ~1e-7/|v| (exact for H = 2^n)
            assert np.allclose(r["depth"][i], exp, rtol=1e-6 + 2e-7 / -v[i], atol=0)
            assert (r["depth"][i] == r["depth"][i, 0]).all()          # constant along the row
    if (H, W) == (32, 32):
        for i, d in ((16, 51.2), (17, 17.066667), (20, 5.688889), (31, 1.651613)):
            assert abs(r["depth"][i, 0] - d) < 1e-5 * d


@pytest.mark.parametrize("pitch_deg", [-5.0, -2.0, 3.0])
def test_cf2_ground_depth_with_pitch(pitch_deg):
    # depth(i) = h / -(sin p + v_i cos p) wherever that is positive.  For odd H the centre row
    # has v = 0: depth = h / sin|p| and the hit lies h / tan|p| ahead on the ground
    # (BASELINE.json north_star: "ground-plane hit distance h/tan(pitch) per pixel row").
    H = W = 33
    p = math.radians(pitch_deg)
    cp, sp = np.float32(math.cos(p)), np.float32(math.sin(p))
    par = oracle.make_params(t_max=1e9)
    r = oracle.render_view(stack(ego_at_origin()), 0, H, W, par, cp=cp, sp=sp)
    v = rows_v(H, W)
    dz = float(sp) + v * float(cp)
    for i in range(H):
        if dz[i] < -1e-9:
            assert np.allclose(r["depth"][i], float(np.float32(1.6)) / -dz[i], rtol=2e-6 + 3e-7 / -dz[i])
        elif dz[i] > 1e-9:
            assert (r["cls"][i] == SKY).all() and (r["depth"][i] == 0).all()
    if pitch_deg < 0:
        centre = r["depth"][16, 0]
        assert abs(centre * float(cp) - 1.6 / math.tan(-p)) < 1e-5 * centre


# ---------------------------------------------------------------- CF3 / CF4: horizon, empty world
@pytest.mark.parametrize("H,first", [(32, 16), (64, 33), (128, 65), (192, 98), (256, 130)])
def test_cf3_cf4_horizon_row_and_empty_world(H, first):
    # t_max = 100: ground row i visible iff 1.6/|v_i| <= 100 -> i >= H/2 + 0.008 H - 0.5 (reading U2).
    r = oracle.render_view(stack(ego_at_origin()), 0, H, H)
    assert (r["cls"][:first] == SKY).all() and (r["cls"][first:] == GROUND).all()
    assert (r["inst"] == -1).all()
    assert (r["depth"][:first] == 0).all() and (r["depth"][first:] > 0).all()
    assert (np.diff(r["depth"][first:, 0]) < 0).all()                       # I7
    for ch in range(3):
        assert (r["rgb"][ch][:first] == PAL[SKY][ch]).all()
        assert (r["rgb"][ch][first:] == 76).all()                           # 90 * 217 >> 8
    assert shade(PAL[GROUND], 0.8) == (76, 76, 76)
    # without the far plane the horizon is exactly H/2
    r = oracle.render_view(stack(ego_at_origin()), 0, H, H, oracle.make_params(t_max=float("inf")))
    assert (r["cls"][:H // 2] == SKY).all() and (r["cls"][H // 2:] == GROUND).all()


# ---------------------------------------------------------------- CF5: marking on the axis
@pytest.mark.parametrize("H,half_w", [(32, 1.0), (128, 1.0), (256, 0.075)])
def test_cf5_marking_under_camera_axis(H, half_w):
    quad = make_prim(20, 0, 0.01, 5.0, half_w, 0.0, 1, 0, cls=MARK, inst=7)
    r = oracle.render_view(stack(ego_at_origin(), quad), 0, H, H)
    v, s = rows_v(H, H), cols_s(H)
    n_cov = 0
    for i in range(H):
        if v[i] >= 0:
            continue
        t = 1.59 / -v[i]                     # plane z = 0.01 seen from 1.6
        for j in range(H):
            lat = abs(s[j]) * t
            margin = min(abs(t - 15), abs(t - 25), abs(lat - half_w))
            if margin < 1e-4:
                continue                     # on the analytic boundary: either answer is fine
            covered = 15 < t < 25 and lat < half_w
            assert (r["cls"][i, j] == MARK) == covered, (i, j)
            if covered:
                n_cov += 1
                assert abs(r["depth"][i, j] - t) < 2e-6 * t
                assert r["inst"][i, j] == 7
                g = 1.6 / -v[i]
                assert g - r["depth"][i, j] >= 0.01 - 1e-5      # nearer than the ground under it
                assert tuple(r["rgb"][:, i, j]) == shade(PAL[MARK], 0.8) == (203, 203, 203)
    assert n_cov > 0


# ---------------------------------------------------------------- CF6: top face
def test_cf6_top_face_from_raised_camera():
    par = oracle.make_params(cam_height=3.0)
    box = make_prim(12, 0, .75, 2, .9, .75, inst=1)
    r = oracle.render_view(stack(ego_at_origin(), box), 0, 64, 64, par)
    v, s = rows_v(64, 64), cols_s(64)
    n_top = 0
    for i in range(64):
        for j in range(64):
            if v[i] >= 0:
                continue
            t = 1.5 / -v[i]                                  # plane z = 1.5 seen from 3.0
            on_top = 10 + 1e-4 < t < 14 - 1e-4 and abs(s[j]) * t < 0.9 - 1e-4
            if on_top:
                n_top += 1
                assert r["cls"][i, j] == VEH
                assert abs(r["depth"][i, j] - t) < 2e-6 * t
                assert tuple(r["rgb"][:, i, j]) == shade(PAL[VEH], 0.8) == (33, 67, 186)
    assert n_top >= 4
    # pixels that enter through the front face (t == 10) are unlit: (10, 20, 55)
    front = (r["cls"] == VEH) & (r["depth"] == np.float32(10.0))
    assert front.any()
    assert (r["rgb"][2][front] == 55).all()


# ---------------------------------------------------------------- BF: fp32 slabs vs fp64 face enumeration
def _compare_with_shadow(prims, ego, H, W, par=None, cp=1.0, sp=0.0):
    par = par or oracle.make_params()
    r = oracle.render_view(prims, ego, H, W, par, cp, sp)
    sh = oracle.shadow_view(prims, ego, H, W, par, cp, sp)
    differ = r["win"] != sh["win"]
    # a pixel may legitimately differ only where two candidates are closer than fp32 can tell
    gap = np.minimum(sh["t2"] - sh["depth"], np.where(np.isfinite(r["t2"]), r["t2"].astype(np.float64) - r["depth"], np.inf))
    silhouette = differ & ~(gap <= 1e-4)
    same = ~differ
    hit = same & (sh["win"] > -2)
    tol = 1e-5 * sh["depth"][hit] + 1e-5      # fp32 rounding of ~100 m coordinates: ulp(64) = 7.6e-6 m
    assert (np.abs(r["depth"][hit] - sh["depth"][hit]) <= tol).all()
    assert (r["depth"][same & (sh["win"] == -2)] == 0).all()
    # shading, from the world-space normal (shadow) vs the local-frame light (contract C8)
    pal = np.array([[par.palette[c][ch] for ch in range(3)] for c in range(4)])
    cls = r["cls"].astype(int)
    I = par.ambient + (1.0 - par.ambient) * sh["ndl"]
    for ch in range(3):
        lo = (pal[cls, ch] * np.floor((I - 2e-6) * 256)).astype(int) >> 8
        hi = (pal[cls, ch] * np.floor((I + 2e-6) * 256)).astype(int) >> 8
        got = r["rgb"][ch].astype(int)
        ok = (got >= lo) & (got <= hi)
        assert ok[hit & (r["cls"] > 0)].all()
    return int(differ.sum()), int(silhouette.sum()), H * W


def test_bf_tiny_world_vs_face_enumeration(tiny_world):
    cfg, prims = tiny_world
    tot_diff = tot_sil = 0
    for ego in range(cfg.agents):
        d, s, _ = _compare_with_shadow(prims[0], ego, 32, 32)
        tot_diff += d; tot_sil += s
    assert tot_diff == 0 and tot_sil == 0


@pytest.mark.parametrize("seed", range(6))
def test_bf_random_scenes_vs_face_enumeration(seed):
    # dense little worlds with pitch, odd sizes and a near far-plane
    cfg = gs.SceneConfig("bf", 100 + seed, 2, 6, 20, 30.0, 40, 56, pitch_deg_max=8.0, t_max=40.0)
    a, q = gs.gen_world_prims(cfg)
    prims = np.concatenate([a, q], axis=1)
    pitch = gs.gen_pitch(cfg)
    par = oracle.make_params(t_max=cfg.t_max, fov_rad=np.float32(math.radians(70 + 10 * seed)))
    n_sil = n_px = 0
    for w in range(2):
        for ego in range(cfg.agents):
            d, s, n = _compare_with_shadow(prims[w], ego, cfg.H, cfg.W, par, pitch[w, ego, 0], pitch[w, ego, 1])
            n_sil += s; n_px += n
    # fp-sensitive silhouette pixels: expected <~ 1 per million
    assert n_sil <= 1, (n_sil, n_px)


# ---------------------------------------------------------------- I9: textbook AABB routine
def _aabb_hit(o, d, lo, hi):
    """Kay-Kajiya slab test in the world frame (Glassner [88])."""
    with np.errstate(divide="ignore", invalid="ignore"):
        t0 = (lo - o) / d
        t1 = (hi - o) / d
    tn = np.nanmax(np.minimum(t0, t1)); tf = np.nanmin(np.maximum(t0, t1))
    return tn if (tn <= tf and tn > 0) else None


def test_i9_axis_aligned_scene_matches_textbook_aabb():
    rng = np.random.default_rng(5)
    ego = ego_at_origin()
    boxes = []
    for k in range(12):
        boxes.append(make_prim(rng.uniform(4, 40), rng.uniform(-20, 20), 0.75, rng.uniform(1, 2.5),
                               rng.uniform(0.5, 1.2), 0.75, 1, 0, inst=k + 1))
    prims = stack(ego, *boxes)
    H = W = 48
    r = oracle.render_view(prims, 0, H, W)
    v, s = rows_v(H, W), cols_s(W)
    o = np.array([0.0, 0.0, float(np.float32(1.6))])
    bad = 0
    for i in range(H):
        for j in range(W):
            d = np.array([1.0, -s[j], v[i]])       # f=(1,0,0), r=(0,-1,0), u=(0,0,1)
            best, who = (o[2] / -d[2], -1) if d[2] < 0 and o[2] / -d[2] <= 100 else (np.inf, -2)
            second = np.inf
            for k in range(1, len(prims)):
                p = prims[k]
                c = np.array([p["cx"], p["cy"], p["cz"]], float); h = np.array([p["hx"], p["hy"], p["hz"]], float)
                t = _aabb_hit(o, d, c - h, c + h)
                if t is not None and t <= 100:
                    if t < best: second, best, who = best, t, k
                    elif t < second: second = t
            if second - best < 1e-4:
                continue
            bad += int(r["win"][i, j] != who)
            if who >= -1:
                assert abs(r["depth"][i, j] - best) <= 1e-5 * best
    assert bad == 0


# ---------------------------------------------------------------- invariants I1-I8
def _world(seed=7, n=8, q=16, extent=40.0):
    cfg = gs.SceneConfig("inv", seed, 1, n, q, extent, 48, 64)
    a, qd = gs.gen_world_prims(cfg)
    return cfg, np.concatenate([a, qd], axis=1)[0]


def test_i1_i2_class_instance_depth_consistency():
    cfg, prims = _world()
    for ego in range(cfg.agents):
        r = oracle.render_view(prims, ego, cfg.H, cfg.W)
        veh, mark = r["cls"] == VEH, r["cls"] == MARK
        assert ((r["inst"][veh] >= 0) & (r["inst"][veh] < cfg.agents) & (r["inst"][veh] != ego)).all()
        assert ((r["inst"][mark] >= cfg.agents) & (r["inst"][mark] < cfg.prims)).all()
        assert (r["inst"][~veh & ~mark] == -1).all()
        sky = r["cls"] == SKY
        assert (r["depth"][sky] == 0).all()
        assert ((r["depth"][~sky] > 0) & (r["depth"][~sky] <= 100)).all()
        assert (r["t2"] >= r["depth"])[~sky].all()


def test_i3_rigid_motion_invariance():
    cfg, prims = _world(seed=8)
    ang, tx, ty = 0.7312, 13.5, -4.25
    c, s = math.cos(ang), math.sin(ang)
    moved = prims.copy()
    x, y = prims["cx"].astype(float), prims["cy"].astype(float)
    ck, sk = prims["cos_yaw"].astype(float), prims["sin_yaw"].astype(float)
    moved["cx"] = c * x - s * y + tx; moved["cy"] = s * x + c * y + ty
    moved["cos_yaw"] = c * ck - s * sk; moved["sin_yaw"] = s * ck + c * sk
    for ego in range(3):
        a = oracle.shadow_view(prims, ego, cfg.H, cfg.W)
        b = oracle.shadow_view(moved, ego, cfg.H, cfg.W)
        ra = oracle.render_view(prims, ego, cfg.H, cfg.W)
        rb = oracle.render_view(moved, ego, cfg.H, cfg.W)
        # inputs are re-rounded to fp32 after the motion: only pixels on a silhouette may move
        robust = (a["t2"] - a["depth"] > 1e-3) & (b["t2"] - b["depth"] > 1e-3)
        changed = (a["win"] != b["win"])
        assert changed.mean() < 0.01
        same = ~changed
        assert np.allclose(a["depth"][same], b["depth"][same], rtol=1e-4, atol=1e-4)
        assert ((ra["win"] != rb["win"]) & same & robust).mean() < 0.002


def test_i4_mirror_symmetry():
    cfg, prims = _world(seed=9)
    ego_p = ego_at_origin()
    world = np.concatenate([stack(ego_p), prims[1:]])
    mirrored = world.copy()
    mirrored["cy"] = -world["cy"]; mirrored["sin_yaw"] = -world["sin_yaw"]   # reflect in the x-z plane
    a = oracle.render_view(world, 0, cfg.H, cfg.W)
    b = oracle.render_view(mirrored, 0, cfg.H, cfg.W)
    robust = ((a["t2"] - a["depth"]) > 1e-4) & ((b["t2"] - b["depth"]) > 1e-4)[:, ::-1]
    assert (a["cls"] == b["cls"][:, ::-1])[robust].all()
    assert (a["inst"] == b["inst"][:, ::-1])[robust].all()
    assert np.allclose(a["depth"][robust], b["depth"][:, ::-1][robust], rtol=1e-5)


def test_i5_permutation_of_primitive_order():
    cfg, prims = _world(seed=10)
    perm = np.concatenate([[0], np.random.default_rng(0).permutation(np.arange(1, len(prims)))])
    a = oracle.render_view(prims, 0, cfg.H, cfg.W)
    b = oracle.render_view(prims[perm], 0, cfg.H, cfg.W)
    untied = a["t2"] > a["depth"]
    assert (a["inst"] == b["inst"])[untied].all() and (a["cls"] == b["cls"])[untied].all()
    assert (a["depth"] == b["depth"]).all()
    assert (a["rgb"] == b["rgb"])[:, untied].all()


def test_i6_invisible_primitives_change_nothing():
    cfg, prims = _world(seed=11)
    world = np.concatenate([stack(ego_at_origin()), prims[1:]])
    extra = stack(make_prim(-30, 0, .75, 2, 1, .75, inst=90),            # behind the camera
                  make_prim(5, 40, .75, 2, 1, .75, .6, .8, inst=91),      # outside the 90 deg frustum
                  make_prim(150, 3, .75, 2, 1, .75, inst=92),             # beyond t_max
                  make_prim(-8, -3, 0.01, 4, .075, 0, .8, .6, cls=MARK, inst=93))
    a = oracle.render_view(world, 0, cfg.H, cfg.W)
    b = oracle.render_view(np.concatenate([world, extra]), 0, cfg.H, cfg.W)
    for k in ("cls", "inst", "depth", "rgb"):
        assert (a[k] == b[k]).all()


def test_i8_ego_is_excluded():
    cfg, prims = _world(seed=12)
    huge = prims.copy()
    huge["hx"][2] = 500.0; huge["hy"][2] = 500.0; huge["hz"][2] = 50.0
    # keep the camera where it was: o = c + hx * (cos, sin)
    huge["cx"][2] = prims["cx"][2] + (prims["hx"][2] - 500.0) * prims["cos_yaw"][2]
    huge["cy"][2] = prims["cy"][2] + (prims["hx"][2] - 500.0) * prims["sin_yaw"][2]
    a = oracle.render_view(prims, 2, cfg.H, cfg.W)
    b = oracle.render_view(huge, 2, cfg.H, cfg.W)
    assert (a["cls"] == b["cls"]).mean() > 0.999 and (a["inst"] == b["inst"]).mean() > 0.999
    assert (b["inst"] != 2).all()


def test_camera_inside_a_box_sees_through_it():
    # reading U3: a box the ray starts inside of is skipped (t_n <= 0)
    box = make_prim(0, 0, 1.0, 3, 3, 2.0, inst=5)
    a = oracle.render_view(stack(ego_at_origin(), box), 0, 16, 16)
    b = oracle.render_view(stack(ego_at_origin()), 0, 16, 16)
    assert (a["cls"] == b["cls"]).all() and (a["depth"] == b["depth"]).all()
    sh = oracle.shadow_view(stack(ego_at_origin(), box), 0, 16, 16)
    assert (sh["win"] < 0).all()


def test_ties_between_coplanar_quads_go_to_lower_index():
    q1 = make_prim(15, 0, 0.01, 6, 1.0, 0, 1, 0, cls=MARK, inst=11)
    q2 = make_prim(15, 0, 0.01, 1.0, 6, 0, 1, 0, cls=MARK, inst=22)
    r = oracle.render_view(stack(ego_at_origin(), q1, q2), 0, 64, 64)
    both = (r["t2"] == r["depth"]) & (r["cls"] == MARK)
    assert both.any() and (r["inst"][both] == 11).all()
    r2 = oracle.render_view(stack(ego_at_origin(), q2, q1), 0, 64, 64)
    assert (r2["inst"][both] == 22).all()


def test_primitive_beats_the_ground_at_equal_depth():
    # C6: the ground takes k = +inf.  A quad lying exactly in the plane z = 0 has bit-identical depth
    # (0 - o.z) * (1/d.z) to the ground on every pixel it covers, and must win there.
    quad = make_prim(12, 0, 0.0, 4.0, 1.5, 0.0, 1, 0, cls=MARK, inst=9)
    r = oracle.render_view(stack(ego_at_origin(), quad), 0, 64, 64)
    g = oracle.render_view(stack(ego_at_origin()), 0, 64, 64)
    covered = r["cls"] == MARK
    assert covered.sum() > 20
    assert (r["depth"][covered] == g["depth"][covered]).all()
    assert (r["t2"][covered] == r["depth"][covered]).all()          # the ground is the tied runner-up
    assert (r["inst"][covered] == 9).all()


def test_u10_ray_through_a_vertical_box_edge_takes_the_x_face():
    # Reading U10: on an exact edge (lo_x == lo_y == t_n) the entry face is x.  A 1 x 1 image has s = v = 0
    # exactly, so the single ray is the optical axis; a box with yaw 45 deg (cos == sin in fp32) and hx == hy
    # centred on the axis presents its vertical edge to it, and the two slab entries are the same fp32 number
    # by symmetry.  Camera heading -x: the two candidate faces are +x_local (n.L = (0.48 + 0.36) c) and
    # -y_local (n.L = (0.48 - 0.36) c), c = cos 45 deg — different shades, so the choice is visible.
    c = np.float32(math.sqrt(0.5))
    D, h = 20.0, 1.0
    box = make_prim(-D, 0.0, 1.6, h, h, 1.0, c, c, inst=4)
    r = oracle.render_view(stack(ego_at_origin(-1, 0), box), 0, 1, 1)
    assert r["cls"][0, 0] == VEH and r["inst"][0, 0] == 4
    assert abs(r["depth"][0, 0] - (D - h * math.sqrt(2.0))) < 1e-5 * D
    x_face = shade(PAL[VEH], (0.48 + 0.36) * float(c))
    y_face = shade(PAL[VEH], (0.48 - 0.36) * float(c))
    assert x_face != y_face
    assert tuple(int(v) for v in r["rgb"][:, 0, 0]) == x_face


# ---------------------------------------------------------------- far plane on primitive hits (reading U2)
def test_far_plane_on_a_box_is_inclusive_and_cuts_the_whole_face():
    # CF1's box: its near face is the plane 10 m ahead, so every pixel on it has planar depth exactly 10.0f.
    # t_max = 10 keeps the face (C5: hit iff t_n <= t_max, inclusive); t_max = 9.99 removes it, and since rows 16-18 meet
    # the ground at 51.2 / 17.07 / 10.24 m - all beyond either t_max - those six pixels are then sky, like the rest.
    world = stack(ego_at_origin(), make_prim(12, 0, .75, 2, .9, .75, 1, 0, inst=1))
    hit = np.zeros((32, 32), bool)
    hit[16:19, 15:17] = True
    on = oracle.render_view(world, 0, 32, 32, params=oracle.make_params(t_max=10.0))
    assert ((on["cls"] == VEH) == hit).all() and (on["depth"][hit] == np.float32(10.0)).all() and (on["inst"][hit] == 1).all()
    off = oracle.render_view(world, 0, 32, 32, params=oracle.make_params(t_max=9.99))
    assert (off["cls"][hit] == SKY).all() and (off["depth"][hit] == 0.0).all() and (off["inst"] == -1).all()
    assert not (off["cls"] == VEH).any()
    # a face partly beyond the far plane: the box of test_cf1_box_left_and_right_columns shows its near face (depth 10,
    # columns 10-12) and its inner side face (column 13, depth 13.44); t_max = 11 lies between them, so the near face stays
    # and column 13 falls back to ground (row 18 would meet it at 10.24 m) or sky
    left = stack(ego_at_origin(), make_prim(12, 3.0, .75, 2, .9, .75, inst=1))
    mid = oracle.render_view(left, 0, 32, 32, params=oracle.make_params(t_max=11.0))
    assert sorted(set(np.nonzero(mid["cls"] == VEH)[1].tolist())) == [10, 11, 12]
    assert (mid["depth"][mid["cls"] == VEH] == np.float32(10.0)).all()
    assert mid["cls"][16, 13] == SKY and mid["cls"][17, 13] == SKY and mid["cls"][18, 13] == GROUND


def test_i6_tall_box_beyond_the_far_plane_covers_pixel_centres_and_stays_invisible():
    # A 10 x 6 m wall whose near face is 118 m ahead spans heights 0..6 m: v = (z - 1.6) / 118 in [-0.0136, 0.0373] and
    # s in +-0.0424.  At 48 x 64 (tv = 0.75) row 23 has v = +0.015625 and columns 31, 32 have s = -+0.015625: two pixel
    # centres lie on the wall.  With t_max = 100 it is out of range: they are sky and nothing changes; with t_max = 120 they
    # are the wall at planar depth exactly 118.
    ego, wall = ego_at_origin(), make_prim(120, 0, 3.0, 2, 5, 3.0, inst=7)
    base = oracle.render_view(stack(ego), 0, 48, 64)
    far = oracle.render_view(stack(ego, wall), 0, 48, 64)
    for k in ("cls", "inst", "depth", "rgb"):
        assert (base[k] == far[k]).all()
    near = oracle.render_view(stack(ego, wall), 0, 48, 64, params=oracle.make_params(t_max=120.0))
    on = np.zeros((48, 64), bool)
    on[23, 31:33] = True
    assert ((near["inst"] == 7) == on).all()
    assert (near["depth"][on] == np.float32(118.0)).all() and (near["cls"][on] == VEH).all()


def test_flat_quad_seen_from_below_is_lit_as_from_above():
    # C8: a flat quad is shaded with its +z normal whichever side the ray comes from (sigma = +1 for h.z == 0).  A 6 x 6 m
    # marking 3 m above the ground, centred 8 m ahead of a camera at 1.6 m: rays with d.z > 0 meet it from below at
    # t = 1.4 / v.  n.L = 0.8 -> s8 = int((0.25 + 0.75 * 0.8) * 256) = 217 -> 240 * 217 >> 8 = 203 per channel.
    quad = make_prim(8, 0, 3.0, 3, 3, 0, cls=MARK, inst=5)
    r = oracle.render_view(stack(ego_at_origin(), quad), 0, 32, 32)
    got = r["inst"] == 5
    v = rows_v(32, 32)[:, None] * np.ones((1, 32))
    s = cols_s(32)[None, :] * np.ones((32, 1))
    with np.errstate(divide="ignore"):
        t = np.where(v > 0, 1.4 / np.where(v > 0, v, 1.0), np.inf)
    want = (t >= 5) & (t <= 11) & (np.abs(s * t) <= 3)
    assert want.sum() >= 20 and (got == want).all()
    assert np.allclose(r["depth"][got], t[got], rtol=1e-6)
    assert shade(PAL[MARK], 0.8) == (203, 203, 203)
    for ch in range(3):
        assert (r["rgb"][ch][got] == 203).all()
    assert (r["cls"][got] == MARK).all()
