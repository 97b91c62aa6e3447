"""Pins of the NEXT-4 oracle (oracle/gp_sim_oracle.c): jerk-actuated kinematic bicycle and the
vectorised observation O_vec.

The paper prints no value for either; every expectation is a closed form of the discrete recurrences, a saturation
value, a hand-placed configuration whose answer is elementary geometry, or an independent fp64 numpy computation
(argsort) on tie-free inputs.  CPU only.
"""
import math

import numpy as np
import pytest

import gp_scenes as gs
import oracle
from conftest import make_prim, make_sphere, stack

JLON = (-15.0, -4.0, 0.0, 4.0)
JLAT = (-4.0, 0.0, 4.0)


def act(lon, lat):
    return JLON.index(lon) * 3 + JLAT.index(lat)


def fresh(n=1, v=0.0, psi=0.0, x=0.0, y=0.0, a_lon=0.0, a_lat=0.0, steer=0.0):
    st = np.zeros((n, 8), np.float32)
    st[:, 0], st[:, 1], st[:, 2], st[:, 3], st[:, 4] = v, a_lon, a_lat, steer, psi
    ps = np.zeros((n, 4), np.float32)
    ps[:, 0], ps[:, 1], ps[:, 2], ps[:, 3] = x, y, np.cos(psi), np.sin(psi)
    return st, ps


def run(par, actions, half_len, st, ps):
    """actions: [steps][n]"""
    traj = [(st.copy(), ps.copy())]
    for a in actions:
        st, ps = oracle.dynamics_step(par, a, half_len, st, ps)
        traj.append((st.copy(), ps.copy()))
    return traj


# ------------------------------------------------------------------------------------------------ dynamics
def test_action_table_is_the_product_of_the_papers_jerk_sets():
    # twelve actions = {-15, -4, 0, 4} x {-4, 0, 4} m/s^3; one step from rest integrates the jerk once
    par = oracle.make_dyn_params(dt=0.1, a_lon_max=10.0, a_lat_max=10.0)
    seen = set()
    for a in range(12):
        st, ps = fresh()
        s1, _ = oracle.dynamics_step(par, [a], [2.0], st, ps)
        jl, jt = s1[0, 1] / 0.1, s1[0, 2] / 0.1
        assert abs(jl - JLON[a // 3]) < 1e-5 and abs(jt - JLAT[a % 3]) < 1e-5
        seen.add((round(float(jl)), round(float(jt))))
    assert seen == {(int(l), int(t)) for l in JLON for t in JLAT}
    with pytest.raises(ValueError):
        oracle.dynamics_step(par, [12], [2.0], *fresh())


@pytest.mark.parametrize("psi_deg", [0.0, 30.0, -135.0])
def test_straight_line_under_constant_jerk_closed_form(psi_deg):
    # zero lateral jerk, steer 0: a_n = n j dt, v_n = v0 + j dt^2 n(n+1)/2, s_n = n v0 dt + j dt^3 n(n+1)(n+2)/6
    # along the heading (position moves with the NEW speed: semi-implicit Euler, contract D5); heading never changes
    par = oracle.make_dyn_params(dt=0.1, a_lon_max=6.0, v_max=30.0)
    psi = math.radians(psi_deg)
    v0, j, n, dt = 3.0, 4.0, 12, 0.1
    st, ps = fresh(v=v0, psi=psi, x=1.5, y=-2.0)
    traj = run(par, [[act(j, 0.0)]] * n, [2.2], st, ps)
    for k, (s, p) in enumerate(traj):
        a_k = k * j * dt
        v_k = v0 + j * dt * dt * k * (k + 1) / 2
        d_k = k * v0 * dt + j * dt ** 3 * k * (k + 1) * (k + 2) / 6
        assert abs(s[0, 1] - a_k) < 1e-5 and abs(s[0, 0] - v_k) < 1e-5
        assert abs(p[0, 0] - (1.5 + d_k * math.cos(psi))) < 2e-5 and abs(p[0, 1] - (-2.0 + d_k * math.sin(psi))) < 2e-5
        assert s[0, 3] == 0.0 and abs(s[0, 4] - psi) < 1e-6
        assert abs(p[0, 2] - math.cos(psi)) < 1e-6 and abs(p[0, 3] - math.sin(psi)) < 1e-6


def test_constant_curvature_arc():
    # constant speed, steering angle d0 held (the lateral acceleration is the one that demands exactly d0): the heading
    # advances D = v tan(d0) / L dt per step and the vertices lie on a circle of radius v dt / (2 sin(D / 2)), which
    # tends to the bicycle's turning radius L / tan(d0)
    par = oracle.make_dyn_params(dt=0.1, a_lat_max=50.0, steer_max=0.7)
    hx, v, d0 = 2.5, 8.0, 0.2
    L = 0.6 * 2 * hx
    a_lat = v * v * math.tan(d0) / L
    st, ps = fresh(v=v, steer=d0, a_lat=a_lat, psi=0.3)
    traj = run(par, [[act(0.0, 0.0)]] * 60, [hx], st, ps)
    D = v * math.tan(d0) / L * 0.1
    pts = np.array([[p[0, 0], p[0, 1]] for _, p in traj], dtype=np.float64)
    for k, (s, p) in enumerate(traj):
        assert abs(s[0, 0] - v) < 1e-6 and abs(s[0, 3] - d0) < 1e-6
        want = (0.3 + k * D + math.pi) % (2 * math.pi) - math.pi
        assert abs(((s[0, 4] - want + math.pi) % (2 * math.pi)) - math.pi) < 2e-5
    # circumcentre from the first three vertices, then every vertex is at the same distance
    (x1, y1), (x2, y2), (x3, y3) = pts[0], pts[20], pts[40]
    d = 2 * (x1 * (y2 - y3) + x2 * (y3 - y1) + x3 * (y1 - y2))
    cx = ((x1**2 + y1**2) * (y2 - y3) + (x2**2 + y2**2) * (y3 - y1) + (x3**2 + y3**2) * (y1 - y2)) / d
    cy = ((x1**2 + y1**2) * (x3 - x2) + (x2**2 + y2**2) * (x1 - x3) + (x3**2 + y3**2) * (x2 - x1)) / d
    rad = np.hypot(pts[:, 0] - cx, pts[:, 1] - cy)
    rho = v * 0.1 / (2 * math.sin(D / 2))
    assert np.allclose(rad, rho, rtol=2e-5)
    assert abs(rho / (L / math.tan(d0)) - 1) < D * D / 20          # ~ 1 + D^2 / 24
    # left turn for a positive steering angle: the centre is to the LEFT of the initial heading
    left = np.array([-math.sin(0.3), math.cos(0.3)])
    assert (np.array([cx, cy]) - pts[0]) @ left > 0


def test_wheelbase_is_sixty_percent_of_the_vehicle_length():
    par = oracle.make_dyn_params(dt=0.1, a_lat_max=50.0)
    st, ps = fresh(n=2, v=5.0, steer=0.1)
    st[:, 2] = [25.0 * math.tan(0.1) / (0.6 * 4.0), 25.0 * math.tan(0.1) / (0.6 * 6.0)]    # hold the angle
    s1, _ = oracle.dynamics_step(par, [7, 7], [2.0, 3.0], st, ps)
    assert abs(s1[0, 4] - 5.0 * math.tan(0.1) / (0.6 * 4.0) * 0.1) < 1e-6
    assert abs(s1[1, 4] - 5.0 * math.tan(0.1) / (0.6 * 6.0) * 0.1) < 1e-6


def test_every_limit_saturates():
    par = oracle.make_dyn_params(dt=0.1, a_lon_max=3.0, a_lat_max=2.0, v_max=9.0, steer_max=0.35, steer_rate_max=0.5)
    # longitudinal acceleration and speed (upper limits), then braking to a standstill: no reversing
    traj = run(par, [[act(4.0, 0.0)]] * 60, [2.0], *fresh(v=1.0))
    assert traj[-1][0][0, 1] == np.float32(3.0) and traj[-1][0][0, 0] == np.float32(9.0)
    assert max(t[0][0, 1] for t in traj) == np.float32(3.0) and max(t[0][0, 0] for t in traj) == np.float32(9.0)
    traj = run(par, [[act(-15.0, 0.0)]] * 60, [2.0], *traj[-1])
    assert traj[-1][0][0, 1] == np.float32(-3.0) and traj[-1][0][0, 0] == 0.0
    assert min(t[0][0, 0] for t in traj) == 0.0
    x_stop = traj[-1][1][0, 0]
    traj = run(par, [[act(-15.0, 0.0)]] * 5, [2.0], *traj[-1])
    assert traj[-1][1][0, 0] == x_stop                                  # standing still
    # lateral acceleration, steering rate, steering angle
    traj = run(par, [[act(0.0, 4.0)]] * 40, [2.0], *fresh(v=2.0))
    assert traj[-1][0][0, 2] == np.float32(2.0)
    steer = np.array([t[0][0, 3] for t in traj], dtype=np.float64)
    assert (np.diff(steer) <= 0.5 * 0.1 + 1e-7).all() and np.diff(steer).max() > 0.5 * 0.1 - 1e-6     # rate-limited
    assert abs(steer[-1] - 0.35) < 1e-7 and steer.max() <= 0.35 + 1e-7
    traj = run(par, [[act(0.0, -4.0)]] * 60, [2.0], *traj[-1])
    assert abs(traj[-1][0][0, 3] + 0.35) < 1e-7 and traj[-1][0][0, 2] == np.float32(-2.0)


def test_low_speed_uses_v_eps_in_the_curvature_demand():
    par = oracle.make_dyn_params(dt=0.1, v_eps=0.5, steer_rate_max=100.0, steer_max=1.5)
    st, ps = fresh(v=0.0, a_lat=1.0)
    s1, _ = oracle.dynamics_step(par, [7], [2.0], st, ps)
    assert abs(s1[0, 3] - math.atan(0.6 * 4.0 * 1.0 / 0.25)) < 1e-6


def test_heading_and_position_wrap():
    par = oracle.make_dyn_params(dt=0.1, extent=40.0, a_lat_max=50.0)
    # heading just below pi, turning left: wraps to just above -pi; cos / sin stay continuous
    L = 0.6 * 4.0
    st, ps = fresh(v=10.0, steer=0.3, psi=math.pi - 0.01, a_lat=100.0 * math.tan(0.3) / L)
    s1, p1 = oracle.dynamics_step(par, [7], [2.0], st, ps)
    exp = math.pi - 0.01 + 10.0 * math.tan(0.3) / L * 0.1 - 2 * math.pi
    assert -math.pi <= s1[0, 4] < math.pi and abs(s1[0, 4] - exp) < 1e-6
    assert abs(p1[0, 2] - math.cos(exp)) < 1e-6 and abs(p1[0, 3] - math.sin(exp)) < 1e-6
    # position leaving the square [-20, 20) re-enters on the other side
    st, ps = fresh(v=10.0, x=19.5)
    _, p1 = oracle.dynamics_step(par, [7], [2.0], st, ps)
    assert abs(p1[0, 0] - (19.5 + 1.0 - 40.0)) < 1e-5
    st, ps = fresh(v=10.0, psi=-math.pi / 2, y=-19.8)
    _, p1 = oracle.dynamics_step(par, [7], [2.0], st, ps)
    assert abs(p1[0, 1] - (-19.8 - 1.0 + 40.0)) < 1e-5


# ------------------------------------------------------------------------------------------------ O_vec
def veh(x, y, yaw_deg=0.0, hx=2.0, hy=0.9, inst=0):
    a = math.radians(yaw_deg)
    return make_prim(x, y, 0.75, hx, hy, 0.75, np.float32(math.cos(a)), np.float32(math.sin(a)), cls=3, inst=inst)


def seg(x, y, yaw_deg=0.0, half_len=4.0, cls=2):
    a = math.radians(yaw_deg)
    return make_prim(x, y, 0.01, half_len, 0.075, 0.0, np.float32(math.cos(a)), np.float32(math.sin(a)), cls=cls)


@pytest.mark.parametrize("ego_yaw", [0.0, 90.0, 180.0])
def test_hand_placed_neighbours_in_the_ego_frame(ego_yaw):
    # ego at (3, -2); in ITS frame: neighbour A 10 m ahead, B 5 m to the left, C 7 m behind.  Placed in the world by
    # rotating with the ego's heading, so the expected ego-frame coordinates are the same for every heading.
    a = math.radians(ego_yaw)
    c, s = math.cos(a), math.sin(a)

    def world(fx, fy):
        return 3 + c * fx - s * fy, -2 + s * fx + c * fy
    prims = stack(veh(3, -2, ego_yaw), veh(*world(10, 0), ego_yaw + 90, hx=2.5, hy=1.0), veh(*world(0, 5), ego_yaw),
                  veh(*world(-7, 0), ego_yaw + 180, hx=1.0, hy=0.4), seg(*world(6, -3), ego_yaw + 90, cls=2),
                  seg(*world(2, 1), ego_yaw, half_len=7.5, cls=6), make_sphere(*world(1, 0), 4.0, 0.3),
                  make_prim(*world(1, 1), 0.5, 0.5, 0.5, 0.5, cls=6))           # a sphere and a tall static: not road
    speed = np.array([[4.0, 6.5, -1.0, 0.0]], np.float32)
    o = oracle.observe_vec(prims[None], 4, speed, K=4, M=3, radius=100.0)
    assert o["agent_idx"][0, 0].tolist() == [2, 3, 1, -1]                       # by distance 5, 7, 10; padded
    f = o["agent_feat"][0, 0]
    exp = [(0, 5, 4.0, 1.8, 1, 0, -5.0, 1), (-7, 0, 2.0, 0.8, -1, 0, -4.0, 1), (10, 0, 5.0, 2.0, 0, 1, 2.5, 1), (0,) * 8]
    assert np.allclose(f, np.array(exp, np.float32), atol=2e-6)
    assert o["road_idx"][0, 0].tolist() == [5, 4, -1]                           # centres at distance sqrt(5), sqrt(45)
    g = o["road_feat"][0, 0]
    expg = [(2, 1, 15.0, 1, 0, 6, 1, 0), (6, -3, 8.0, 0, 1, 2, 1, 0), (0,) * 8]
    assert np.allclose(g, np.array(expg, np.float32), atol=2e-6)
    # the view from neighbour C (heading reversed): the ego is 7 m BEHIND... no: C looks away from the ego -> ego at (-7, 0)
    assert o["agent_idx"][0, 3, 0] == 0 and np.allclose(o["agent_feat"][0, 3, 0, :2], (-7, 0), atol=2e-6)
    assert np.allclose(o["agent_feat"][0, 3, 0, 4:7], (-1, 0, 4.0), atol=2e-6)


def test_radius_boundary_ties_and_self_exclusion():
    # on the radius: included (d2 <= r^2); beyond: excluded; equal distances: lower index first; never itself
    prims = stack(veh(0, 0), veh(0, -30.0), veh(100.0, 0), veh(0, 30.0), veh(100.5, 0), veh(-60.0, 80.0))
    speed = np.zeros((1, 6), np.float32)
    o = oracle.observe_vec(prims[None], 6, speed, K=6, M=0, radius=100.0)
    assert o["agent_idx"][0, 0].tolist() == [1, 3, 2, 5, -1, -1]
    assert (o["agent_feat"][0, 0, 4:] == 0).all() and (o["agent_feat"][0, 0, :4, 7] == 1).all()
    for i in range(6):
        assert i not in o["agent_idx"][0, i].tolist()
    o2 = oracle.observe_vec(prims[None], 6, speed, K=2, M=0, radius=100.0)      # K smaller than the neighbourhood
    assert o2["agent_idx"][0, 0].tolist() == [1, 3]
    assert np.array_equal(o2["agent_feat"][0, 0], o["agent_feat"][0, 0, :2])


@pytest.mark.parametrize("seed", range(4))
def test_random_scenes_against_an_independent_fp64_argsort(seed):
    cfg = gs.SceneConfig("ov", 60 + seed, 3, 24, 80, 120.0, 32, 32)
    agents, quads = gs.gen_world_prims(cfg)
    prims = np.concatenate([agents, quads], axis=1)
    rng = np.random.default_rng(seed)
    speed = rng.uniform(-2, 15, (cfg.n_worlds, cfg.agents)).astype(np.float32)
    K, M, R = 8, 12, 45.0
    o = oracle.observe_vec(prims, cfg.agents, speed, K, M, R)
    for w in range(cfg.n_worlds):
        x, y = prims[w]["cx"].astype(np.float64), prims[w]["cy"].astype(np.float64)
        ck, sk = prims[w]["cos_yaw"].astype(np.float64), prims[w]["sin_yaw"].astype(np.float64)
        for i in range(cfg.agents):
            d = np.hypot(x - x[i], y - y[i])
            for lo, hi, cnt, idx, feat in ((0, cfg.agents, K, o["agent_idx"][w, i], o["agent_feat"][w, i]),
                                           (cfg.agents, cfg.prims, M, o["road_idx"][w, i], o["road_feat"][w, i])):
                cand = [j for j in range(lo, hi) if j != i and d[j] <= R - 1e-4]
                edge = [j for j in range(lo, hi) if j != i and abs(d[j] - R) <= 1e-4]
                order = sorted(cand, key=lambda j: d[j])
                gaps = np.diff([d[j] for j in order])
                if edge or (len(gaps) and gaps.min() < 1e-4):
                    continue                                            # fp32 could legitimately order these differently
                want = (order + [-1] * cnt)[:cnt]
                assert idx.tolist() == want, (w, i)
                for r, j in enumerate(want):
                    if j < 0:
                        assert (feat[r] == 0).all()
                        continue
                    dx, dy = x[j] - x[i], y[j] - y[i]
                    rel = (ck[i] * dx + sk[i] * dy, -sk[i] * dx + ck[i] * dy)
                    assert np.allclose(feat[r, :2], rel, atol=1e-4)
                    dc, ds = ck[i] * ck[j] + sk[i] * sk[j], ck[i] * sk[j] - sk[i] * ck[j]
                    if lo == 0:
                        assert np.allclose(feat[r, 2:4], (2 * prims[w]["hx"][j], 2 * prims[w]["hy"][j]))
                        assert np.allclose(feat[r, 4:6], (dc, ds), atol=1e-6)
                        assert feat[r, 6] == speed[w, j] - speed[w, i] and feat[r, 7] == 1
                    else:
                        assert feat[r, 2] == 2 * prims[w]["hx"][j] and np.allclose(feat[r, 3:5], (dc, ds), atol=1e-6)
                        assert feat[r, 5] == prims[w]["cls"][j] and feat[r, 6] == 1 and feat[r, 7] == 0


# ------------------------------------------------------------------------------------------------ update order D3-D5
# PAPER.md:335 gives no update order (it defers to [16]); DESIGN.md "Dynamics contract" reads it as: accelerations, then
# speed, then the steering demand from the NEW speed and NEW lateral acceleration, then the heading from the NEW speed and
# NEW angle, then the position from the NEW speed and NEW heading.  One-step closed forms that tell each choice from "old":
def test_d5_position_uses_the_new_heading():
    # heading 0, speed 10, angle d0 held (a_lat demands exactly d0, no jerks): psi1 = v tan(d0) / L dt, and the step is
    # taken along psi1 - so y1 = v sin(psi1) dt is not 0, as it would be along the old heading
    L, v, d0, dt = 0.6 * 2 * 2.0, 10.0, 0.2, 0.1
    par = oracle.make_dyn_params(dt=dt, a_lat_max=20.0, v_max=30.0)
    st, ps = fresh(v=v, a_lat=v * v * math.tan(d0) / L, steer=d0)
    s1, p1 = oracle.dynamics_step(par, [act(0.0, 0.0)], [2.0], st, ps)
    psi1 = v * math.tan(d0) / L * dt
    assert abs(s1[0, 3] - d0) < 1e-6 and abs(s1[0, 4] - psi1) < 1e-6
    assert abs(p1[0, 1] - v * math.sin(psi1) * dt) < 1e-6 and p1[0, 1] > 0.08
    assert abs(p1[0, 0] - v * math.cos(psi1) * dt) < 1e-6


def test_d4_heading_uses_the_new_speed():
    # angle frozen by a zero steering rate, longitudinal acceleration 4 held: psi1 = v' tan(d0) / L dt with v' = v + a_lon dt
    # (with the old speed it would be 3.4e-3 rad less); the position moves with v' as well
    L, v, d0, dt, a_lon = 0.6 * 2 * 2.0, 10.0, 0.2, 0.1, 4.0
    par = oracle.make_dyn_params(dt=dt, steer_rate_max=0.0, v_max=30.0)
    st, ps = fresh(v=v, a_lon=a_lon, steer=d0)
    s1, p1 = oracle.dynamics_step(par, [act(0.0, 0.0)], [2.0], st, ps)
    v1 = v + a_lon * dt
    psi1 = v1 * math.tan(d0) / L * dt
    assert abs(s1[0, 0] - v1) < 1e-5 and s1[0, 3] == np.float32(d0)
    assert abs(s1[0, 4] - psi1) < 1e-6 and abs(psi1 - v * math.tan(d0) / L * dt) > 3e-3
    assert abs(p1[0, 0] - v1 * math.cos(psi1) * dt) < 1e-6 and abs(p1[0, 1] - v1 * math.sin(psi1) * dt) < 1e-6


def test_d3_steering_demand_uses_the_new_speed_and_lateral_acceleration():
    # demand neither rate- nor magnitude-limited: d1 = atan(L a_lat' / v'^2) with a_lat' = a_lat + j_lat dt and
    # v' = v + a_lon dt; and since tan(d1) / L = a_lat' / v'^2, the heading advances by exactly a_lat' / v' dt (yaw rate =
    # lateral acceleration / speed, D4 with the new angle)
    L, v, dt, a_lon, a_lat = 0.6 * 2 * 2.0, 10.0, 0.1, 4.0, 2.0
    par = oracle.make_dyn_params(dt=dt, steer_rate_max=100.0, steer_max=1.0, v_max=30.0, a_lat_max=10.0)
    st, ps = fresh(v=v, a_lon=a_lon, a_lat=a_lat)
    s1, _ = oracle.dynamics_step(par, [act(0.0, 4.0)], [2.0], st, ps)
    v1, al1 = v + a_lon * dt, a_lat + 4.0 * dt
    d1 = math.atan(L * al1 / (v1 * v1))
    assert abs(s1[0, 2] - al1) < 1e-6 and abs(s1[0, 3] - d1) < 1e-6
    assert abs(d1 - math.atan(L * al1 / (v * v))) > 3e-3 and abs(d1 - math.atan(L * a_lat / (v1 * v1))) > 3e-3
    assert abs(s1[0, 4] - al1 / v1 * dt) < 1e-6


def test_heading_wrap_after_more_than_a_full_turn_in_one_step():
    # D4 wraps the heading into [-pi, pi); a short vehicle at full lock turns several times in one step:
    # v = 20, angle 1.2 frozen, L = 0.6 * 2 * 0.25 = 0.3 -> 20 tan(1.2) / 0.3 * 0.1 = 17.15 rad = 2.73 turns.  ADVICE r2.
    for psi0, sgn in ((0.3, 1.0), (-2.0, -1.0)):
        par = oracle.make_dyn_params(dt=0.1, steer_max=1.3, steer_rate_max=0.0, v_max=30.0)
        st, ps = fresh(v=20.0, steer=sgn * 1.2, psi=psi0)
        s1, p1 = oracle.dynamics_step(par, [act(0.0, 0.0)], [0.25], st, ps)
        turned = psi0 + sgn * 20.0 * math.tan(1.2) / 0.3 * 0.1
        assert abs(turned) > 2 * math.pi + 1.0
        want = (turned + math.pi) % (2 * math.pi) - math.pi
        assert -math.pi <= s1[0, 4] < math.pi and abs(s1[0, 4] - want) < 1e-5
        assert abs(p1[0, 2] - math.cos(turned)) < 1e-5 and abs(p1[0, 3] - math.sin(turned)) < 1e-5
        assert abs(p1[0, 0] - 2.0 * math.cos(turned)) < 1e-5 and abs(p1[0, 1] - 2.0 * math.sin(turned)) < 1e-5


def test_zero_length_agent_is_left_untouched():
    # the wheelbase is 0.6 * length: an agent record of zero length has no curvature tan(steer) / L, so the step skips it
    # like an agent with an invalid action instead of writing inf / NaN into its state
    par = oracle.make_dyn_params()
    st, ps = fresh(n=2, v=5.0, steer=0.1, a_lat=1.0)
    with pytest.raises(ValueError):
        oracle.dynamics_step(par, [act(4.0, 4.0)] * 2, [2.0, 0.0], st, ps)
    s1, p1 = oracle.dynamics_step(par, [act(4.0, 4.0)] * 2, [2.0, 0.0], st, ps, strict=False)
    assert np.array_equal(s1[1], st[1]) and np.array_equal(p1[1], ps[1])
    assert s1[0, 0] > 5.0 and p1[0, 0] > 0.4 and np.isfinite(s1).all() and np.isfinite(p1).all()
