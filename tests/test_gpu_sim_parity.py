"""Parity of gp_dynamics_step and gp_observe_vec (through the C ABI) with the CPU oracle (oracle/gp_sim_oracle.c).
Needs a B200: `pytest -m gpu`.

O_vec: indices and features bit-exact (contract O1-O3 is fp32 add / mul / fma in a fixed order on both sides).
Dynamics: fp32 kernel with atanf / tanf / sincosf against the fp64 oracle — tolerance, derived in DESIGN.md
"Dynamics contract": every quantity is a handful of fp32 operations (each <= 0.5 ulp) and at most three libm calls
(<= 4 ulp each) away from its inputs, so per step |error| <= ~8 ulp of the quantity's magnitude bound:
    speed, accelerations (|.| <= 30)       2e-5 absolute
    steering angle, heading (|.| <= pi)    4e-6 absolute (heading compared modulo 2 pi)
    cos, sin                               4e-6 absolute
    position (|.| <= 100 m)                4e-5 absolute (compared modulo the torus extent)
"""
import math

import numpy as np
import pytest

import gp_scenes as gs
import oracle
from parity_util import gpu_render, world_prims

pytestmark = pytest.mark.gpu

TOL_V, TOL_ANG, TOL_CS, TOL_POS = 2e-5, 4e-6, 4e-6, 4e-5
PAR = dict(dt=0.1, a_lon_max=6.0, a_lat_max=4.0, v_max=20.0, steer_max=0.6, steer_rate_max=0.8, v_eps=0.5, extent=0.0)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a GPU"
    return torch


def renderer_for(cfg, agents, quads):
    from paper_2606_19641_b200 import Renderer
    r = Renderer(0)
    r.scene_upload(agents, quads, cam_height=cfg.cam_height, t_max=cfg.t_max)
    return r


def initial_state(cfg, agents, seed):
    rng = np.random.default_rng(seed)
    Wn, A = agents.shape
    st = np.zeros((Wn, A, 8), np.float32)
    psi = np.arctan2(agents["sin_yaw"].astype(np.float64), agents["cos_yaw"].astype(np.float64))
    st[..., 0] = rng.uniform(0, 18, (Wn, A))
    st[..., 1] = rng.uniform(-5, 5, (Wn, A))
    st[..., 2] = rng.uniform(-3.5, 3.5, (Wn, A))
    st[..., 3] = rng.uniform(-0.5, 0.5, (Wn, A))
    st[..., 4] = psi
    st[..., 5:] = rng.uniform(-1, 1, (Wn, A, 3))                 # unused slots must be carried through untouched
    pose = np.stack([agents["cx"], agents["cy"], np.cos(psi), np.sin(psi)], axis=-1).astype(np.float32)
    return st, pose


def ang_diff(a, b):
    return np.abs((a.astype(np.float64) - b + math.pi) % (2 * math.pi) - math.pi)


def check_dyn(g_st, g_pose, o_st, o_pose, extent):
    assert np.abs(g_st[..., 0:3].astype(np.float64) - o_st[..., 0:3]).max() <= TOL_V
    assert np.abs(g_st[..., 3].astype(np.float64) - o_st[..., 3]).max() <= TOL_ANG
    assert ang_diff(g_st[..., 4], o_st[..., 4]).max() <= TOL_ANG
    assert ((g_st[..., 4] >= -math.pi - 1e-6) & (g_st[..., 4] < math.pi + 1e-6)).all()
    assert np.array_equal(g_st[..., 5:], o_st[..., 5:])
    assert np.abs(g_pose[..., 2:].astype(np.float64) - o_pose[..., 2:]).max() <= TOL_CS
    d = g_pose[..., :2].astype(np.float64) - o_pose[..., :2]
    if extent > 0:
        d = (d + 0.5 * extent) % extent - 0.5 * extent
    assert np.abs(d).max() <= TOL_POS


@pytest.mark.parametrize("extent", [0.0, 150.0])
def test_dynamics_single_steps_all_actions(torch_cuda, extent):
    # every agent of a paper-shaped batch takes every one of the twelve actions from a random state: each GPU step is
    # compared with the oracle's step FROM THE SAME fp32 state (no accumulation)
    torch = torch_cuda
    cfg = gs.config("paper", n_worlds=24)
    agents, quads = gs.gen_world_prims(cfg)
    r = renderer_for(cfg, agents, quads)
    par = dict(PAR, extent=extent)
    opar = oracle.make_dyn_params(**par)
    half_len = agents["hx"].reshape(-1)
    rng = np.random.default_rng(3)
    for rep in range(4):
        st, pose = initial_state(cfg, agents, 10 + rep)
        if extent > 0:                                              # put some agents next to the torus seam
            pose[0, :, 0] = extent / 2 - rng.uniform(0, 0.3, cfg.agents)
            pose[1, :, 1] = -extent / 2 + rng.uniform(0, 0.3, cfg.agents)
        st[2, :, 4] = np.float32(math.pi) - rng.uniform(0, 0.02, cfg.agents).astype(np.float32)     # next to the heading wrap
        pose[2, :, 2], pose[2, :, 3] = np.cos(st[2, :, 4]), np.sin(st[2, :, 4])
        action = rng.integers(0, 12, agents.shape).astype(np.int32)
        action[3, :12] = np.arange(12)
        d_st, d_pose = torch.from_numpy(st).cuda(), torch.from_numpy(pose).cuda()
        r.dynamics_step(par, torch.from_numpy(action).cuda(), d_st, d_pose)
        o_st, o_pose = oracle.dynamics_step(opar, action, half_len, st.reshape(-1, 8), pose.reshape(-1, 4))
        check_dyn(d_st.cpu().numpy(), d_pose.cpu().numpy(), o_st.reshape(st.shape), o_pose.reshape(pose.shape), extent)
    r.close()


def test_dynamics_limits_and_invalid_actions(torch_cuda):
    torch = torch_cuda
    cfg = gs.config("small", n_worlds=4)
    agents, quads = gs.gen_world_prims(cfg)
    r = renderer_for(cfg, agents, quads)
    par = dict(PAR, a_lon_max=2.0, a_lat_max=1.5, v_max=6.0, steer_max=0.3, steer_rate_max=0.4)
    opar = oracle.make_dyn_params(**par)
    st, pose = initial_state(cfg, agents, 5)
    half_len = agents["hx"].reshape(-1)
    d_st, d_pose = torch.from_numpy(st).cuda(), torch.from_numpy(pose).cuda()
    o_st, o_pose = st.reshape(-1, 8).copy(), pose.reshape(-1, 4).copy()
    rng = np.random.default_rng(1)
    for step in range(40):                      # saturate: everybody accelerates and steers hard
        action = np.where(rng.random(agents.shape) < 0.8, 11, 0).astype(np.int32)
        d_act = torch.from_numpy(action).cuda()
        # one GPU step from the ORACLE's current state (inputs flow oracle -> GPU, never the other way) ...
        s_st, s_pose = torch.from_numpy(o_st.reshape(st.shape)).cuda(), torch.from_numpy(o_pose.reshape(pose.shape)).cuda()
        r.dynamics_step(par, d_act, s_st, s_pose)
        o_st, o_pose = oracle.dynamics_step(opar, action, half_len, o_st, o_pose)
        check_dyn(s_st.cpu().numpy().reshape(-1, 8), s_pose.cpu().numpy().reshape(-1, 4), o_st, o_pose, 0.0)
        # ... and the GPU's own free-running trajectory with the same actions
        r.dynamics_step(par, d_act, d_st, d_pose)
    g = d_st.cpu().numpy()
    assert g[..., 0].max() <= 6.0 and g[..., 0].min() >= 0.0 and np.abs(g[..., 1]).max() <= 2.0
    assert np.abs(g[..., 2]).max() <= 1.5 and np.abs(g[..., 3]).max() <= 0.3 + 1e-7
    assert (g[..., 0] == 6.0).any() and (np.abs(g[..., 3]) >= 0.3 - 1e-6).any()
    # 40 accumulated steps: the two trajectories stay within a millimetre
    assert np.abs(d_pose.cpu().numpy().reshape(-1, 4)[:, :2].astype(np.float64) - o_pose[:, :2]).max() < 1e-3
    # invalid actions leave an agent untouched
    before = (d_st.clone(), d_pose.clone())
    bad = np.full(agents.shape, 12, np.int32); bad[0, 0] = -1
    r.dynamics_step(par, torch.from_numpy(bad).cuda(), d_st, d_pose)
    assert torch.equal(before[0], d_st) and torch.equal(before[1], d_pose)
    r.close()


def test_dynamics_full_turns_zero_length_and_steer_limit(torch_cuda):
    """more than a full turn in one step still lands in [-pi, pi); an agent record of zero length (no wheelbase)
    is left untouched instead of turning NaN; steer_max >= pi/2 is refused."""
    torch = torch_cuda
    from paper_2606_19641_b200 import GpError, gp
    cfg = gs.config("small", n_worlds=4)
    agents, quads = gs.gen_world_prims(cfg)
    agents = agents.copy()
    agents["hx"][1, :] = 0.25                                    # L = 0.3 m: 17 rad per step at full lock
    agents["hx"][2, ::2] = 0.0                                   # zero length
    r = renderer_for(cfg, agents, quads)
    par = dict(PAR, steer_max=1.3, steer_rate_max=0.0, v_max=30.0)
    st, pose = initial_state(cfg, agents, 21)
    st[1, :, 0] = 20.0
    st[1, :, 3] = np.where(np.arange(cfg.agents) % 2, 1.2, -1.2)
    action = np.full(agents.shape, 7, np.int32)                  # zero jerks
    d_st, d_pose = torch.from_numpy(st).cuda(), torch.from_numpy(pose).cuda()
    r.dynamics_step(par, torch.from_numpy(action).cuda(), d_st, d_pose)
    o_st, o_pose = oracle.dynamics_step(oracle.make_dyn_params(**par), action, agents["hx"].reshape(-1), st.reshape(-1, 8),
                                        pose.reshape(-1, 4), strict=False)
    g_st, g_pose = d_st.cpu().numpy(), d_pose.cpu().numpy()
    o_st, o_pose = o_st.reshape(st.shape), o_pose.reshape(pose.shape)
    assert np.isfinite(g_st).all() and np.isfinite(g_pose).all()
    assert np.array_equal(g_st[2, ::2], st[2, ::2]) and np.array_equal(g_pose[2, ::2], pose[2, ::2])
    assert np.array_equal(o_st[2, ::2], st[2, ::2])
    assert ((g_st[..., 4] >= -math.pi) & (g_st[..., 4] < math.pi + 1e-6)).all()
    turned = np.abs(20.0 * math.tan(1.2) / 0.3 * 0.1)
    assert turned > 4 * math.pi
    # a heading of 17 rad before the wrap carries ~8 ulp(17) = 1.5e-5 of fp32 error: the tolerance scales with it
    assert ang_diff(g_st[..., 4], o_st[..., 4]).max() <= 3e-5
    assert np.abs(g_pose[..., 2:].astype(np.float64) - o_pose[..., 2:]).max() <= 3e-5
    assert np.abs(g_pose[..., :2].astype(np.float64) - o_pose[..., :2]).max() <= 1e-4
    keep = np.ones(agents.shape, bool); keep[1] = False
    check_dyn(g_st[keep], g_pose[keep], o_st[keep], o_pose[keep], 0.0)      # everyone else at the usual tolerance
    for bad in (math.pi / 2, 2.0):
        with pytest.raises(GpError) as ei:
            r.dynamics_step(dict(PAR, steer_max=bad), torch.from_numpy(action).cuda(), d_st, d_pose)
        assert ei.value.code == gp.GP_ERR_ARG
    r.close()


def test_dynamics_feeds_the_renderer_without_the_host(torch_cuda):
    # gp_dynamics_step also performs the pose update a0: rendering right after it must equal, bit for bit, rendering
    # after an explicit gp_agents_update with the pose buffer it produced (render parity itself: test_gpu_parity.py)
    torch = torch_cuda
    cfg = gs.config("small", n_worlds=6)
    agents, quads = gs.gen_world_prims(cfg)
    st, pose = initial_state(cfg, agents, 8)
    r = renderer_for(cfg, agents, quads)
    d_st, d_pose = torch.from_numpy(st).cuda(), torch.from_numpy(pose).cuda()
    rng = np.random.default_rng(2)
    for _ in range(3):
        r.dynamics_step(PAR, torch.from_numpy(rng.integers(0, 12, agents.shape).astype(np.int32)).cuda(), d_st, d_pose)
    a = gpu_render(r, cfg, 0, cfg.n_worlds)
    r2 = renderer_for(cfg, agents, quads)
    r2.agents_update(d_pose)
    b = gpu_render(r2, cfg, 0, cfg.n_worlds)
    for x, y in zip(a, b):
        assert torch.equal(x, y)
    r.close(); r2.close()


# ------------------------------------------------------------------------------------------------ O_vec
def obs_gpu(torch, r, cfg, speed, K, M, radius):
    Wn, A = cfg.n_worlds, cfg.agents
    st = np.zeros((Wn, A, 8), np.float32)
    st[..., 0] = speed
    dev = "cuda"
    out = (torch.full((Wn, A, max(K, 1)), -7, dtype=torch.int32, device=dev)[:, :, :K].contiguous(),
           torch.full((Wn, A, K, 8), float("nan"), dtype=torch.float32, device=dev),
           torch.full((Wn, A, max(M, 1)), -7, dtype=torch.int32, device=dev)[:, :, :M].contiguous(),
           torch.full((Wn, A, M, 8), float("nan"), dtype=torch.float32, device=dev))
    r.observe_vec(torch.from_numpy(st).cuda(), K, M, radius, out[0] if K else None, out[1] if K else None,
                  out[2] if M else None, out[3] if M else None)
    torch.cuda.synchronize()
    return [o.cpu().numpy() for o in out]


def check_obs(got, ref, K, M):
    if K:
        assert np.array_equal(got[0], ref["agent_idx"])
        assert np.array_equal(got[1].view(np.uint32), ref["agent_feat"].view(np.uint32))        # bit-exact, signed zeros included
    if M:
        assert np.array_equal(got[2], ref["road_idx"])
        assert np.array_equal(got[3].view(np.uint32), ref["road_feat"].view(np.uint32))


@pytest.mark.parametrize("name,n_worlds,K,M,radius", [("tiny", 1, 3, 5, 100.0), ("small", 24, 8, 16, 40.0),
                                                      ("paper", 12, 16, 32, 100.0), ("paper", 6, 63, 200, 1000.0),
                                                      ("dense", 3, 16, 32, 30.0), ("rig4", 6, 12, 24, 60.0)])
def test_observe_vec_bit_exact(torch_cuda, name, n_worlds, K, M, radius):
    torch = torch_cuda
    cfg = gs.config(name, n_worlds=n_worlds)
    agents, quads = gs.gen_world_prims(cfg)
    r = renderer_for(cfg, agents, quads)
    speed = np.random.default_rng(4).uniform(-3, 18, agents.shape).astype(np.float32)
    got = obs_gpu(torch, r, cfg, speed, K, M, radius)
    ref = oracle.observe_vec(world_prims(agents, quads), cfg.agents, speed, K, M, radius)
    check_obs(got, ref, K, M)
    if name == "paper" and K == 63:
        assert (got[0] >= 0).all() and (got[2] >= 0).all()          # everything is within 1000 m: full lists
    if name == "rig4":                                              # spheres and tall statics are not road segments
        P = world_prims(agents, quads)
        sel = got[2][got[2] >= 0]
        assert len(sel) and (P[0]["hz"][sel % P.shape[1]] == 0).all()
    r.close()


def test_observe_vec_follows_pose_updates_and_edge_cases(torch_cuda):
    torch = torch_cuda
    cfg = gs.config("small", n_worlds=5)
    agents, quads = gs.gen_world_prims(cfg)
    speedv, yaw_rate = gs.gen_dynamics(cfg)
    pose = gs.poses_at_frames(cfg, agents, speedv, yaw_rate, [7])[7]
    r = renderer_for(cfg, agents, quads)
    r.agents_update(torch.from_numpy(pose).cuda())
    moved = agents.copy()
    moved["cx"], moved["cy"], moved["cos_yaw"], moved["sin_yaw"] = pose[..., 0], pose[..., 1], pose[..., 2], pose[..., 3]
    speed = speedv.astype(np.float32)
    for K, M, radius in ((8, 8, 25.0), (0, 4, 50.0), (4, 0, 50.0), (40, 130, 5.0), (1, 1, 0.0)):
        got = obs_gpu(torch, r, cfg, speed, K, M, radius)
        ref = oracle.observe_vec(world_prims(moved, quads), cfg.agents, speed, K, M, radius)
        check_obs(got, ref, K, M)
    # coincident agents (distance exactly 0) and exact ties: lower index first
    tie = agents.copy()
    tie["cx"][:, 1:5] = tie["cx"][:, :1]; tie["cy"][:, 1:5] = tie["cy"][:, :1]
    r2 = renderer_for(cfg, tie, quads)
    got = obs_gpu(torch, r2, cfg, speed, 6, 3, 80.0)
    ref = oracle.observe_vec(world_prims(tie, quads), cfg.agents, speed, 6, 3, 80.0)
    check_obs(got, ref, 6, 3)
    assert got[0][0, 0, :4].tolist() == [1, 2, 3, 4] and got[0][0, 2, :4].tolist() == [0, 1, 3, 4]
    from paper_2606_19641_b200 import gp
    with pytest.raises(gp.GpError):
        r.observe_vec(torch.zeros((5, 32, 8), device="cuda"), 0, 0, 10.0, None, None, None, None)
    r.close(); r2.close()
