"""ctypes front end of the CPU oracle (gp_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from the CUDA path.
"""
from __future__ import annotations

import ctypes
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from .build import build as _build

_PRIM_BYTES = 48


class Params(ctypes.Structure):
    _fields_ = [("cam_height", ctypes.c_float), ("t_max", ctypes.c_float),
                ("fov_rad", ctypes.c_float), ("ambient", ctypes.c_float),
                ("light", ctypes.c_float * 3), ("palette", (ctypes.c_uint8 * 3) * 8)]


class Cam(ctypes.Structure):
    """One camera of the per-agent rig: cos / sin of the yaw offset (positive = left), mount position
    along the agent's axis in half lengths (+1 front-centre, -1 rear-centre)."""
    _fields_ = [("cd", ctypes.c_float), ("sd", ctypes.c_float), ("mount", ctypes.c_float)]


class DynParams(ctypes.Structure):
    """Limits of the jerk-actuated kinematic bicycle (gp_sim_oracle.c)."""
    _fields_ = [("dt", ctypes.c_float), ("a_lon_max", ctypes.c_float), ("a_lat_max", ctypes.c_float),
                ("v_max", ctypes.c_float), ("steer_max", ctypes.c_float), ("steer_rate_max", ctypes.c_float),
                ("v_eps", ctypes.c_float), ("extent", ctypes.c_float)]


def make_dyn_params(dt=0.1, a_lon_max=6.0, a_lat_max=4.0, v_max=20.0, steer_max=0.6, steer_rate_max=0.8, v_eps=0.5,
                    extent=0.0) -> DynParams:
    p = DynParams()
    p.dt, p.a_lon_max, p.a_lat_max, p.v_max = dt, a_lon_max, a_lat_max, v_max
    p.steer_max, p.steer_rate_max, p.v_eps, p.extent = steer_max, steer_rate_max, v_eps, extent
    return p


PALETTE = ((135, 206, 235), (90, 90, 90), (240, 240, 240), (40, 80, 220),
           (220, 60, 60), (240, 160, 40), (150, 110, 70), (250, 240, 80))


def make_params(cam_height=1.6, t_max=100.0, fov_rad=np.float32(np.pi / 2), ambient=0.25,
                light=(0.48, 0.36, 0.8), palette=PALETTE) -> Params:
    p = Params()
    p.cam_height, p.t_max, p.fov_rad, p.ambient = cam_height, t_max, float(fov_rad), ambient
    for i in range(3):
        p.light[i] = light[i]
    for c in range(8):
        for ch in range(3):
            p.palette[c][ch] = int(palette[c][ch]) if c < len(palette) else 0
    return p


def _cam(cam):
    if cam is None:
        return None
    c = Cam()
    c.cd, c.sd, c.mount = float(np.float32(cam[0])), float(np.float32(cam[1])), float(np.float32(cam[2]))
    return ctypes.byref(c)


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build())
        vp, ci, cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
        L.orc_render_view.argtypes = [vp, ci, ci, cf, cf, vp, ctypes.POINTER(Params), ci, ci,
                                      vp, vp, vp, vp, vp, vp]
        L.orc_render_view.restype = ci
        L.orc_shadow_view.argtypes = [vp, ci, ci, cf, cf, vp, ctypes.POINTER(Params), ci, ci,
                                      vp, vp, vp, vp]
        L.orc_shadow_view.restype = ci
        L.orc_polyline_quads.argtypes = [vp, ci, ci, cf, cf, ci, ci, vp]
        L.orc_polyline_quads.restype = ci
        L.orc_dynamics_step.argtypes = [ctypes.POINTER(DynParams), ci, vp, vp, vp, vp]
        L.orc_dynamics_step.restype = ci
        L.orc_observe_vec.argtypes = [vp, ci, ci, vp, ci, ci, cf, vp, vp, vp, vp]
        L.orc_observe_vec.restype = ci
        _lib = L
    return _lib


def polyline_quads(points, half_width=0.075, z=0.01, cls=2, inst0=0, dtype=None):
    """C1p: polylines [n_lines][pts][2] fp32 -> flat quads, one per segment (structured array of 48-byte
    records; pass the generator's PRIM_DTYPE as `dtype`)."""
    pts = np.ascontiguousarray(points, dtype=np.float32)
    assert pts.ndim == 3 and pts.shape[2] == 2 and pts.shape[1] >= 2
    n = pts.shape[0] * (pts.shape[1] - 1)
    out = np.zeros(n, dtype=dtype if dtype is not None else np.dtype([("raw", "u1", (_PRIM_BYTES,))]))
    assert out.dtype.itemsize == _PRIM_BYTES
    rc = lib().orc_polyline_quads(pts.ctypes.data, pts.shape[0], pts.shape[1], float(half_width), float(z),
                                  int(cls), int(inst0), out.ctypes.data)
    if rc != n:
        raise ValueError("orc_polyline_quads: bad arguments")
    return out


def _check_prims(prims):
    prims = np.ascontiguousarray(prims)
    assert prims.dtype.itemsize == _PRIM_BYTES and prims.ndim == 1, (prims.dtype, prims.shape)
    return prims


def render_view(prims, ego, H, W, params=None, cp=1.0, sp=0.0, rgb=True, cam=None):
    """fp32-contract render of one view.  prims: 1-D structured array (48-byte records) of the
    ego's world.  cam: (cos d, sin d, mount) of the rig camera, None = the front camera (1, 0, 1).  Returns dict(cls u8[H,W], inst i32[H,W], depth f32[H,W], rgb u8[3,H,W] or None,
    t2 f32[H,W], win i32[H,W])."""
    prims = _check_prims(prims)
    params = params or make_params()
    out = {"cls": np.empty((H, W), np.uint8), "inst": np.empty((H, W), np.int32),
           "depth": np.empty((H, W), np.float32),
           "rgb": np.empty((3, H, W), np.uint8) if rgb else None,
           "t2": np.empty((H, W), np.float32), "win": np.empty((H, W), np.int32)}
    rc = lib().orc_render_view(prims.ctypes.data, len(prims), int(ego), float(cp), float(sp), _cam(cam),
                               ctypes.byref(params), H, W,
                               out["cls"].ctypes.data, out["inst"].ctypes.data, out["depth"].ctypes.data,
                               out["rgb"].ctypes.data if rgb else None,
                               out["t2"].ctypes.data, out["win"].ctypes.data)
    if rc != 0:
        raise ValueError("orc_render_view: bad arguments")
    return out


def shadow_view(prims, ego, H, W, params=None, cp=1.0, sp=0.0, cam=None):
    """fp64 face-enumeration render of one view: dict(win i32, depth f64, t2 f64, ndl f64)."""
    prims = _check_prims(prims)
    params = params or make_params()
    out = {"win": np.empty((H, W), np.int32), "depth": np.empty((H, W), np.float64),
           "t2": np.empty((H, W), np.float64), "ndl": np.empty((H, W), np.float64)}
    rc = lib().orc_shadow_view(prims.ctypes.data, len(prims), int(ego), float(cp), float(sp), _cam(cam),
                               ctypes.byref(params), H, W, out["win"].ctypes.data,
                               out["depth"].ctypes.data, out["t2"].ctypes.data, out["ndl"].ctypes.data)
    if rc != 0:
        raise ValueError("orc_shadow_view: bad arguments")
    return out


def render_views(world_prims, views, H, W, params=None, pitch_cs=None, rgb=True, threads=1,
                 shadow=False, rig=None):
    """Render a list of (world, agent) or, with a rig [(cos d, sin d, mount), ...], (world, agent,
    camera) views.  world_prims: [Wn][P] structured array.  The
    renderer itself is single-threaded; `threads` > 1 runs the same code over disjoint views
    (ctypes releases the GIL).  Returns a list of dicts in the order of `views`."""
    params = params or make_params()

    def one(wa):
        w, a = wa[0], wa[1]
        cp, sp = (1.0, 0.0) if pitch_cs is None else (float(pitch_cs[w, a, 0]), float(pitch_cs[w, a, 1]))
        fn = shadow_view if shadow else render_view
        kw = {} if shadow else {"rgb": rgb}
        if len(wa) > 2:
            kw["cam"] = rig[wa[2]]
        return fn(world_prims[w], a, H, W, params, cp, sp, **kw)

    if threads <= 1:
        return [one(v) for v in views]
    with ThreadPoolExecutor(max_workers=threads) as ex:
        return list(ex.map(one, views))


def dynamics_step(params, action, half_len, state, pose, strict=True):
    """One step of the jerk bicycle for n agents (fp64 inside, fp32 in / out).  action int32 [n], half_len fp32 [n],
    state fp32 [n][8] = (v, a_lon, a_lat, steer, psi, -, -, -), pose fp32 [n][4] = (x, y, cos psi, sin psi).
    Returns (new_state, new_pose); the inputs are not modified.  An action outside [0, 12) or a half length <= 0 leaves
    that agent untouched: ValueError when `strict`, otherwise the result with those agents unchanged."""
    action = np.ascontiguousarray(action, dtype=np.int32).reshape(-1)
    n = action.size
    half_len = np.ascontiguousarray(half_len, dtype=np.float32).reshape(n)
    st = np.array(state, dtype=np.float32, copy=True).reshape(n, 8)
    ps = np.array(pose, dtype=np.float32, copy=True).reshape(n, 4)
    rc = lib().orc_dynamics_step(ctypes.byref(params), n, action.ctypes.data, half_len.ctypes.data,
                                 st.ctypes.data, ps.ctypes.data)
    if rc != 0 and (strict or rc != -2):
        raise ValueError("orc_dynamics_step: bad arguments (%d)" % rc)
    return st.reshape(np.shape(state)), ps.reshape(np.shape(pose))


def observe_vec(world_prims, n_agents, speed, K, M, radius=100.0):
    """O_vec of every agent of every world.  world_prims [Wn][P] 48-byte records (agents first), speed fp32 [Wn][A].
    Returns dict(agent_idx i32 [Wn][A][K], agent_feat f32 [Wn][A][K][8], road_idx i32 [Wn][A][M], road_feat f32
    [Wn][A][M][8])."""
    prims = np.ascontiguousarray(world_prims)
    assert prims.ndim == 2 and prims.dtype.itemsize == _PRIM_BYTES
    Wn, P = prims.shape
    A = int(n_agents)
    speed = np.ascontiguousarray(speed, dtype=np.float32).reshape(Wn, A)
    out = {"agent_idx": np.empty((Wn, A, K), np.int32), "agent_feat": np.empty((Wn, A, K, 8), np.float32),
           "road_idx": np.empty((Wn, A, M), np.int32), "road_feat": np.empty((Wn, A, M, 8), np.float32)}
    for w in range(Wn):
        rc = lib().orc_observe_vec(prims[w].ctypes.data, P, A, speed[w].ctypes.data, int(K), int(M), float(radius),
                                   out["agent_idx"][w].ctypes.data, out["agent_feat"][w].ctypes.data,
                                   out["road_idx"][w].ctypes.data, out["road_feat"][w].ctypes.data)
        if rc != 0:
            raise ValueError("orc_observe_vec: bad arguments")
    return out
