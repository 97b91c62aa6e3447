"""Counter-based, seeded generator of the five BASELINE.json workloads.

Everything here is plain numpy in float64, rounded once to float32 at the
end, so that the oracle and the CUDA path consume bit-identical inputs.
No renderer arithmetic lives here.

G1 RNG       : splitmix64; stream key = mix(seed, world, stream); draw n of a
               stream is mix64(key + (n+1)*GOLDEN); U[0,1) = (x >> 11) * 2^-53.
G2 vehicles  : per attempt L~U[4,5], W~U[1.8,2.1], cx,cy~U[-E/2,E/2); accepted
               iff its bounding circle (radius hypot(L,W)/2) touches no accepted
               circle; after acceptance yaw~U[-pi,pi); H = 1.5 m, bottom on z=0.
G3 quads     : cx,cy~U[-E/2,E/2), len~U[3,20], yaw~U[-pi,pi); 0.15 m wide, z=0.01,
               zero thickness.
G4 dynamics  : speed~U[0,15] m/s, yaw_rate~U[-0.3,0.3] rad/s, dt = 0.1 s,
               explicit Euler, positions wrap onto the torus [-E/2,E/2).
G5 cameras   : pitch 0, except 'dense' where pitch~U[-5,5] deg per camera.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

CLASS_SKY, CLASS_GROUND, CLASS_MARKING, CLASS_VEHICLE = 0, 1, 2, 3
CLASS_PEDESTRIAN, CLASS_CYCLIST, CLASS_OBSTACLE, CLASS_LIGHT = 4, 5, 6, 7      # PAPER.md:62 entity kinds
DEFAULT_PALETTE = np.array(
    [[135, 206, 235], [90, 90, 90], [240, 240, 240], [40, 80, 220],
     [220, 60, 60], [240, 160, 40], [150, 110, 70], [250, 240, 80]], dtype=np.uint8)

# Camera rigs: (yaw offset in degrees, positive = left; mount along the agent's axis in half lengths).
RIG_FRONT = ((0.0, 1.0),)                                         # BASELINE.json configs[0]
RIG_PAPER4 = ((0.0, 1.0), (60.0, 1.0), (-60.0, 1.0), (180.0, -1.0))  # front, front-left, front-right, rear


def rig_array(rig) -> np.ndarray:
    """[C][4] fp32 = (cos d, sin d, mount, 0) of a rig given as ((deg, mount), ...)."""
    out = np.zeros((len(rig), 4), dtype=np.float32)
    for i, (deg, mount) in enumerate(rig):
        q = round(deg / 90.0)
        if abs(deg - 90.0 * q) < 1e-12:          # exact quarter turns
            c, s_ = [(1.0, 0.0), (0.0, 1.0), (-1.0, 0.0), (0.0, -1.0)][q % 4]
        else:
            c, s_ = math.cos(math.radians(deg)), math.sin(math.radians(deg))
        out[i] = (c, s_, mount, 0.0)
    return out
DEFAULT_LIGHT = (0.48, 0.36, 0.8)
DEFAULT_AMBIENT = 0.25

# 48-byte primitive record: the layout both renderers read (SURVEY.md §8(b) gp_prim).
PRIM_DTYPE = np.dtype([
    ("cx", "<f4"), ("cy", "<f4"), ("cz", "<f4"),
    ("hx", "<f4"), ("hy", "<f4"), ("hz", "<f4"),
    ("cos_yaw", "<f4"), ("sin_yaw", "<f4"),
    ("cls", "<i4"), ("inst", "<i4"), ("shape", "<i4"), ("pad", "<i4"),
])
assert PRIM_DTYPE.itemsize == 48

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
SHAPE_BOX, SHAPE_SPHERE = 0, 1     # cuboids / planes (flat boxes), spheres for traffic lights
_STREAM_VEHICLES, _STREAM_QUADS, _STREAM_DYNAMICS, _STREAM_PITCH = 0, 1, 2, 3


@dataclasses.dataclass(frozen=True)
class SceneConfig:
    name: str
    seed: int
    n_worlds: int
    agents: int
    quads: int
    extent: float
    H: int
    W: int
    fov_deg: float = 90.0
    pitch_deg_max: float = 0.0
    t_max: float = 100.0
    cam_height: float = 1.6
    rgb: bool = True
    dt: float = 0.1
    rig: tuple = RIG_FRONT          # cameras per agent
    class_mix: bool = False         # some agents become vans (taller than the camera), pedestrians, cyclists
    lights: int = 0                 # traffic-light spheres per world, appended to the static primitives

    @property
    def statics(self) -> int:
        return self.quads + self.lights

    @property
    def prims(self) -> int:
        return self.agents + self.quads + self.lights

    @property
    def cams(self) -> int:
        return len(self.rig)

    @property
    def views(self) -> int:
        return self.n_worlds * self.agents * len(self.rig)

    @property
    def fov_rad(self) -> float:
        return math.radians(self.fov_deg)

    def replace(self, **kw) -> "SceneConfig":
        return dataclasses.replace(self, **kw)


# BASELINE.json configs[0..4]; seeds 0..4.
CONFIGS = {
    "tiny": SceneConfig("tiny", 0, 1, 4, 12, 60.0, 32, 32, rgb=False),
    "small": SceneConfig("small", 1, 256, 32, 120, 100.0, 64, 64),
    "paper": SceneConfig("paper", 2, 1024, 64, 200, 150.0, 128, 128),
    "sweep": SceneConfig("sweep", 3, 512, 64, 200, 150.0, 128, 128),
    "dense": SceneConfig("dense", 4, 2048, 128, 500, 100.0, 256, 256, pitch_deg_max=5.0),
    # the paper's training cameras (4 cameras at 210 x 126) and
    # entity kinds (vehicles, pedestrians, cyclists) on the paper-scale world recipe
    "rig4": SceneConfig("rig4", 5, 256, 64, 200, 150.0, 126, 210, rig=RIG_PAPER4, class_mix=True, lights=16),
}


def config(name: str, **overrides) -> SceneConfig:
    c = CONFIGS[name]
    return c.replace(**overrides) if overrides else c


def _mix64(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def _stream_keys(seed: int, worlds: np.ndarray, stream: int) -> np.ndarray:
    with np.errstate(over="ignore"):
        k = (np.uint64(seed) * _GOLDEN + worlds.astype(np.uint64)) * np.uint64(4) + np.uint64(stream)
        return _mix64(k * _GOLDEN + _GOLDEN)


def _draws(keys: np.ndarray, counter: np.ndarray) -> np.ndarray:
    """U[0,1) double: draw number `counter` (0-based) of each stream in `keys`."""
    with np.errstate(over="ignore"):
        x = _mix64(keys + (counter.astype(np.uint64) + np.uint64(1)) * _GOLDEN)
    return (x >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def splitmix64_stream(seed: int, world: int, stream: int, n: int) -> np.ndarray:
    """First n U[0,1) draws of one stream (used by tests to pin the RNG)."""
    keys = _stream_keys(seed, np.array([world]), stream)
    return _draws(np.repeat(keys, n), np.arange(n))


def _gen_vehicles(cfg: SceneConfig, worlds: np.ndarray):
    n, A, E = len(worlds), cfg.agents, cfg.extent
    keys = _stream_keys(cfg.seed, worlds, _STREAM_VEHICLES)
    ctr = np.zeros(n, dtype=np.int64)
    count = np.zeros(n, dtype=np.int64)
    cx = np.zeros((n, A)); cy = np.zeros((n, A)); rad = np.zeros((n, A))
    Ls = np.zeros((n, A)); Ws = np.zeros((n, A)); yaw = np.zeros((n, A))
    slot = np.arange(A)[None, :]
    for _ in range(100000):
        idx = np.nonzero(count < A)[0]
        if idx.size == 0:
            break
        k = keys[idx]; c = ctr[idx]
        L = 4.0 + _draws(k, c)
        Wd = 1.8 + 0.3 * _draws(k, c + 1)
        x = -0.5 * E + E * _draws(k, c + 2)
        y = -0.5 * E + E * _draws(k, c + 3)
        r = 0.5 * np.hypot(L, Wd)
        dx = cx[idx] - x[:, None]; dy = cy[idx] - y[:, None]
        rr = rad[idx] + r[:, None]
        clash = ((dx * dx + dy * dy) < rr * rr) & (slot < count[idx][:, None])
        ok = ~clash.any(axis=1)
        psi = -math.pi + 2.0 * math.pi * _draws(k, c + 4)   # consumed only on acceptance
        ctr[idx] = c + 4 + ok.astype(np.int64)
        ai = idx[ok]; s = count[ai]
        cx[ai, s] = x[ok]; cy[ai, s] = y[ok]; rad[ai, s] = r[ok]
        Ls[ai, s] = L[ok]; Ws[ai, s] = Wd[ok]; yaw[ai, s] = psi[ok]
        count[ai] += 1
    else:  # pragma: no cover
        raise RuntimeError("vehicle placement did not converge")
    return cx, cy, Ls, Ws, yaw


def gen_world_prims(cfg: SceneConfig, world_begin: int = 0, n_worlds: int | None = None):
    """Return (agents[Wn][A], statics[Wn][Q + lights]) structured arrays of PRIM_DTYPE at t=0."""
    n = cfg.n_worlds - world_begin if n_worlds is None else n_worlds
    worlds = np.arange(world_begin, world_begin + n)
    A, Q, E = cfg.agents, cfg.quads, cfg.extent
    agents = np.zeros((n, A), dtype=PRIM_DTYPE)
    if A:
        cx, cy, Ls, Ws, yaw = _gen_vehicles(cfg, worlds)
        agents["cx"] = cx; agents["cy"] = cy; agents["cz"] = 0.75
        agents["hx"] = 0.5 * Ls; agents["hy"] = 0.5 * Ws; agents["hz"] = 0.75
        agents["cos_yaw"] = np.cos(yaw); agents["sin_yaw"] = np.sin(yaw)
        agents["cls"] = CLASS_VEHICLE
        agents["inst"] = np.arange(A, dtype=np.int32)[None, :]
        if cfg.class_mix:
            # kind from the length draw u = L - 4: [0,.7) car, [.7,.8) van 3.2 m tall (taller than the
            # camera), [.8,.9) pedestrian 0.6 x 0.6 x 1.8, [.9,1) cyclist 1.8 x 0.6 x 1.7; footprints only
            # shrink, so the overlap rejection still holds
            u = Ls - 4.0
            van, ped, cyc = (u >= .7) & (u < .8), (u >= .8) & (u < .9), u >= .9
            hx, hy, hz = agents["hx"].copy(), agents["hy"].copy(), agents["hz"].copy()
            hz[van] = 1.6
            hx[ped] = 0.3; hy[ped] = 0.3; hz[ped] = 0.9
            hx[cyc] = 0.9; hy[cyc] = 0.3; hz[cyc] = 0.85
            agents["hx"] = hx; agents["hy"] = hy; agents["hz"] = hz; agents["cz"] = hz
            cls = agents["cls"].copy()
            cls[ped] = CLASS_PEDESTRIAN; cls[cyc] = CLASS_CYCLIST
            agents["cls"] = cls
    quads = np.zeros((n, Q), dtype=PRIM_DTYPE)
    if Q:
        keys = _stream_keys(cfg.seed, worlds, _STREAM_QUADS)
        kk = np.repeat(keys, Q * 4).reshape(n, Q, 4)
        cc = np.broadcast_to(np.arange(Q * 4).reshape(1, Q, 4), (n, Q, 4))
        u = _draws(kk.ravel(), cc.ravel()).reshape(n, Q, 4)
        quads["cx"] = -0.5 * E + E * u[..., 0]
        quads["cy"] = -0.5 * E + E * u[..., 1]
        quads["cz"] = 0.01
        quads["hx"] = 0.5 * (3.0 + 17.0 * u[..., 2])
        quads["hy"] = 0.075; quads["hz"] = 0.0
        psi = -math.pi + 2.0 * math.pi * u[..., 3]
        quads["cos_yaw"] = np.cos(psi); quads["sin_yaw"] = np.sin(psi)
        quads["cls"] = CLASS_MARKING
        quads["inst"] = (A + np.arange(Q, dtype=np.int32))[None, :]
    Lt = cfg.lights
    if Lt:
        # traffic lights: spheres of radius 0.2 m, 4-6 m up, uniform over the world;
        # draws continue the quad stream (counters Q*4 ..)
        keys = _stream_keys(cfg.seed, worlds, _STREAM_QUADS)
        kk = np.repeat(keys, Lt * 4).reshape(n, Lt, 4)
        cc = np.broadcast_to(Q * 4 + np.arange(Lt * 4).reshape(1, Lt, 4), (n, Lt, 4))
        u = _draws(kk.ravel(), cc.ravel()).reshape(n, Lt, 4)
        lights = np.zeros((n, Lt), dtype=PRIM_DTYPE)
        lights["cx"] = -0.5 * E + E * u[..., 0]
        lights["cy"] = -0.5 * E + E * u[..., 1]
        lights["cz"] = 4.0 + 2.0 * u[..., 2]
        lights["hx"] = 0.2; lights["hy"] = 0.2; lights["hz"] = 0.2
        lights["cos_yaw"] = 1.0
        lights["cls"] = CLASS_LIGHT
        lights["shape"] = SHAPE_SPHERE
        lights["inst"] = (A + Q + np.arange(Lt, dtype=np.int32))[None, :]
        quads = np.concatenate([quads, lights], axis=1)
    return agents, quads


def gen_lane_polylines(cfg: SceneConfig, n_lines: int, pts_per_line: int = 9, step: float = 5.0,
                       world_begin: int = 0, n_worlds: int | None = None) -> np.ndarray:
    """Lane-like polylines [Wn][n_lines][pts_per_line][2] fp32: arcs of constant curvature ~U[-0.03, 0.03] 1/m from
    a uniform start point and heading, vertices `step` metres apart (draws: the quad stream, counters 2^20 ..)."""
    n = cfg.n_worlds - world_begin if n_worlds is None else n_worlds
    worlds = np.arange(world_begin, world_begin + n)
    E = cfg.extent
    keys = _stream_keys(cfg.seed, worlds, _STREAM_QUADS)
    kk = np.repeat(keys, n_lines * 4).reshape(n, n_lines, 4)
    cc = np.broadcast_to((1 << 20) + np.arange(n_lines * 4).reshape(1, n_lines, 4), (n, n_lines, 4))
    u = _draws(kk.ravel(), cc.ravel()).reshape(n, n_lines, 4)
    x = -0.5 * E + E * u[..., 0]; y = -0.5 * E + E * u[..., 1]
    psi = -math.pi + 2.0 * math.pi * u[..., 2]
    kappa = -0.03 + 0.06 * u[..., 3]
    out = np.zeros((n, n_lines, pts_per_line, 2), dtype=np.float32)
    for i in range(pts_per_line):
        out[..., i, 0] = x; out[..., i, 1] = y
        x = x + step * np.cos(psi); y = y + step * np.sin(psi)
        psi = psi + kappa * step
    return out


def gen_dynamics(cfg: SceneConfig, world_begin: int = 0, n_worlds: int | None = None):
    """(speed[Wn][A] m/s, yaw_rate[Wn][A] rad/s) in float64 (G4)."""
    n = cfg.n_worlds - world_begin if n_worlds is None else n_worlds
    worlds = np.arange(world_begin, world_begin + n)
    A = cfg.agents
    keys = _stream_keys(cfg.seed, worlds, _STREAM_DYNAMICS)
    kk = np.repeat(keys, A * 2)
    cc = np.tile(np.arange(A * 2), n)
    u = _draws(kk, cc).reshape(n, A, 2)
    return 15.0 * u[..., 0], -0.3 + 0.6 * u[..., 1]


def gen_pitch(cfg: SceneConfig, world_begin: int = 0, n_worlds: int | None = None) -> np.ndarray:
    """Per-camera (cos p, sin p) fp32 pairs, [Wn][A][2]; (1,0) when the config has no pitch (G5)."""
    n = cfg.n_worlds - world_begin if n_worlds is None else n_worlds
    A = cfg.agents
    out = np.zeros((n, A, 2), dtype=np.float32)
    out[..., 0] = 1.0
    if cfg.pitch_deg_max > 0.0:
        worlds = np.arange(world_begin, world_begin + n)
        keys = _stream_keys(cfg.seed, worlds, _STREAM_PITCH)
        u = _draws(np.repeat(keys, A), np.tile(np.arange(A), n)).reshape(n, A)
        p = np.radians(cfg.pitch_deg_max) * (2.0 * u - 1.0)
        out[..., 0] = np.cos(p); out[..., 1] = np.sin(p)
    return out


def poses_at_frames(cfg: SceneConfig, agents: np.ndarray, speed: np.ndarray,
                    yaw_rate: np.ndarray, frames) -> dict:
    """Explicit-Euler pose advance (G4).  Returns {frame: pose[Wn][A][4] fp32}
    with pose = (cx, cy, cos yaw, sin yaw).  Frame 0 reproduces `agents` exactly."""
    frames = sorted(set(int(f) for f in frames))
    E, dt = cfg.extent, cfg.dt
    x = agents["cx"].astype(np.float64).copy()
    y = agents["cy"].astype(np.float64).copy()
    psi = np.arctan2(agents["sin_yaw"].astype(np.float64), agents["cos_yaw"].astype(np.float64))
    out = {}
    last = frames[-1] if frames else -1
    for f in range(last + 1):
        if f in frames:
            pose = np.empty(agents.shape + (4,), dtype=np.float32)
            if f == 0:
                pose[..., 0] = agents["cx"]; pose[..., 1] = agents["cy"]
                pose[..., 2] = agents["cos_yaw"]; pose[..., 3] = agents["sin_yaw"]
            else:
                pose[..., 0] = x; pose[..., 1] = y
                pose[..., 2] = np.cos(psi); pose[..., 3] = np.sin(psi)
            out[f] = pose
        x = x + speed * np.cos(psi) * dt
        y = y + speed * np.sin(psi) * dt
        psi = psi + yaw_rate * dt
        x = (x + 0.5 * E) % E - 0.5 * E
        y = (y + 0.5 * E) % E - 0.5 * E
    return out
