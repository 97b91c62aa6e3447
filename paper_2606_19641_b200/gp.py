"""Thin ctypes binding of libgp.so (include/gp.h).  Argument marshalling only.

torch is used for device memory and the current stream; nothing here computes.  If libgp.so is
missing (not built) importing the library raises: there is no fallback path.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgp.so")

GP_OK, GP_ERR_ARG, GP_ERR_ALIGN, GP_ERR_STATE, GP_ERR_RANGE, GP_ERR_CUDA, GP_ERR_ARCH, GP_ERR_NOMEM = \
    0, -1, -2, -3, -4, -5, -6, -7
GP_ERR_LIMIT = -8
GP_STATIC_MAX_VIEWS, GP_STATIC_MAX_PRIMS, GP_STATIC_MAX_ENTRIES = 4096, 32768, 131072
GP_OPT_PATH, GP_OPT_STATS, GP_OPT_TIMING, GP_OPT_STAGE_CAP, GP_OPT_STRIP_PX, GP_OPT_GATHER, GP_OPT_SPHERES = 1, 2, 3, 4, 5, 6, 7
GP_OPT_VARIANT, GP_OPT_TILE_PX, GP_OPT_PIPELINE, GP_OPT_LIST_CAP = 8, 9, 10, 11
GP_VARIANT_RAY, GP_VARIANT_RASTER = 0, 1
GP_KERNEL_UPDATE, GP_KERNEL_CULL, GP_KERNEL_RENDER, GP_KERNEL_BRUTE, GP_KERNEL_DYNAMICS, GP_KERNEL_OBSERVE = 0, 1, 2, 3, 4, 5
GP_PATH_FAST, GP_PATH_BRUTE = 0, 1
GP_PROBE_STORE, GP_PROBE_FMA, GP_PROBE_RCP, GP_PROBE_STORE_VIEW = 0, 1, 2, 3

EXPORTS = ("gp_create", "gp_destroy", "gp_set_option", "gp_scene_upload", "gp_agents_update",
           "gp_cameras_set", "gp_render_batch", "gp_render_batch_host", "gp_stats", "gp_kernel_time",
           "gp_launch_count", "gp_camera_rig_set", "gp_statics_from_polylines", "gp_statics_update",
           "gp_dynamics_step", "gp_observe_vec", "gp_probe", "gp_reserve", "gp_render_static", "gp_error_string")


class SceneDesc(ctypes.Structure):
    _fields_ = [("n_worlds", ctypes.c_int32), ("agents_per_world", ctypes.c_int32),
                ("quads_per_world", ctypes.c_int32), ("cam_height", ctypes.c_float),
                ("t_max", ctypes.c_float), ("light", ctypes.c_float * 3), ("ambient", ctypes.c_float),
                ("palette", (ctypes.c_uint8 * 3) * 8)]


class DynParams(ctypes.Structure):
    _fields_ = [("dt", ctypes.c_float), ("a_lon_max", ctypes.c_float), ("a_lat_max", ctypes.c_float),
                ("v_max", ctypes.c_float), ("steer_max", ctypes.c_float), ("steer_rate_max", ctypes.c_float),
                ("v_eps", ctypes.c_float), ("extent", ctypes.c_float)]


class Camera(ctypes.Structure):
    _fields_ = [("cos_yaw_off", ctypes.c_float), ("sin_yaw_off", ctypes.c_float), ("mount", ctypes.c_float),
                ("pad", ctypes.c_float)]


DEFAULT_PALETTE = ((135, 206, 235), (90, 90, 90), (240, 240, 240), (40, 80, 220),
                   (220, 60, 60), (240, 160, 40), (150, 110, 70), (250, 240, 80))


class GpError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("gp error %d: %s" % (code, text))
        self.code = code


_lib = None


def lib():
    """Load libgp.so (raises OSError if it has not been built; see paper_2606_19641_b200/build.py)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OSError("libgp.so is not built (run `python -m paper_2606_19641_b200.build`); "
                          "there is no fallback renderer")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
        L.gp_create.argtypes = [ctypes.POINTER(vp), ci]
        L.gp_destroy.argtypes = [vp]
        L.gp_set_option.argtypes = [vp, ci, ci]
        L.gp_scene_upload.argtypes = [vp, ctypes.POINTER(SceneDesc), vp, vp, vp]
        L.gp_agents_update.argtypes = [vp, vp, vp]
        L.gp_cameras_set.argtypes = [vp, vp, vp]
        L.gp_render_batch.argtypes = [vp, ci, ci, ci, ci, ci, cf, vp, vp, vp, vp, vp]
        L.gp_render_batch_host.argtypes = [vp, vp, ci, ci, ci, ci, ci, cf, vp, vp, vp, vp, vp]
        L.gp_stats.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]
        L.gp_kernel_time.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_uint64)]
        L.gp_launch_count.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64)]
        L.gp_camera_rig_set.argtypes = [vp, ci, vp]
        L.gp_statics_update.argtypes = [vp, vp, ci, ci, vp]
        L.gp_statics_from_polylines.argtypes = [vp, vp, ci, ci, cf, cf, ci, ci, vp]
        L.gp_dynamics_step.argtypes = [vp, ctypes.POINTER(DynParams), vp, vp, vp, vp]
        L.gp_observe_vec.argtypes = [vp, vp, ci, ci, cf, vp, vp, vp, vp, vp]
        L.gp_probe.argtypes = [vp, ci, ctypes.c_size_t, ci, vp, vp, vp, vp, vp, ctypes.POINTER(ctypes.c_double),
                               ctypes.POINTER(ctypes.c_double)]
        L.gp_reserve.argtypes = [vp, ci, ci, ci]
        L.gp_render_static.argtypes = [ci, ctypes.POINTER(SceneDesc), vp, vp, ci, ci, cf, vp, vp, vp, vp, vp]
        L.gp_error_string.argtypes = [ci]
        L.gp_error_string.restype = ctypes.c_char_p
        for name in EXPORTS[:-1]:
            getattr(L, name).restype = ci
        _lib = L
    return _lib


def _check(rc):
    if rc != GP_OK:
        raise GpError(rc, lib().gp_error_string(rc).decode())


def _stream(device):
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _dptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def render_static(d_prims, agents_per_world, H, W, fov_rad, d_class, d_instance, d_depth, d_rgb=None, d_pitch_cs=None,
                  cam_height=1.6, t_max=100.0, light=(0.48, 0.36, 0.8), ambient=0.25, palette=DEFAULT_PALETTE, device=0):
    """gp_render_static: render every view of a scene that already sits in device memory without the library allocating
    anything - for processes in which the training framework holds all of HBM, or whose loop cannot take the stall of a
    cudaMalloc.  No Renderer is needed.  The intermediates live in a fixed 9.1 MiB array inside libgp.so, which limits the
    scene (GP_STATIC_MAX_VIEWS / _PRIMS / _ENTRIES; GpError with code GP_ERR_LIMIT beyond them) and is shared by all calls
    on a device: keep them on one stream, or order them, so that they never overlap on the GPU.  The first call on a device
    does a one-off set-up; make it before any stream capture.

    d_prims: CUDA uint8 tensor [Wn][P][48] of gp_prim records, the agents first in each world; d_pitch_cs: CUDA float32
    [Wn][A][2] or None (pitch 0); outputs as for Renderer.render_batch with one front camera per agent."""
    assert d_prims.dim() == 3 and d_prims.shape[2] == 48 and d_prims.is_contiguous()
    d = SceneDesc()
    d.n_worlds, d.agents_per_world = int(d_prims.shape[0]), int(agents_per_world)
    d.quads_per_world = int(d_prims.shape[1]) - int(agents_per_world)
    d.cam_height, d.t_max, d.ambient = cam_height, t_max, ambient
    for i in range(3):
        d.light[i] = light[i]
    for c in range(min(8, len(palette))):
        for ch in range(3):
            d.palette[c][ch] = int(palette[c][ch])
    _check(lib().gp_render_static(int(device), ctypes.byref(d), _dptr(d_prims), _dptr(d_pitch_cs), int(H), int(W),
                                  float(fov_rad), _dptr(d_class), _dptr(d_instance), _dptr(d_depth), _dptr(d_rgb),
                                  _stream(device)))


class Renderer:
    """One gp_ctx.  Methods mirror the C ABI one to one."""

    def __init__(self, device: int = 0):
        self._h = ctypes.c_void_p()
        _check(lib().gp_create(ctypes.byref(self._h), int(device)))
        self.device = int(device)
        self.desc = None
        self.n_cams = 1

    def close(self):
        if getattr(self, "_h", None):
            lib().gp_destroy(self._h)
            self._h = None

    __del__ = close

    def set_option(self, key: int, value: int):
        _check(lib().gp_set_option(self._h, key, value))

    def scene_upload(self, agents: np.ndarray, quads: np.ndarray | None, cam_height=1.6, t_max=100.0,
                     light=(0.48, 0.36, 0.8), ambient=0.25, palette=DEFAULT_PALETTE):
        """agents [Wn][A], quads [Wn][Q] (or None): host arrays of 48-byte gp_prim records."""
        agents = np.ascontiguousarray(agents)
        assert agents.ndim == 2 and agents.dtype.itemsize == 48
        Wn, A = agents.shape
        Q = 0
        if quads is not None and quads.size:
            quads = np.ascontiguousarray(quads)
            assert quads.ndim == 2 and quads.shape[0] == Wn and quads.dtype.itemsize == 48
            Q = quads.shape[1]
        d = SceneDesc()
        d.n_worlds, d.agents_per_world, d.quads_per_world = Wn, A, Q
        d.cam_height, d.t_max, d.ambient = cam_height, t_max, ambient
        for i in range(3):
            d.light[i] = light[i]
        for c in range(min(8, len(palette))):
            for ch in range(3):
                d.palette[c][ch] = int(palette[c][ch])
        _check(lib().gp_scene_upload(self._h, ctypes.byref(d), agents.ctypes.data,
                                     quads.ctypes.data if Q else None, _stream(self.device)))
        self.desc = d

    def agents_update(self, d_pose):
        """d_pose: CUDA float32 tensor [Wn][A][4] = (cx, cy, cos yaw, sin yaw)."""
        _check(lib().gp_agents_update(self._h, _dptr(d_pose), _stream(self.device)))

    def cameras_set(self, d_pitch_cs=None):
        """d_pitch_cs: CUDA float32 tensor [Wn][A][2] = (cos p, sin p), or None for pitch 0."""
        _check(lib().gp_cameras_set(self._h, _dptr(d_pitch_cs), _stream(self.device)))

    def statics_update(self, d_prims, q_begin=0):
        """d_prims: CUDA uint8 tensor [Wn][n][48] of gp_prim records replacing static slots q_begin .. of every world."""
        assert d_prims.dim() == 3 and d_prims.shape[2] == 48 and d_prims.is_contiguous()
        _check(lib().gp_statics_update(self._h, _dptr(d_prims), int(d_prims.shape[1]), int(q_begin), _stream(self.device)))

    def statics_from_polylines(self, d_points, half_width=0.075, z=0.01, cls=2, q_begin=0):
        """d_points: CUDA float32 tensor [Wn][n_lines][pts_per_line][2]; one flat quad per segment replaces the
        static primitives q_begin .. of every world."""
        assert d_points.dim() == 4 and d_points.shape[3] == 2 and d_points.is_contiguous()
        _check(lib().gp_statics_from_polylines(self._h, _dptr(d_points), int(d_points.shape[1]), int(d_points.shape[2]),
                                               float(half_width), float(z), int(cls), int(q_begin), _stream(self.device)))

    def dynamics_step(self, params, d_action, d_state, d_pose):
        """params: dict or DynParams; d_action CUDA int32 [Wn][A]; d_state CUDA float32 [Wn][A][8] and d_pose CUDA
        float32 [Wn][A][4], both updated in place; the scene's agent records follow the new poses."""
        if not isinstance(params, DynParams):
            q = DynParams()
            for k, v in dict(params).items():
                setattr(q, k, float(v))
            params = q
        _check(lib().gp_dynamics_step(self._h, ctypes.byref(params), _dptr(d_action), _dptr(d_state), _dptr(d_pose),
                                      _stream(self.device)))

    def observe_vec(self, d_state, K, M, radius, d_agent_idx, d_agent_feat, d_road_idx, d_road_feat):
        """O_vec into caller-owned CUDA tensors: int32 [Wn][A][K], float32 [Wn][A][K][8], int32 [Wn][A][M], float32 [Wn][A][M][8]."""
        _check(lib().gp_observe_vec(self._h, _dptr(d_state), int(K), int(M), float(radius), _dptr(d_agent_idx),
                                    _dptr(d_agent_feat), _dptr(d_road_idx), _dptr(d_road_feat), _stream(self.device)))

    def probe(self, kind, n_pixels=0, iters=10, planes=(None, None, None, None)):
        """(best, median) rate of a calibration probe: GB/s for GP_PROBE_STORE, TFLOP/s for GP_PROBE_FMA."""
        best, med = ctypes.c_double(), ctypes.c_double()
        _check(lib().gp_probe(self._h, int(kind), int(n_pixels), int(iters), *[_dptr(t) for t in planes],
                              _stream(self.device), ctypes.byref(best), ctypes.byref(med)))
        return best.value, med.value

    def camera_rig_set(self, rig):
        """rig: array-like [C][>=3] = (cos yaw offset, sin yaw offset, mount) per camera of every agent."""
        rig = np.asarray(rig, dtype=np.float32)
        arr = (Camera * len(rig))()
        for i, r in enumerate(rig):
            arr[i].cos_yaw_off, arr[i].sin_yaw_off, arr[i].mount, arr[i].pad = float(r[0]), float(r[1]), float(r[2]), 0.0
        _check(lib().gp_camera_rig_set(self._h, len(rig), ctypes.cast(arr, ctypes.c_void_p)))
        self.n_cams = len(rig)

    def render_batch(self, world_begin, n_worlds, H, W, fov_rad, d_class, d_instance, d_depth, d_rgb=None):
        """Outputs: CUDA tensors uint8 [n][H][W], int32 [n][H][W], float32 [n][H][W], uint8 [n][3][H][W],
        n = n_worlds * agents * cameras."""
        _check(lib().gp_render_batch(self._h, int(world_begin), int(n_worlds), int(self.desc.agents_per_world),
                                     int(H), int(W), float(fov_rad), _dptr(d_class), _dptr(d_instance),
                                     _dptr(d_depth), _dptr(d_rgb), _stream(self.device)))

    def render_batch_host(self, h_pose, world_begin, n_worlds, H, W, fov_rad, h_class, h_instance, h_depth,
                          h_rgb=None):
        """Host-buffer variant (torch CPU tensors, ideally pinned, or numpy arrays)."""
        def hp(x):
            if x is None:
                return None
            return ctypes.c_void_p(x.ctypes.data if isinstance(x, np.ndarray) else x.data_ptr())
        _check(lib().gp_render_batch_host(self._h, hp(h_pose), int(world_begin), int(n_worlds),
                                          int(self.desc.agents_per_world), int(H), int(W), float(fov_rad),
                                          hp(h_class), hp(h_instance), hp(h_depth), hp(h_rgb), _stream(self.device)))

    def stats(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        _check(lib().gp_stats(self._h, ctypes.byref(a), ctypes.byref(b)))
        return {"executed_tests": a.value, "listed_pairs": b.value}

    def kernel_time(self, kernel: int):
        """(total_ms, launches) of one kernel since the last call (needs GP_OPT_TIMING = 1)."""
        ms, n = ctypes.c_double(), ctypes.c_uint64()
        _check(lib().gp_kernel_time(self._h, kernel, ctypes.byref(ms), ctypes.byref(n)))
        return ms.value, n.value

    def launch_count(self) -> int:
        a = ctypes.c_uint64()
        _check(lib().gp_launch_count(self._h, ctypes.byref(a)))
        return a.value

    def reserve(self, n_worlds, H, W):
        """Size the per-view scratch so that render_batch(..., n_worlds' <= n_worlds, H, W, ...) allocates nothing."""
        _check(lib().gp_reserve(self._h, int(n_worlds), int(H), int(W)))

    def alloc_outputs(self, n_views, H, W, rgb=True):
        import torch
        dev = torch.device("cuda", self.device)
        return (torch.empty((n_views, H, W), dtype=torch.uint8, device=dev),
                torch.empty((n_views, H, W), dtype=torch.int32, device=dev),
                torch.empty((n_views, H, W), dtype=torch.float32, device=dev),
                torch.empty((n_views, 3, H, W), dtype=torch.uint8, device=dev) if rgb else None)
