"""gp_render_static: the render step for callers that cannot let the library allocate device memory.

Why it exists: every other render call goes through a gp_ctx, whose scene copy and per-view lists come from cudaMalloc.
A training process whose framework has already taken all of HBM for its own pool, an actor loop that cannot take the
device-wide stall of an allocation, or a deployment that budgets device memory up front cannot use that.  For them
gp_render_static reads the scene from the caller's device memory, writes the caller's planes, and keeps what lies in
between (shading table, view headers, per-view lists) in one fixed 9.1 MiB array that is part of libgp.so.  That array
is shared by all calls on a device and is never cleared between them, hence the shape of the test below: calls back to
back, a large scene followed by a small one and the large one again, each compared with the ordinary path.

This file sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure here
should not hide the rest of the suite.  It must pass alone in a fresh process and after the other tests alike, so it
assumes nothing about what ran before on the device.
"""
import ctypes

import numpy as np
import pytest

import gp_scenes as gs
from parity_util import DEPTH_RTOL, fov32, world_prims


def _desc(gp, n_worlds, agents, quads):
    d = gp.SceneDesc()
    d.n_worlds, d.agents_per_world, d.quads_per_world = n_worlds, agents, quads
    d.cam_height, d.t_max, d.ambient = 1.6, 100.0, 0.25
    d.light[0], d.light[1], d.light[2] = 0.48, 0.36, 0.8
    return d


def test_static_scratch_limits_are_refused_before_the_device_is_touched():
    """Scenes beyond the fixed array are turned away with GP_ERR_LIMIT and a text that names the limits.  The size check
    comes before any CUDA call, so this runs without a GPU (the pointers are never dereferenced)."""
    from paper_2606_19641_b200 import build, gp
    build.build()
    L = gp.lib()
    fake = ctypes.c_void_p(0x1000)          # aligned, never used
    call = lambda d: L.gp_render_static(0, ctypes.byref(d), fake, None, 64, 64, 1.5, fake, fake, fake, None, None)
    assert call(_desc(gp, gp.GP_STATIC_MAX_VIEWS + 1, 1, 0)) == gp.GP_ERR_LIMIT                  # too many views
    assert call(_desc(gp, 1, 1, gp.GP_STATIC_MAX_PRIMS)) == gp.GP_ERR_LIMIT                      # too many records
    assert call(_desc(gp, 8, 64, 200)) == gp.GP_ERR_LIMIT                                        # 512 views x 264 list slots
    assert b"GP_STATIC_MAX" in L.gp_error_string(gp.GP_ERR_LIMIT)
    assert call(_desc(gp, 0, 1, 0)) == gp.GP_ERR_ARG
    assert L.gp_render_static(0, None, fake, None, 64, 64, 1.5, fake, fake, fake, None, None) == gp.GP_ERR_ARG
    d = _desc(gp, 1, 4, 12)
    assert L.gp_render_static(0, ctypes.byref(d), fake, None, 63, 63, 1.5, fake, fake, fake, None, None) == gp.GP_ERR_ARG
    assert L.gp_render_static(0, ctypes.byref(d), ctypes.c_void_p(0x1004), None, 64, 64, 1.5, fake, fake, fake, None,
                              None) == gp.GP_ERR_ALIGN


def _reference(torch, cfg, agents, quads, pitch):
    """The existing path: a context, its own device copy of the scene, gp_render_batch."""
    from paper_2606_19641_b200 import Renderer
    r = Renderer(0)
    r.scene_upload(agents, quads, cam_height=cfg.cam_height, t_max=cfg.t_max)
    if pitch is not None:
        r.cameras_set(torch.from_numpy(pitch).cuda())
    out = r.alloc_outputs(cfg.views, cfg.H, cfg.W)
    r.render_batch(0, cfg.n_worlds, cfg.H, cfg.W, fov32(cfg), *out)
    torch.cuda.synchronize()
    r.close()
    return out


def _poisoned_outputs(torch, cfg):
    dev = torch.device("cuda", 0)
    n, H, W = cfg.views, cfg.H, cfg.W
    return (torch.full((n, H, W), 0x5A, dtype=torch.uint8, device=dev),
            torch.full((n, H, W), 123456, dtype=torch.int32, device=dev),
            torch.full((n, H, W), 123456.0, dtype=torch.float32, device=dev),
            torch.full((n, 3, H, W), 0x5A, dtype=torch.uint8, device=dev))


def _same(torch, want, got, what):
    """The tolerance of the parity suite: ids and colour bit for bit, depth within 1e-5 relative (sky exactly 0)."""
    assert torch.equal(want[0], got[0]), what + ": class plane differs"
    assert torch.equal(want[1], got[1]), what + ": instance plane differs"
    assert torch.equal(want[3], got[3]), what + ": rgb planes differ"
    dw, dg = want[2].double(), got[2].double()
    assert bool(((dw - dg).abs() <= DEPTH_RTOL * dw.abs()).all()), what + ": depth beyond 1e-5 relative"


@pytest.mark.gpu
def test_render_static_matches_the_context_path_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs a GPU"
    from paper_2606_19641_b200 import gp

    big = gs.config("small").replace(n_worlds=8, lights=3, pitch_deg_max=5.0)      # 256 views, 64 x 64, boxes + quads + spheres
    tiny = gs.config("tiny")                                                        # 4 views, 32 x 32, pitch 0
    scenes = {}
    for cfg in (big, tiny):
        agents, quads = gs.gen_world_prims(cfg)
        pitch = gs.gen_pitch(cfg) if cfg.pitch_deg_max > 0 else None
        prims = np.ascontiguousarray(world_prims(agents, quads))
        d_prims = torch.from_numpy(prims.view(np.uint8).reshape(cfg.n_worlds, prims.shape[1], 48)).cuda()
        d_pitch = torch.from_numpy(pitch).cuda() if pitch is not None else None
        scenes[cfg.name] = (cfg, d_prims, d_pitch, _reference(torch, cfg, agents, quads, pitch))

    def call(name):
        cfg, d_prims, d_pitch, _ = scenes[name]
        out = _poisoned_outputs(torch, cfg)
        gp.render_static(d_prims, cfg.agents, cfg.H, cfg.W, fov32(cfg), *out, d_pitch_cs=d_pitch,
                         cam_height=cfg.cam_height, t_max=cfg.t_max)
        return out

    first = call(big.name)                   # also the one-off set-up on this device
    torch.cuda.synchronize()
    _same(torch, scenes[big.name][3], first, "first call")

    # back to back on one stream, no synchronisation in between: the small scene runs in the array the large one just
    # filled, then the large one again over the small one's leftovers; the allocator must not move meanwhile
    outs_small = _poisoned_outputs(torch, tiny)
    outs_big = _poisoned_outputs(torch, big)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for name, out in ((tiny.name, outs_small), (big.name, outs_big)):
        cfg, d_prims, d_pitch, _ = scenes[name]
        gp.render_static(d_prims, cfg.agents, cfg.H, cfg.W, fov32(cfg), *out, d_pitch_cs=d_pitch,
                         cam_height=cfg.cam_height, t_max=cfg.t_max)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "gp_render_static changed the device memory in use by %d bytes" % (free0 - free1)
    _same(torch, scenes[tiny.name][3], outs_small, "second call (small scene after a large one)")
    _same(torch, scenes[big.name][3], outs_big, "third call (large scene after a small one)")

    # a scene over the limit is refused through the binding with the dedicated code
    cfg, d_prims, d_pitch, _ = scenes[big.name]
    with pytest.raises(gp.GpError) as ei:
        gp.render_static(d_prims.repeat(4, 1, 1), cfg.agents, cfg.H, cfg.W, fov32(cfg), *outs_big)   # 1024 views x 155 slots
    assert ei.value.code == gp.GP_ERR_LIMIT
