"""Helpers shared by the -m gpu parity tests: run the CUDA path, run the oracle, compare under the
rules of BASELINE.json north_star (ids bit-exact except pixels whose two nearest hits lie within
1e-5 m; depth within 1e-5 relative; RGB bit-exact)."""
from __future__ import annotations

import os

import numpy as np

import gp_scenes as gs

DEPTH_RTOL = 1e-5          # BASELINE.json north_star
TIE_GAP_M = 1e-5           # exclusion rule


def fov32(cfg):
    return float(np.float32(cfg.fov_rad))


def world_prims(agents, quads):
    return np.concatenate([agents, quads], axis=1) if quads is not None and quads.size else agents


def gpu_render(renderer, cfg, world_begin, n_worlds, path=0, rgb=True, H=None, W=None, fov=None, gather=None, variant=None):
    """Render a world range through the C ABI; returns numpy planes."""
    import torch
    from paper_2606_19641_b200 import gp
    H = H or cfg.H; W = W or cfg.W
    renderer.set_option(gp.GP_OPT_PATH, path)
    renderer.set_option(gp.GP_OPT_GATHER, -1 if gather is None else gather)
    renderer.set_option(gp.GP_OPT_VARIANT, -1 if variant is None else variant)
    outs = renderer.alloc_outputs(n_worlds * cfg.agents * renderer.n_cams, H, W, rgb=rgb)
    for t in outs:
        if t is not None:
            t.fill_(0x5A if t.dtype == torch.uint8 else 123456)      # poison: every element must be written
    renderer.render_batch(world_begin, n_worlds, H, W, fov if fov is not None else fov32(cfg), *outs)
    torch.cuda.synchronize()
    renderer.set_option(gp.GP_OPT_PATH, gp.GP_PATH_FAST)
    return outs


def oracle_threads():
    return max(1, min(32, (os.cpu_count() or 1)))


REPORT = {}          # label -> summed compare_views reports; written to gpurun_out/parity_report.json at session end


def record(label, rep):
    acc = REPORT.setdefault(label, {})
    for k, v in rep.items():
        acc[k] = acc.get(k, 0) + v


def compare_views(gpu_planes, view_indices, refs, label=None):
    """gpu_planes: (cls, inst, depth, rgb) torch tensors; view_indices: indices into them; refs: oracle
    dicts.  Returns a report dict; raises AssertionError on any violation of the parity rules.
    Rules (BASELINE.json north_star): ids bit-exact except pixels whose two nearest hits lie within 1e-5 m (excluded
    from the ID and colour comparison only, and counted); depth within 1e-5 relative on EVERY pixel — on an excluded
    pixel the other of the two near-equal hits may have won, so its tolerance is widened by the 1e-5 m gap."""
    cls, inst, depth, rgb = gpu_planes
    rep = {"pixels": 0, "excluded": 0, "excluded_matched": 0, "id_mismatch": 0, "depth_bad": 0,
           "rgb_mismatch": 0, "depth_bitexact": 0}
    for vi, ref in zip(view_indices, refs):
        g_cls = cls[vi].cpu().numpy(); g_inst = inst[vi].cpu().numpy(); g_dep = depth[vi].cpu().numpy()
        excl = (ref["t2"].astype(np.float64) - ref["depth"].astype(np.float64)) <= TIE_GAP_M
        excl &= ref["win"] != -2
        keep = ~excl
        ids_ok = (g_cls == ref["cls"]) & (g_inst == ref["inst"])
        rep["pixels"] += ids_ok.size
        rep["excluded"] += int(excl.sum())
        rep["excluded_matched"] += int((ids_ok & excl).sum())
        rep["id_mismatch"] += int((~ids_ok & keep).sum())
        d_err = np.abs(g_dep.astype(np.float64) - ref["depth"])
        d_ok = d_err <= DEPTH_RTOL * np.abs(ref["depth"]) + np.where(excl, TIE_GAP_M, 0.0)
        rep["depth_bad"] += int((~d_ok).sum())
        rep["depth_bitexact"] += int((g_dep == ref["depth"]).sum())
        if rgb is not None and ref.get("rgb") is not None:
            g_rgb = rgb[vi].cpu().numpy()
            rep["rgb_mismatch"] += int(((g_rgb != ref["rgb"]).any(axis=0) & keep).sum())
    rep["views"] = len(view_indices)
    assert rep["id_mismatch"] == 0, rep
    assert rep["depth_bad"] == 0, rep
    assert rep["rgb_mismatch"] == 0, rep
    if label:
        record(label, rep)
    return rep


def oracle_refs(prims, views, H, W, par, pitch=None, rgb=True, rig=None):
    """views: (world, agent) or, with rig = [C][>=3] (cos d, sin d, mount), (world, agent, camera)."""
    import oracle
    return oracle.render_views(prims, views, H, W, par, pitch_cs=pitch, rgb=rgb, threads=oracle_threads(), rig=rig)


def planes_equal(a, b):
    """Exact equality of two sets of device planes (fast path vs brute force)."""
    import torch
    bad = {}
    for name, x, y in zip(("cls", "inst", "depth", "rgb"), a, b):
        if x is None:
            continue
        if x.dtype == torch.float32:
            eq = torch.equal(x.view(torch.int32), y.view(torch.int32))
        else:
            eq = torch.equal(x, y)
        if not eq:
            diff = (x != y)
            bad[name] = int(diff.sum().item())
    return bad
