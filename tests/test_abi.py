"""The C-ABI library loads and exports every symbol include/gp.h declares.  CPU only (no compute)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libgp():
    from paper_2606_19641_b200 import build, gp
    build.build()
    return gp.lib()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gp_[a-z_]+)\s*\(", text)))


def test_header_declares_the_calls_of_the_scope_table():
    names = declared_functions()
    for need in ("gp_create", "gp_destroy", "gp_scene_upload", "gp_agents_update", "gp_cameras_set",
                 "gp_render_batch", "gp_stats", "gp_error_string"):
        assert need in names


def test_library_exports_every_declared_symbol(libgp):
    from paper_2606_19641_b200 import gp
    names = declared_functions()
    assert sorted(gp.EXPORTS) == names
    for n in names:
        assert getattr(libgp, n) is not None


def test_error_strings(libgp):
    from paper_2606_19641_b200 import gp
    assert libgp.gp_error_string(0) == b"ok"
    for code in range(-7, 0):
        assert len(libgp.gp_error_string(code)) > 3
    assert b"no fallback" in libgp.gp_error_string(gp.GP_ERR_ARCH)


def test_struct_layouts_match_header():
    from paper_2606_19641_b200 import gp
    import gp_scenes as gs
    assert ctypes.sizeof(gp.SceneDesc) == 3 * 4 + 2 * 4 + 3 * 4 + 4 + 24      # palette[8][3]
    assert ctypes.sizeof(gp.Camera) == 16
    import oracle
    assert tuple(map(tuple, gs.DEFAULT_PALETTE.tolist())) == tuple(gp.DEFAULT_PALETTE) == tuple(oracle.PALETTE)
    assert gs.PRIM_DTYPE.itemsize == 48


def test_null_arguments_are_rejected_without_a_gpu(libgp):
    from paper_2606_19641_b200 import gp
    assert libgp.gp_create(None, 0) == gp.GP_ERR_ARG
    assert libgp.gp_destroy(None) == gp.GP_ERR_ARG
    assert libgp.gp_render_batch(None, 0, 1, 1, 8, 8, 1.0, None, None, None, None, None) == gp.GP_ERR_ARG
    assert libgp.gp_stats(None, None, None) == gp.GP_ERR_ARG
    assert libgp.gp_camera_rig_set(None, 1, None) == gp.GP_ERR_ARG
    assert libgp.gp_statics_update(None, None, 1, 0, None) == gp.GP_ERR_ARG
    assert libgp.gp_statics_from_polylines(None, None, 1, 2, 0.1, 0.0, 2, 0, None) == gp.GP_ERR_ARG


def test_no_cpu_fallback_create_fails_loudly_without_b200(libgp):
    import torch
    from paper_2606_19641_b200 import gp, Renderer, GpError
    if torch.cuda.is_available():
        pytest.skip("GPU present: covered by the gpu tests")
    with pytest.raises(GpError) as ei:
        Renderer(0)
    assert ei.value.code in (gp.GP_ERR_CUDA, gp.GP_ERR_ARG, gp.GP_ERR_ARCH)


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_19641_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                for pat in (r"^\s*(import|from)\s+oracle", r"#include\s+[\"<].*oracle", r"gp_oracle", r"orc_"):
                    assert not re.search(pat, src, flags=re.M), (f, pat)
