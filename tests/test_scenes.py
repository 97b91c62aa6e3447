"""The seeded input generator (gp_scenes): determinism, ranges, structure.  CPU only."""
import numpy as np

import gp_scenes as gs
from gp_scenes import generator as g


def test_splitmix64_reference_vector():
    # first outputs of splitmix64 seeded with 0 (Steele/Lea/Flood reference sequence)
    with np.errstate(over="ignore"):
        x1 = g._mix64(np.array([0x9E3779B97F4A7C15], dtype=np.uint64))[0]
        x2 = g._mix64(np.array([0x9E3779B97F4A7C15], dtype=np.uint64) * np.uint64(2))[0]
    assert int(x1) == 0xE220A8397B1DCDAF
    assert int(x2) == 0x6E789E6AA1B965F4


def test_draws_are_uniform_and_deterministic():
    u = gs.splitmix64_stream(3, 5, 1, 20000)
    assert (u >= 0).all() and (u < 1).all()
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1 / 12) < 0.005
    assert (u == gs.splitmix64_stream(3, 5, 1, 20000)).all()
    assert (u != gs.splitmix64_stream(3, 6, 1, 20000)).any()


def test_record_layout():
    assert gs.PRIM_DTYPE.itemsize == 48
    assert [gs.PRIM_DTYPE.fields[n][1] for n in ("cx", "hx", "cos_yaw", "cls", "inst")] == [0, 12, 24, 32, 36]


def test_tiny_matches_baseline_config():
    cfg = gs.config("tiny")
    a, q = gs.gen_world_prims(cfg)
    assert a.shape == (1, 4) and q.shape == (1, 12) and cfg.seed == 0 and (cfg.H, cfg.W) == (32, 32)
    assert ((2 * a["hx"] >= 4) & (2 * a["hx"] <= 5) & (2 * a["hy"] >= 1.8) & (2 * a["hy"] <= 2.1)).all()
    assert (a["cz"] == 0.75).all() and (a["hz"] == 0.75).all() and (a["cls"] == 3).all()
    assert (np.abs(a["cx"]) <= 30).all() and (np.abs(a["cy"]) <= 30).all()
    assert (q["hy"] == np.float32(0.075)).all() and (q["hz"] == 0).all() and (q["cz"] == np.float32(0.01)).all()
    assert ((2 * q["hx"] >= 3) & (2 * q["hx"] <= 20)).all() and (q["cls"] == 2).all()
    assert (a["inst"][0] == np.arange(4)).all() and (q["inst"][0] == 4 + np.arange(12)).all()
    for p in (a, q):
        assert np.allclose(p["cos_yaw"].astype(float) ** 2 + p["sin_yaw"].astype(float) ** 2, 1, atol=1e-6)


def test_vehicles_do_not_overlap_and_worlds_are_independent_of_range():
    cfg = gs.config("dense", n_worlds=6)
    a, q = gs.gen_world_prims(cfg)
    x, y = a["cx"].astype(float), a["cy"].astype(float)
    r = 0.5 * np.hypot(2 * a["hx"].astype(float), 2 * a["hy"].astype(float))
    d = np.hypot(x[:, :, None] - x[:, None, :], y[:, :, None] - y[:, None, :])
    rr = r[:, :, None] + r[:, None, :]
    iu = np.triu_indices(cfg.agents, 1)
    assert (d[:, iu[0], iu[1]] >= rr[:, iu[0], iu[1]] - 1e-4).all()
    a2, q2 = gs.gen_world_prims(cfg, 3, 2)
    assert (a2 == a[3:5]).all() and (q2 == q[3:5]).all()
    assert (a[0] != a[1]).any()


def test_pitch_and_dynamics():
    cfg = gs.config("dense", n_worlds=3)
    p = gs.gen_pitch(cfg)
    ang = np.degrees(np.arctan2(p[..., 1].astype(float), p[..., 0].astype(float)))
    assert p.shape == (3, 128, 2) and (np.abs(ang) <= 5).all() and ang.std() > 1
    assert (gs.gen_pitch(gs.config("paper", n_worlds=2)) == np.array([1, 0], np.float32)).all()
    sp, yr = gs.gen_dynamics(gs.config("paper", n_worlds=2))
    assert ((sp >= 0) & (sp < 15)).all() and ((yr >= -0.3) & (yr < 0.3)).all()


def test_pose_advance():
    cfg = gs.config("paper", n_worlds=2)
    a, _ = gs.gen_world_prims(cfg)
    sp, yr = gs.gen_dynamics(cfg)
    poses = gs.poses_at_frames(cfg, a, sp, yr, [0, 1, 10, 999])
    assert (poses[0][..., 0] == a["cx"]).all() and (poses[0][..., 3] == a["sin_yaw"]).all()
    E = cfg.extent
    wrap = lambda d: (d.astype(float) + E / 2) % E - E / 2
    step = np.hypot(wrap(poses[1][..., 0] - poses[0][..., 0]), wrap(poses[1][..., 1] - poses[0][..., 1]))
    assert np.allclose(step, sp * cfg.dt, atol=1e-4)
    for f in (10, 999):
        assert (np.abs(poses[f][..., :2]) <= cfg.extent / 2).all()
        assert np.allclose(np.hypot(poses[f][..., 2], poses[f][..., 3]), 1, atol=1e-6)
    dpsi = np.arctan2(poses[10][..., 3], poses[10][..., 2]) - np.arctan2(poses[0][..., 3], poses[0][..., 2])
    dpsi = (dpsi + np.pi) % (2 * np.pi) - np.pi
    assert np.allclose(dpsi, 10 * cfg.dt * yr, atol=1e-5)
