"""Pins for oracle/points.py.  CPU only.
BJ north_star: "pure forward translation must project to the principal point"."""
import math

import numpy as np
import pytest

from oracle import points as op

K = dict(fx=200.0, fy=210.0, cx=112.0, cy=96.0)


def _rot(axis, a):
    c, s = math.cos(a), math.sin(a)
    m = {0: [[1, 0, 0], [0, c, -s], [0, s, c]], 1: [[c, 0, s], [0, 1, 0], [-s, 0, c]],
         2: [[c, -s, 0], [s, c, 0], [0, 0, 1]]}[axis]
    return np.array(m, dtype=np.float64)


def _w2c(r_c2w, pos):
    m = np.eye(4)
    m[:3, :3] = r_c2w.T
    m[:3, 3] = -r_c2w.T @ pos
    return m


def _frames(poses, **kw):
    args = dict(width=224, height=192, n_points=1, sigma=20.0)
    args.update(K)
    args.update(kw)
    return op.motion_points(poses, **args)


def test_forward_motion_hits_principal_point_exactly():
    # R = I, z_t quadratic (accelerating straight ahead): a_c || optical axis
    poses = [_w2c(np.eye(3), np.array([0.0, 0.0, 0.25 * t * t])) for t in range(6)]
    fr = _frames(poses)
    assert fr[0]["focus_index"] == -1 and fr[1]["focus_index"] == -1       # t < 2: no point
    assert math.isnan(fr[0]["focus_uv"][0])
    for f in fr[2:]:
        assert f["focus_uv"] == (np.float32(112.0), np.float32(96.0))
        assert f["focus_index"] == 96 * 224 + 112
    # velocity mode with constant forward speed
    poses = [_w2c(np.eye(3), np.array([0.0, 0.0, 0.5 * t])) for t in range(5)]
    fr = _frames(poses, vec=op.VELOCITY)
    assert fr[0]["focus_index"] == -1
    assert all(f["focus_index"] == 96 * 224 + 112 for f in fr[1:])
    # constant velocity has zero acceleration: no point in ACCEL mode (reading C1)
    fr = _frames(poses, vec=op.ACCEL)
    assert all(f["focus_index"] == -1 and not f["points"] for f in fr)


def test_known_directions():
    for d, exp_uv in [((1.0, 0.0, 1.0), (112.0 + 200.0, 96.0)), ((0.0, 1.0, 1.0), (112.0, 96.0 + 210.0)),
                      ((-0.5, 0.25, 1.0), (12.0, 148.5)), ((0.5, 0.0, -1.0), (12.0, 96.0))]:
        d = np.array(d)
        poses = [_w2c(np.eye(3), 0.125 * d * t * t) for t in range(4)]
        f = _frames(poses)[3]
        assert f["focus_uv"] == (np.float32(exp_uv[0]), np.float32(exp_uv[1]))
    # half-up rounding (C8) and off-image -> -1 (C9)
    poses = [_w2c(np.eye(3), 0.125 * np.array([-0.5, 0.25, 1.0]) * t * t) for t in range(4)]
    assert _frames(poses)[3]["focus_index"] == 149 * 224 + 12
    poses = [_w2c(np.eye(3), 0.125 * np.array([1.0, 0.0, 1.0]) * t * t) for t in range(4)]
    f = _frames(poses)[3]
    assert f["focus_index"] == -1 and len(f["points"]) == 1


def test_eq1_matches_general_inverse():
    rng = np.random.default_rng(1)
    for _ in range(20):
        a = rng.normal(0, 1, 3)
        r = _rot(1, a[1]) @ _rot(0, a[0]) @ _rot(2, a[2])
        m = _w2c(r, rng.normal(0, 3, 3))
        from oracle.chain import from_4x4
        assert np.abs(np.array(op.centre(from_4x4(m))) - np.linalg.inv(m)[:3, 3]).max() < 1e-12


def test_second_difference_closed_forms():
    from oracle.chain import from_4x4
    # p_t = p0 + v t + a t^2/2 with dyadic coefficients -> Eq. 3 returns a bit-exactly
    p0, v, a = np.array([1.0, -2.0, 0.5]), np.array([0.25, 0.5, -0.125]), np.array([0.5, -0.25, 1.0])
    cs = [op.centre(from_4x4(_w2c(np.eye(3), p0 + v * t + a * t * t / 2))) for t in range(8)]
    for t in range(2, 8):
        assert op.world_vector(cs, t, op.ACCEL) == list(a)
        assert op.world_vector(cs, t, op.VELOCITY) == list(v + a * (2 * t - 1) / 2)
    # cubic: second difference of b t^3 is 6 b (t-1)
    b = np.array([0.125, 0.0, -0.25])
    cs = [op.centre(from_4x4(_w2c(np.eye(3), p0 + a * t * t / 2 + b * t ** 3))) for t in range(8)]
    for t in range(2, 8):
        assert op.world_vector(cs, t, op.ACCEL) == list(a + 6 * b * (t - 1))
    assert op.world_vector(cs, 1, op.ACCEL) is None and op.world_vector(cs, 0, op.VELOCITY) is None


def _random_traj(rng, n):
    poses = []
    for t in range(n):
        a = rng.normal(0, 0.3, 3)
        poses.append(_w2c(_rot(1, a[1]) @ _rot(0, a[0]) @ _rot(2, a[2]), rng.normal(0, 1, 3) + [0, 0, t]))
    return poses


def test_gauge_invariance_and_scale():
    rng = np.random.default_rng(2)
    poses = _random_traj(rng, 10)
    base = _frames(poses, n_points=4, mag=op.MAG_RAW, sigma=3.0)
    g = np.eye(4)
    g[:3, :3] = _rot(0, 0.7) @ _rot(2, -1.1)
    g[:3, 3] = [3.0, -1.0, 2.0]
    moved = _frames([m @ g for m in poses], n_points=4, mag=op.MAG_RAW, sigma=3.0)
    lam = 2.5
    scaled_poses = []
    for m in poses:
        m2 = m.copy()
        m2[:3, 3] *= lam
        scaled_poses.append(m2)
    scaled = _frames(scaled_poses, n_points=4, mag=op.MAG_RAW, sigma=3.0)
    for fb, fm, fs in zip(base, moved, scaled):
        assert len(fb["points"]) == len(fm["points"]) == len(fs["points"])
        for pb, pm, ps in zip(fb["points"], fm["points"], fs["points"]):
            assert np.allclose(pb, pm, rtol=1e-5)
            assert np.allclose(pb[:2], ps[:2], rtol=1e-5) and np.isclose(ps[2], lam * pb[2], rtol=1e-5)
        assert fb["focus_index"] == fm["focus_index"] == fs["focus_index"]


def test_rotation_preserves_norm_and_magnitude_modes():
    rng = np.random.default_rng(3)
    poses = _random_traj(rng, 6)
    from oracle.chain import from_4x4
    ps = [from_4x4(m) for m in poses]
    cs = [op.centre(p) for p in ps]
    for t in range(2, 6):
        a_w = op.world_vector(cs, t, op.ACCEL)
        a_c = np.array(ps[t][0]) @ np.array(a_w)
        assert abs(np.linalg.norm(a_c) - op.norm3(a_w)) < 1e-12
        u, v, s = op.project(a_w, ps[t][0], 200.0, 210.0, 112.0, 96.0, 2.0, op.MAG_RAW, 1e-6)
        assert abs(s - 2.0 * np.linalg.norm(a_w)) < 1e-12
        assert abs(u - (112.0 + 200.0 * a_c[0] / a_c[2])) < 1e-9
        assert abs(v - (96.0 + 210.0 * a_c[1] / a_c[2])) < 1e-9
        assert op.project(a_w, ps[t][0], 200.0, 210.0, 112.0, 96.0, 2.0, op.MAG_UNIT, 1e-6)[2] == 2.0


def test_validity_rules():
    ident = [[1.0, 0, 0], [0, 1.0, 0], [0, 0, 1.0]]
    pr = lambda a: op.project(a, ident, 1.0, 1.0, 0.0, 0.0, 1.0, op.MAG_UNIT, 1e-6)
    assert pr(None) is None
    assert pr([0.0, 0.0, 1e-13]) is None                      # |a_w| < 1e-12
    assert pr([1.0, 0.0, 1e-7]) is None                       # a_z ~ 0 relative to |a_c|
    assert pr([1.0, 0.0, 1e-5]) is not None
    assert pr([0.5, 0.0, -1.0])[0] == -0.5                    # a_z < 0 projected literally (C3)
    assert op.project([1e-9, 0, 1e-9], ident, 1.0, 1.0, 0.0, 0.0, 1.0, op.MAG_RAW, 1e-6)[2] == op.SIGMA_MIN


def test_trailing_window_and_frame_choice():
    rng = np.random.default_rng(4)
    poses = _random_traj(rng, 9)
    cur = _frames(poses, n_points=3)
    own = _frames(poses, n_points=3, pts=op.PTS_OWN_FRAME)
    one = _frames(poses, n_points=1)
    assert [len(f["points"]) for f in cur] == [0, 0, 1, 2, 3, 3, 3, 3, 3]
    for t in range(2, 9):
        assert cur[t]["points"][-1] == one[t]["points"][0] == own[t]["points"][-1]
        assert cur[t]["focus_index"] == own[t]["focus_index"] == one[t]["focus_index"]
        if t >= 3:      # OWN_FRAME: the previous frame's own point, unchanged (C6)
            assert own[t]["points"][-2] == one[t - 1]["points"][0]
            assert cur[t]["points"][-2] != one[t - 1]["points"][0]
    sub = _frames(poses, n_points=3, render_begin=4, render_end=7)
    assert [f["points"] for f in sub] == [f["points"] for f in cur[4:7]]
