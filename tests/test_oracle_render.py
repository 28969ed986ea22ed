"""Pins for oracle/render.py (Eq. 7).  CPU only."""
import math

import numpy as np

from oracle import render as orr

f32 = np.float32


def _pts(*triples):
    return [(f32(u), f32(v), f32(s)) for (u, v, s) in triples]


def test_single_point_closed_form():
    pts = _pts((20, 12, 4))
    m, g = orr.focus_map(pts, 48, 32, orr.NORM_MAX)
    assert g is None
    assert m[12, 20] == 1.0 and m.max() == 1.0
    e = math.exp(-0.5)                                           # 0.6065306597...
    for (x, y) in [(24, 12), (16, 12), (20, 16), (20, 8)]:      # distance sigma along an axis
        assert abs(m[y, x] - e) < 1e-15
    assert abs(m[15, 24] - math.exp(-(16 + 9) / 32.0)) < 1e-15
    # 4-fold symmetry about the point and monotone decrease along a ray
    assert np.array_equal(m[12, 20:41], m[12, 20::-1]) and np.array_equal(m[12:24, 20], m[12:0:-1, 20])
    assert (np.diff(m[12, 20:]) < 0).all()
    assert (m >= 0).all() and (m <= 1).all()


def test_brute_force_and_separable_identity_small():
    rng = np.random.default_rng(1)
    pts = _pts(*[(rng.uniform(-4, 36), rng.uniform(-4, 28), rng.uniform(1, 9)) for _ in range(5)])
    u_map = orr.unnormalised(pts, 32, 24)
    for (x, y) in [(0, 0), (31, 23), (7, 19), (16, 3)]:
        assert abs(u_map[y, x] - orr.brute_force_pixel(pts, x, y)) < 1e-14
    # independent evaluation route: product of 1-D tables
    xs, ys = np.arange(32.0), np.arange(24.0)
    sep = sum(np.outer(np.exp(-(ys - float(v)) ** 2 / (2 * float(s) ** 2)),
                       np.exp(-(xs - float(u)) ** 2 / (2 * float(s) ** 2))) for (u, v, s) in pts)
    assert np.abs(sep - u_map).max() < 1e-13


def test_normalisations():
    pts = _pts((100.3, 80.7, 6.0), (140.0, 90.0, 9.5), (60.0, 110.0, 4.0))
    u_map = orr.unnormalised(pts, 256, 192)
    m_sum, _ = orr.focus_map(pts, 256, 192, orr.NORM_SUM)
    assert abs(m_sum.sum() - 1.0) < 1e-12
    # kernels well inside the image, sigma >~ 1 px: sum -> 2 pi sum sigma_i^2
    assert abs(u_map.sum() / (2 * math.pi * (36 + 9.5 ** 2 + 16)) - 1) < 1e-9
    m_none, _ = orr.focus_map(pts, 256, 192, orr.NORM_NONE)
    assert np.array_equal(m_none, u_map)
    m_max, _ = orr.focus_map(pts, 256, 192, orr.NORM_MAX)
    assert m_max.max() == 1.0 and np.allclose(m_max * u_map.max(), u_map, rtol=1e-15)
    # no points -> M = 0 (reading C2)
    m0, g0 = orr.focus_map([], 16, 8, orr.NORM_MAX, depth=np.ones((8, 16), dtype=np.float32))
    assert not m0.any() and not g0.any()


def test_translation_and_permutation():
    pts = _pts((30.5, 20.25, 5.0), (44.0, 31.0, 7.0))
    shifted = _pts((30.5 + 7, 20.25 + 3, 5.0), (44.0 + 7, 31.0 + 3, 7.0))
    a = orr.unnormalised(pts, 96, 64)
    b = orr.unnormalised(shifted, 96, 64)
    assert np.allclose(b[3:, 7:], a[:-3, :-7], rtol=1e-14, atol=0)
    c = orr.unnormalised(pts[::-1], 96, 64)
    assert np.abs(c - a).max() < 1e-15


def test_off_image_points_contribute_tails():
    pts = _pts((-10.0, 5.0, 8.0))
    m, _ = orr.focus_map(pts, 32, 16, orr.NORM_NONE)
    assert abs(m[5, 0] - math.exp(-100 / 128.0)) < 1e-15 and m[5, 0] == m.max()


def test_guided_depth():
    rng = np.random.default_rng(2)
    pts = _pts((10.0, 8.0, 3.0), (20.0, 9.0, 5.0))
    d = rng.uniform(1, 30, (16, 32)).astype(np.float32)
    m, g = orr.focus_map(pts, 32, 16, orr.NORM_MAX, depth=d)
    assert np.array_equal(g, m * d.astype(np.float64))
    m1, g1 = orr.focus_map(pts, 32, 16, orr.NORM_MAX, depth=np.ones_like(d))
    assert np.array_equal(g1, m1) and (g <= d).all()


def test_sigma_per_point_is_used():
    # guards against a shared sigma: the wide kernel dominates far from both centres
    pts = _pts((8.0, 8.0, 1.0), (24.0, 8.0, 6.0))
    u_map = orr.unnormalised(pts, 32, 16)
    assert abs(u_map[8, 12] - (math.exp(-16 / 2.0) + math.exp(-144 / 72.0))) < 1e-15


def test_upsample_bilinear_pins():
    import torch
    rng = np.random.default_rng(3)
    lo = rng.uniform(1.0, 30.0, (7, 9))
    for (h, w) in [(14, 18), (20, 31), (7, 9), (5, 4), (33, 64)]:
        up = orr.upsample_bilinear(lo, w, h)
        ref = torch.nn.functional.interpolate(torch.from_numpy(lo)[None, None], size=(h, w), mode="bilinear",
                                              align_corners=False)[0, 0].numpy()
        assert np.abs(up - ref).max() < 1e-12
    assert np.array_equal(orr.upsample_bilinear(lo, 9, 7), lo)                       # same size: identity
    assert np.abs(orr.upsample_bilinear(np.full((3, 5), 4.25), 40, 24) - 4.25).max() < 1e-15   # constants are kept
    # a linear ramp is reproduced exactly away from the clamped border: D(x) = a (x + 1/2) w_lo / W - a/2
    ramp = np.tile(np.arange(6, dtype=np.float64) * 2.0, (4, 1))
    up = orr.upsample_bilinear(ramp, 24, 4)
    x = np.arange(24)
    src = np.clip((x + 0.5) * 6 / 24 - 0.5, 0.0, 5.0)
    assert np.abs(up[0] - 2.0 * src).max() < 1e-13
    # 2x upscale of two samples (hand values): src = -0.25 -> 0, 0.25, 0.75, 1.25 -> clamped to sample 1
    assert np.allclose(orr.upsample_bilinear(np.array([[0.0, 8.0]]), 4, 1), [[0.0, 2.0, 6.0, 8.0]], atol=1e-15)
    # a transposed call must differ (rows and columns are not interchangeable)
    assert orr.upsample_bilinear(lo, 18, 14).shape == (14, 18)
