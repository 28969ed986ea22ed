"""Pins for oracle/depth.py (reading F2: least-squares depth scale on the window overlap).
The paper prints no value for this step (it is silent on the depth scale, P:68 / P:76), so the pins are what the
mathematics fixes: hand values, gauge recovery, numpy's least-squares solver, optimality, the invalid-pixel rule."""
import numpy as np
import pytest

from oracle import depth as od
from oracle import windows as ow


def _stream(n, h, w, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(0.5, 40.0, (n, h, w))


def _cut(stream, w, stride, gauges):
    starts = ow.window_starts(stream.shape[0], w, stride)
    return np.stack([stream[s:s + w] / g for s, g in zip(starts, gauges)])


def test_hand_values():
    # W = 2, stride = 1, N = 3, one row of two pixels.  Shared frame t = 1: a = (1, 3) in window 0, b = (0.5, 1.5) in
    # window 1  ->  r = (0.5 + 4.5) / (0.25 + 2.25) = 2;  frame 2 = 2 * (7, 9).
    loc = np.array([[[[2.0, 4.0]], [[1.0, 3.0]]], [[[0.5, 1.5]], [[7.0, 9.0]]]])
    out, c = od.align_depth(loc, 2, 1, 3)
    assert c.tolist() == [1.0, 2.0]
    assert out[:, 0, :].tolist() == [[2.0, 4.0], [1.0, 3.0], [14.0, 18.0]]
    # the ratio is previous / current, not the other way round
    assert od.overlap_ratio([4.0, 8.0], [2.0, 4.0]) == 2.0
    assert od.overlap_ratio([2.0, 4.0], [4.0, 8.0]) == 0.5


@pytest.mark.parametrize("n,w,stride", [(12, 4, 2), (13, 4, 2), (17, 6, 5), (9, 5, 1), (8, 8, 3), (23, 8, 4)])
def test_gauge_recovery(n, w, stride):
    # every window sees the true stream divided by its own unknown scale: the chain recovers the stream in window 0's scale,
    # with regular strides, a tail window (larger last overlap) and a single window
    stream = _stream(n, 3, 5, 7)
    nw = ow.num_windows(n, w, stride)
    g = np.random.default_rng(8).uniform(0.3, 3.0, nw)
    out, c = od.align_depth(_cut(stream, w, stride, g), w, stride, n)
    assert np.abs(c - g / g[0]).max() <= 1e-12 * np.abs(c).max()
    assert np.abs(out - stream / g[0]).max() <= 1e-11
    assert c[0] == 1.0


def test_chain_is_a_product_of_ratios():
    stream = _stream(10, 2, 3, 1)
    g = [1.0, 2.0, 0.5, 4.0]
    loc = _cut(stream, 4, 2, g)
    _, c = od.align_depth(loc, 4, 2, 10)
    r = [od.overlap_ratio(loc[k - 1, 2:4], loc[k, 0:2]) for k in range(1, 4)]
    assert np.allclose(c, np.cumprod([1.0] + r), rtol=1e-15)
    assert np.allclose(r, [2.0, 0.25, 8.0], rtol=1e-13)


def test_least_squares_against_numpy_and_optimality():
    rng = np.random.default_rng(5)
    b = rng.uniform(1.0, 20.0, 400)
    a = 1.7 * b + rng.normal(0.0, 0.3, 400)                # noisy: no exact ratio exists
    r = od.overlap_ratio(a, b)
    ref = np.linalg.lstsq(b[:, None], a, rcond=None)[0][0]
    assert abs(r - ref) <= 1e-12
    res = lambda s: float(np.sum((s * b - a) ** 2))
    assert res(r) < res(r * (1 + 1e-4)) and res(r) < res(r * (1 - 1e-4))
    assert abs(np.dot(r * b - a, b)) <= 1e-8              # normal equation: the residual is orthogonal to b


def test_invalid_pixels_are_ignored():
    a = np.array([2.0, np.nan, 6.0, 8.0, -1.0, 3.0, np.inf, 5.0])
    b = np.array([1.0, 5.0, 3.0, 0.0, 2.0, np.nan, 1.0, -np.inf])
    assert od.overlap_ratio(a, b) == 2.0                   # only pixels 0 and 2 count
    assert od.overlap_ratio([np.nan, 0.0], [1.0, 1.0]) == 1.0      # nothing valid: scale kept
    assert od.overlap_ratio([], []) == 1.0


def test_emitted_frames_come_from_the_owning_window():
    # different content per window (not a common stream): frame t must be c_n times window n's own map
    rng = np.random.default_rng(2)
    n, w, stride = 11, 4, 3
    nw = ow.num_windows(n, w, stride)
    loc = rng.uniform(1.0, 9.0, (nw, w, 2, 2))
    out, c = od.align_depth(loc, w, stride, n)
    for t, (k, j) in enumerate(ow.owner_of_frames(n, w, stride)):
        assert np.array_equal(out[t], c[k] * loc[k, j])
