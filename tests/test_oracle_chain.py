"""Pins for oracle/windows.py and oracle/chain.py.  CPU only.
BJ north_star: "composing the pose chain with identity overlaps must be exact"."""
import math

import numpy as np
import pytest

from oracle import chain as oc
from oracle import windows as ow


def _rot(axis, a):
    c, s = math.cos(a), math.sin(a)
    m = {0: [[1, 0, 0], [0, c, -s], [0, s, c]], 1: [[c, 0, s], [0, 1, 0], [-s, 0, c]],
         2: [[c, -s, 0], [s, c, 0], [0, 0, 1]]}[axis]
    return np.array(m, dtype=np.float64)


def _rigid(rng, yaw_only=False):
    g = np.eye(4)
    a = rng.normal(0, 0.7, 3)
    g[:3, :3] = _rot(1, a[1]) if yaw_only else _rot(1, a[1]) @ _rot(0, a[0]) @ _rot(2, a[2])
    g[:3, 3] = rng.normal(0, 2.0, 3)
    return g


def _truth(n, rng):
    return np.stack([_rigid(rng) for _ in range(n)])


def _cut(truth, w, stride, gauges):
    """Window n's local poses: T^G_t . G_n (a different world gauge per window)."""
    starts = ow.window_starts(len(truth), w, stride)
    return [[truth[s + k] @ gauges[n] for k in range(w)] for n, s in enumerate(starts)]


# ---- windows (reading B6) --------------------------------------------------------

def test_window_counts_match_configs():
    # BASELINE.json configs: tiny, suburban, city, campus, town
    assert ow.num_windows(4, 4, 2) == 1
    assert ow.num_windows(240, 8, 4) == 59
    assert ow.num_windows(600, 16, 8) == 74
    assert ow.num_windows(1800, 32, 16) == 112
    assert ow.num_windows(720, 64, 32) == 22
    assert ow.window_starts(1800, 32, 16)[-2:] == [1760, 1768]      # tail window, larger overlap
    assert ow.window_starts(720, 64, 32)[-2:] == [640, 656]


@pytest.mark.parametrize("n,w,stride", [(4, 4, 2), (10, 4, 2), (11, 4, 3), (9, 4, 1), (23, 8, 7), (50, 8, 4)])
def test_emitted_frames_partition_the_clip(n, w, stride):
    em = ow.emitted(n, w, stride)
    assert em[0] == (0, w) and em[-1][1] == n
    assert all(em[i][1] == em[i + 1][0] for i in range(len(em) - 1))      # contiguous, disjoint
    starts = ow.window_starts(n, w, stride)
    for (b, e), s in zip(em, starts):
        assert s <= b < e <= s + w                                         # inside its window
    owner = ow.owner_of_frames(n, w, stride)
    assert all(starts[nn] + k == t for t, (nn, k) in enumerate(owner))
    for i in range(1, len(starts)):                                        # overlap >= 1: anchor shared
        assert starts[i] <= starts[i - 1] + w - 1 < starts[i] + w


# ---- chain ---------------------------------------------------------------------------

@pytest.mark.parametrize("n,w,stride", [(12, 4, 2), (13, 4, 3), (9, 4, 1), (30, 8, 7), (19, 8, 4)])
def test_identity_overlap_rigid_recovers_truth(n, w, stride):
    rng = np.random.default_rng(n * 100 + stride)
    truth = _truth(n, rng)
    gauges = [_rigid(rng) for _ in ow.window_starts(n, w, stride)]
    out = np.array(oc.chain_poses(_cut(truth, w, stride, gauges), w, stride, n, oc.RIGID))
    assert np.abs(out - truth @ gauges[0]).max() < 1e-12


def test_identity_overlap_bit_exact_on_exact_inputs():
    # 90-degree rotations and dyadic translations: every fp64 operation is exact
    rng = np.random.default_rng(5)
    q = [np.round(_rot(ax, k * math.pi / 2)) for ax in range(3) for k in range(4)]

    def exact():
        g = np.eye(4)
        g[:3, :3] = q[rng.integers(len(q))] @ q[rng.integers(len(q))]
        g[:3, 3] = rng.integers(-64, 64, 3) / 8.0
        return g
    truth = np.stack([exact() for _ in range(14)])
    gauges = [exact() for _ in ow.window_starts(14, 4, 2)]
    out = np.array(oc.chain_poses(_cut(truth, 4, 2, gauges), 4, 2, 14, oc.RIGID))
    assert np.array_equal(out, truth @ gauges[0])
    yg = [g for g in gauges]
    for g in yg:
        g[:3, :3] = q[4 + rng.integers(4)]              # Y-axis quarter turns
    out = np.array(oc.chain_poses(_cut(truth, 4, 2, yg), 4, 2, 14, oc.YAW_TRANSLATION))
    assert np.array_equal(out, truth @ yg[0])


def test_yaw_mode_exact_for_yaw_gauges_and_not_for_6dof():
    rng = np.random.default_rng(6)
    truth = _truth(16, rng)
    starts = ow.window_starts(16, 4, 2)
    yaw_g = [_rigid(rng, yaw_only=True) for _ in starts]
    out = np.array(oc.chain_poses(_cut(truth, 4, 2, yaw_g), 4, 2, 16, oc.YAW_TRANSLATION))
    assert np.abs(out - truth @ yaw_g[0]).max() < 1e-12
    full_g = [_rigid(rng) for _ in starts]
    out = np.array(oc.chain_poses(_cut(truth, 4, 2, full_g), 4, 2, 16, oc.YAW_TRANSLATION))
    assert np.abs(out - truth @ full_g[0]).max() > 1e-2          # designed: pitch/roll are locked


def test_single_window_is_passthrough():
    rng = np.random.default_rng(7)
    loc = _truth(4, rng).astype(np.float32)
    for mode in (oc.RIGID, oc.YAW_TRANSLATION):
        out = np.array(oc.chain_poses([loc], 4, 2, 4, mode))
        assert np.array_equal(out[:, :3], loc.astype(np.float64)[:, :3])
        assert np.array_equal(out[:, 3], np.tile([0, 0, 0, 1.0], (4, 1)))


@pytest.mark.parametrize("mode", [oc.RIGID, oc.YAW_TRANSLATION])
def test_within_window_relative_poses_preserved(mode):
    rng = np.random.default_rng(8)
    n, w, stride = 14, 4, 2
    local = [[_rigid(rng) for _ in range(w)] for _ in ow.window_starts(n, w, stride)]   # inconsistent overlaps
    out = np.array(oc.chain_poses(local, w, stride, n, mode))
    for (b, e), s, loc in zip(ow.emitted(n, w, stride), ow.window_starts(n, w, stride), local):
        for t in range(b + 1, e):
            rel_g = out[t] @ np.linalg.inv(out[b])
            rel_l = loc[t - s] @ np.linalg.inv(loc[b - s])
            assert np.abs(rel_g - rel_l).max() < 1e-12


def test_yaw_mode_anchor_centres_coincide_and_transforms_are_yaw():
    rng = np.random.default_rng(9)
    n, w, stride = 14, 4, 2
    starts = ow.window_starts(n, w, stride)
    local = [[_rigid(rng) for _ in range(w)] for _ in starts]
    out, a = oc.chain_poses(local, w, stride, n, oc.YAW_TRANSLATION, return_transforms=True)
    a = np.array(a)
    for an in a:
        assert np.array_equal(an[1, :3], [0, 1, 0]) and np.array_equal(an[:3, 1], [0, 1, 0])
        assert abs(np.linalg.det(an[:3, :3]) - 1) < 1e-12
    centre = lambda m: -m[:3, :3].T @ m[:3, 3]
    for i in range(1, len(starts)):
        k_a = starts[i - 1] + w - 1 - starts[i]
        g_prev = np.array(local[i - 1][w - 1]) @ np.linalg.inv(a[i - 1])
        g_cur = np.array(local[i][k_a]) @ np.linalg.inv(a[i])
        assert np.abs(centre(g_prev) - centre(g_cur)).max() < 1e-11


def test_yaw_extraction_direction():
    # window 1's local frame is window 0's rotated by +0.3 rad about Y: B_1 must be that rotation
    th = 0.3
    g = np.eye(4)
    g[:3, :3] = _rot(1, th)
    g[:3, 3] = [1.0, 0.0, 2.0]
    truth = _truth(6, np.random.default_rng(10))
    out, a = oc.chain_poses(_cut(truth, 4, 2, [np.eye(4), g]), 4, 2, 6, oc.YAW_TRANSLATION,
                            return_transforms=True)
    # local_1 = T.G  ->  T = local_1 . G^-1  ->  A_1 = G  (maps window-1 coords to window-0 coords)
    assert np.abs(np.array(a[1]) - g).max() < 1e-12
    assert np.abs(np.array(out) - truth).max() < 1e-12


@pytest.mark.parametrize("mode", [oc.RIGID, oc.YAW_TRANSLATION])
def test_gauge_covariance(mode):
    rng = np.random.default_rng(11)
    n, w, stride = 12, 4, 2
    local = [[_rigid(rng) for _ in range(w)] for _ in ow.window_starts(n, w, stride)]
    g = _rigid(rng, yaw_only=(mode == oc.YAW_TRANSLATION))
    out = np.array(oc.chain_poses(local, w, stride, n, mode))
    local2 = [[m @ g for m in local[0]]] + local[1:]
    out2 = np.array(oc.chain_poses(local2, w, stride, n, mode))
    assert np.abs(out2 - out @ g).max() < 1e-11


def test_fold_equals_sequential_trajectory_alignment():
    """align the current batch to the terminal pose of the previous *trajectory*
    (sequential restatement with numpy inverses, RIGID mode)."""
    rng = np.random.default_rng(12)
    n, w, stride = 15, 4, 3
    starts = ow.window_starts(n, w, stride)
    local = [[_rigid(rng) for _ in range(w)] for _ in starts]
    out = np.array(oc.chain_poses(local, w, stride, n, oc.RIGID))
    traj = {k: np.array(local[0][k]) for k in range(w)}
    for i in range(1, len(starts)):
        t_a = starts[i - 1] + w - 1
        k_a = t_a - starts[i]
        # find X with local_i[k_a] . X = traj[t_a]
        x = np.linalg.inv(np.array(local[i][k_a])) @ traj[t_a]
        for k in range(w):
            t = starts[i] + k
            if t not in traj:
                traj[t] = np.array(local[i][k]) @ x
    ref = np.stack([traj[t] for t in range(n)])
    assert np.abs(out - ref).max() < 1e-11
