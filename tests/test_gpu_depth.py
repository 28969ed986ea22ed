"""GPU parity: mf_align_depth (through the C ABI) vs oracle/depth.py (reading F2).
Bars: window scales c_n within 1e-12 relative (both sides sum exact fp64 products, in different orders); stitched depth within
1e-6 relative (one fp32 rounding of c_n * D, plus the c_n difference); invalid pixels propagate as the product defines."""
import numpy as np
import pytest
import torch

from oracle import depth as od
from oracle import render as orr
from oracle import windows as ow
from paper_2601_07154_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2601_07154_b200 import api as a
    a.lib()
    return a


def _case(api, n, w, stride, h, wd, seed, **kw):
    loc, _ = synth.depth_windows(n, w, ow.window_starts(n, w, stride), h, wd, seed, **kw)
    ref, c_ref = od.align_depth(loc, w, stride, n)
    got, c = api.align_depth(torch.from_numpy(loc).cuda(), stride, n)
    torch.cuda.synchronize()
    got, c = got.cpu().numpy(), c.cpu().numpy()
    assert np.abs(c - c_ref).max() <= 1e-12 * np.abs(c_ref).max(), (c, c_ref)
    fin = np.isfinite(ref)
    assert np.array_equal(np.isnan(got), np.isnan(ref)) and np.array_equal(np.isinf(got), np.isinf(ref))
    assert np.abs(got[fin] - ref[fin]).max() <= 1e-6 * np.abs(ref[fin]).max()
    assert (np.abs(got[fin] - ref[fin]) <= 1e-6 * np.abs(ref[fin]) + 1e-30).all()
    return loc, got, c


@pytest.mark.parametrize("n,w,stride,h,wd", [
    (4, 4, 2, 8, 8),            # one window: pass-through
    (12, 4, 2, 6, 10),          # regular strides, vector path
    (13, 4, 2, 7, 9),           # tail window (larger last overlap), scalar path (63 pixels)
    (23, 8, 7, 5, 12),          # overlap of one frame
    (9, 5, 1, 4, 4),            # stride 1
    (48, 32, 16, 294, 518),     # the BJ campus window at the model's resolution: many tiles, ragged vector tail
    (100, 16, 8, 37, 41),       # odd sizes
])
def test_align_depth_parity(api, n, w, stride, h, wd):
    _case(api, n, w, stride, h, wd, seed=11 + n)


def test_align_depth_recovers_gauges_and_ignores_invalid_pixels(api):
    n, w, stride = 40, 8, 4
    loc, g = synth.depth_windows(n, w, ow.window_starts(n, w, stride), 16, 20, 5, noise=0.0)
    got, c = api.align_depth(torch.from_numpy(loc).cuda(), stride, n)
    assert np.abs(c.cpu().numpy() - g / g[0]).max() <= 1e-6        # fp32 inputs: the gauges come back to fp32 accuracy
    _case(api, n, w, stride, 16, 20, 6, invalid=0.2)               # zeros, NaN, inf, negatives in both windows
    # nothing valid on an overlap: that window keeps the scale of the previous one
    loc2 = loc.copy()
    off = ow.window_starts(n, w, stride)
    loc2[3, :w - stride] = np.nan
    ref, c_ref = od.align_depth(loc2, w, stride, n)
    _, c2 = api.align_depth(torch.from_numpy(loc2).cuda(), stride, n)
    c2 = c2.cpu().numpy()
    assert c2[3] == c2[2] and np.abs(c2 - c_ref).max() <= 1e-12 * np.abs(c_ref).max() and len(off) == len(c2)


def test_align_depth_is_deterministic_and_feeds_the_focus_call(api):
    n, w, stride, h, wd = 48, 32, 16, 294, 518
    loc, _ = synth.depth_windows(n, w, ow.window_starts(n, w, stride), h, wd, 3)
    x = torch.from_numpy(loc).cuda()
    a, ca = api.align_depth(x, stride, n)
    b, cb = api.align_depth(x, stride, n)
    assert torch.equal(a, b) and torch.equal(ca, cb)
    # stitched model-resolution depth -> mf_motion_focus_upsampled: the guided depth is the focus map times the upsampled stream
    cfg = synth.CONFIGS[3]
    poses = torch.from_numpy(np.asarray(synth.trajectory(cfg, 1, n))).cuda()
    out = api.motion_focus_upsampled(poses, cfg["fx"], cfg["fy"], cfg["cx"], cfg["cy"], cfg["width"], cfg["height"],
                                     a[40:42].contiguous(),
                                     api.focus_params(n_points=15, sigma=cfg["sigma"]), render_begin=40, render_end=42)
    torch.cuda.synchronize()
    assert out["focus_map"].max() > 0
    for f in range(2):
        up = orr.upsample_bilinear(a[40 + f].cpu().numpy(), cfg["width"], cfg["height"])      # fp64, reading F1
        want = out["focus_map"][f].cpu().numpy().astype(np.float64) * up
        assert np.abs(out["guided_depth"][f].cpu().numpy() - want).max() <= 1e-5 * np.abs(want).max()


def _random_depth_cases(count, seed):
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(count):
        w = int(rng.integers(2, 12))
        out.append((w + int(rng.integers(0, 40)), w, int(rng.integers(1, w)), int(rng.integers(1, 40)), int(rng.integers(1, 60)),
                    float(rng.choice([0.0, 0.1])), int(rng.integers(1 << 30))))
    return out


@pytest.mark.parametrize("n,w,stride,h,wd,invalid,seed", _random_depth_cases(12, 20260109))
def test_align_depth_random_shapes(api, n, w, stride, h, wd, invalid, seed):
    _case(api, n, w, stride, h, wd, seed, invalid=invalid)


@pytest.mark.parametrize("n,w,stride,h,wd", [(12, 4, 2, 6, 10), (13, 4, 2, 7, 9), (23, 8, 7, 5, 12), (9, 5, 1, 4, 4), (80, 32, 16, 74, 130)])
def test_align_depth_step_reproduces_the_batch_call(api, n, w, stride, h, wd):
    # streaming form: one window per call, scale carried in a device-resident state -> bit-identical to mf_align_depth
    loc, _ = synth.depth_windows(n, w, ow.window_starts(n, w, stride), h, wd, 21 + n, invalid=0.05)
    x = torch.from_numpy(loc).cuda()
    ref, c_ref = api.align_depth(x, stride, n)
    starts = ow.window_starts(n, w, stride)
    state = api.align_depth_state()
    parts = [api.align_depth_step(x[0], state, first=True)]
    for i in range(1, len(starts)):
        parts.append(api.align_depth_step(x[i], state, prev_window=x[i - 1], new_frames=starts[i] - starts[i - 1]))
    got = torch.cat(parts)
    assert got.shape == ref.shape
    assert torch.equal(torch.nan_to_num(got, nan=-7.0), torch.nan_to_num(ref, nan=-7.0))
    c_last = state[:8].view(torch.float64).item()
    assert c_last == c_ref[-1].item()
    with pytest.raises(api.MfError):
        api.align_depth_step(x[1], state, prev_window=x[0], new_frames=w)        # new_frames must be < W
    with pytest.raises(api.MfError):
        api.align_depth_step(x[1], state, new_frames=1)                           # previous window required


def test_streaming_depth_pipeline_matches_batch(api):
    # per window: chain step -> rolling pose buffer, depth scale step -> new frames, render with in-pass upsampling
    # == chain_poses + align_depth + motion_focus_upsampled on the whole clip, bit for bit
    cfg = synth.CONFIGS[1]
    n_frames, w, stride = 48, 8, 4
    width, height, k = 256, 128, (180.0, 180.0, 128.0, 64.0)
    traj = synth.trajectory(cfg, synth.seed_for(1, 21), n_frames)
    loc = torch.from_numpy(synth.local_windows(traj, w, ow.window_starts(n_frames, w, stride), seed=5, perturb_rot=1e-3, perturb_t=1e-3)).cuda()
    dloc = torch.from_numpy(synth.depth_windows(n_frames, w, ow.window_starts(n_frames, w, stride), 36, 64, 31)[0]).cuda()
    prm = api.focus_params(n_points=15, sigma=12.0)
    poses = api.chain_poses(loc, stride, n_frames)
    stream, _ = api.align_depth(dloc, stride, n_frames)
    batch = api.motion_focus_upsampled(poses, *k, width, height, stream, prm)
    ring_len = w + 24
    ring = torch.zeros((ring_len, 4, 4), device="cuda", dtype=torch.float64)
    pstate, dstate = api.chain_state(), api.align_depth_state()
    t_done = 0
    for n in range(loc.shape[0]):
        new = api.chain_poses_step(loc[n], pstate, new_frames=stride, first=n == 0)
        dnew = api.align_depth_step(dloc[n], dstate, prev_window=dloc[n - 1] if n else None, new_frames=stride, first=n == 0)
        m = new.shape[0]
        assert dnew.shape[0] == m and torch.equal(dnew, stream[t_done:t_done + m])
        ring = torch.cat([ring[m:], new])
        t_done += m
        if t_done < ring_len:
            continue
        out = api.motion_focus_upsampled(ring, *k, width, height, dnew, prm, render_begin=ring_len - m, render_end=ring_len)
        sl = slice(t_done - m, t_done)
        assert torch.equal(out["focus_index"], batch["focus_index"][sl])
        assert torch.equal(out["focus_map"], batch["focus_map"][sl]) and torch.equal(out["guided_depth"], batch["guided_depth"][sl])
    assert t_done == n_frames


def test_align_depth_argument_errors(api):
    x = torch.ones((3, 4, 2, 2), device="cuda")
    with pytest.raises(api.MfError):
        api.align_depth(x, 2, 9)                       # 9 frames with W=4, stride=2 make 4 windows, not 3
    with pytest.raises(api.MfError):
        api.align_depth(x, 4, 8)                       # stride >= W
    with pytest.raises(api.MfError):
        api.align_depth(x.double(), 2, 8)
    with pytest.raises(api.MfError):
        api.align_depth(x, 2, 8, workspace=torch.empty((8,), device="cuda", dtype=torch.uint8))
