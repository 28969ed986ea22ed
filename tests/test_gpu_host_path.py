"""GPU parity of the END-TO-END host-buffer entry points (mf_window_attention_host, mf_chain_and_focus_host): the calls
bench.py's `e2e` number goes through.  Each is compared (a) bit for bit with the device-pointer path and (b) with the
oracle within BJ north_star's bars, on pinned and on pageable host memory."""
import numpy as np
import pytest
import torch

from oracle import attention as oa
from oracle import chain as oc
from oracle import points as op
from oracle import render as orr
from oracle import windows as ow
from paper_2601_07154_b200 import synth

pytestmark = pytest.mark.gpu

MAX_ABS, REL_L2 = 2e-2, 1e-2


@pytest.fixture(scope="module")
def api():
    from paper_2601_07154_b200 import api as a
    a.lib()
    return a


def _to64(t):
    return t.detach().float().cpu().numpy().astype(np.float64)


def _host(t, pinned):
    t = t.cpu().contiguous()
    return t.pin_memory() if pinned else t


@pytest.mark.parametrize("pinned", [True, False])
@pytest.mark.parametrize("first_mode", [oa.FRAME, oa.GLOBAL])
@pytest.mark.parametrize("num_layers", [1, 2, 3, 24])
def test_window_attention_host_layers(api, num_layers, first_mode, pinned):
    # The layer stack alternates first_mode / other mode on the SAME q,k,v (include/mf.h), ping-ponging two device buffers;
    # what comes back must be the last layer's output: equal to mf_window_attention in that layer's mode bit for bit, and
    # to the oracle's attention in that mode within the bar.
    windows, w, p, heads = 2, 3, 100, 2
    q, k, v = synth.qkv(windows, w * p, heads, 64, 1000 + num_layers, device="cuda")
    hq, hk, hv = (_host(t, pinned) for t in (q, k, v))
    hout = _host(torch.full_like(q, float("nan")), pinned)
    got = api.window_attention_host(hq, hk, hv, w, p, first_mode, out=hout, num_layers=num_layers)
    assert got.data_ptr() == hout.data_ptr()
    other = oa.FRAME if first_mode == oa.GLOBAL else oa.GLOBAL
    last_mode = first_mode if (num_layers - 1) % 2 == 0 else other
    dev = api.window_attention(q, k, v, w, p, last_mode)
    torch.cuda.synchronize()
    assert torch.equal(got, dev.cpu()), "host path differs from the device path"
    if num_layers > 1:                                   # and it is NOT the other mode's output (the alternation is real)
        assert not torch.equal(got, api.window_attention(q, k, v, w, p, other if last_mode == first_mode else first_mode).cpu())
    ref, _ = oa.window_attention(_to64(q), _to64(k), _to64(v), w, p, last_mode)
    for n in range(windows):
        d = _to64(got[n]) - ref[n]
        assert np.abs(d).max() <= MAX_ABS and np.linalg.norm(d) / np.linalg.norm(ref[n]) <= REL_L2


def test_window_attention_host_head_dim_128_and_errors(api):
    q, k, v = synth.qkv(1, 2 * 70, 2, 128, 3, device="cuda")
    got = api.window_attention_host(q.cpu(), k.cpu(), v.cpu(), 2, 70, oa.GLOBAL, num_layers=2)      # last layer: FRAME
    assert torch.equal(got, api.window_attention(q, k, v, 2, 70, oa.FRAME).cpu())
    ref, _ = oa.window_attention(_to64(q), _to64(k), _to64(v), 2, 70, oa.FRAME)
    d = _to64(got) - ref
    assert np.abs(d).max() <= MAX_ABS and np.linalg.norm(d) / np.linalg.norm(ref) <= REL_L2
    # an unsupported head_dim is rejected before anything is allocated or copied (include/mf.h conventions)
    q32 = torch.zeros((1, 8, 1, 32), dtype=torch.bfloat16)
    free_before = torch.cuda.mem_get_info()[0]
    with pytest.raises(api.MfError, match="MF_ERR_UNSUPPORTED"):
        api.window_attention_host(q32, q32.clone(), q32.clone(), 1, 8, oa.GLOBAL, out=q32.clone())
    assert torch.cuda.mem_get_info()[0] == free_before


def _focus_bar(got, ref):
    floor = 1e-6 * np.abs(ref).max()
    bound = np.maximum(1e-5 * np.maximum(np.abs(ref), floor), 2e-38)
    err = np.abs(got.astype(np.float64) - ref)
    return (err / bound).max() if ref.any() else float(np.abs(got).max())


@pytest.mark.parametrize("pinned", [True, False])
@pytest.mark.parametrize("n_frames,w,stride,rb,re_,align", [
    (40, 8, 4, 0, 40, oc.YAW_TRANSLATION),         # whole clip
    (40, 8, 4, 22, 31, oc.YAW_TRANSLATION),        # sub-range: frames before render_begin supply the trailing points
    (23, 8, 7, 17, 23, oc.RIGID),                  # tail window with a larger overlap, rigid alignment
])
def test_chain_and_focus_host(api, n_frames, w, stride, rb, re_, align, pinned):
    cfg = synth.CONFIGS[1]
    width, height = 256, 144
    k = (190.0, 190.0, 128.0, 72.0)
    traj = synth.trajectory(cfg, synth.seed_for(1, 31), n_frames)
    loc = synth.local_windows(traj, w, ow.window_starts(n_frames, w, stride), seed=9, perturb_rot=1e-3, perturb_t=1e-3)
    count = re_ - rb
    depth = synth.depth(count, height, width, 55)
    prm = api.focus_params(n_points=15, sigma=9.0)
    out = api.chain_and_focus_host(_host(torch.from_numpy(loc), pinned), stride, n_frames, *k, width, height, prm,
                                   depth=_host(depth, pinned), render_begin=rb, render_end=re_, align=align)
    # (a) oracle: poses, focus_uv and focus_index bit-exact; maps within the 1e-5 bar
    ref_poses = oc.chain_poses(loc.tolist(), w, stride, n_frames, align)
    assert np.array_equal(out["global_w2c"].numpy(), np.array(ref_poses))
    frames = op.motion_points(ref_poses, *k, width, height, 15, 9.0, render_begin=rb, render_end=re_)
    assert [int(i) for i in out["focus_index"]] == [f["focus_index"] for f in frames]
    uv_ref = np.array([f["focus_uv"] for f in frames], dtype=np.float32)
    uv = out["focus_uv"].numpy()
    ok = np.isfinite(uv_ref).all(axis=1)
    assert np.array_equal(uv[ok].view(np.uint32), uv_ref[ok].view(np.uint32)) and np.isnan(uv[~ok]).all()
    live = 0
    for f, fr in enumerate(frames):
        m, g = orr.focus_map(fr["points"], width, height, orr.NORM_MAX, depth[f].numpy())
        assert _focus_bar(out["focus_map"][f].numpy(), m) <= 1.0 and _focus_bar(out["guided_depth"][f].numpy(), g) <= 1.0
        live += int(m.any())
    assert live >= count - 2                           # the comparison is not vacuous
    # (b) the device-pointer path, bit for bit
    g_poses = api.chain_poses(torch.from_numpy(loc).cuda(), stride, n_frames, align)
    dev = api.motion_focus(g_poses, *k, width, height, prm, depth=depth.cuda(), render_begin=rb, render_end=re_)
    torch.cuda.synchronize()
    for key in ("focus_map", "guided_depth", "focus_index"):
        assert torch.equal(out[key], dev[key].cpu()), key


def test_chain_and_focus_host_rejects_before_enqueue(api):
    loc = torch.zeros((3, 8, 4, 4), dtype=torch.float32)
    free_before = torch.cuda.mem_get_info()[0]
    with pytest.raises(api.MfError, match="MF_ERR_INVALID_ARG"):       # partition of 16 frames with W=8, stride=4 has 3 windows...
        api.chain_and_focus_host(loc, 4, 17, 100.0, 100.0, 32.0, 32.0, 64, 64)     # ...17 frames has 4
    with pytest.raises(api.MfError, match="MF_ERR_ALIGNMENT"):
        api.chain_and_focus_host(loc, 4, 16, 100.0, 100.0, 32.0, 32.0, 62, 64)     # width % 4
    assert torch.cuda.mem_get_info()[0] == free_before
