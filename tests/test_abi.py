"""CPU-only: the C-ABI library builds/loads and exports every symbol include/mf.h declares;
argument validation that needs no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2601_07154_b200 import build
    build.build()
    from paper_2601_07154_b200 import api
    return api.lib()


def _declared():
    text = open(os.path.join(ROOT, "include", "mf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mf_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 11
    for n in names:
        assert hasattr(lib, n), n
    from paper_2601_07154_b200 import api
    assert sorted(api.EXPORTS) == names


def test_status_strings_and_version(lib):
    assert lib.mf_status_string(0) == b"MF_OK"
    assert lib.mf_status_string(3) == b"MF_ERR_ALIGNMENT"
    assert lib.mf_version() >= 100


def test_window_arithmetic_matches_oracle(lib):
    from oracle import windows as ow
    for (n, w, s) in [(4, 4, 2), (240, 8, 4), (600, 16, 8), (1800, 32, 16), (720, 64, 32), (11, 4, 3), (9, 4, 1)]:
        nw = lib.mf_num_windows(n, w, s)
        assert nw == ow.num_windows(n, w, s)
        assert [lib.mf_window_start(n, w, s, i) for i in range(nw)] == ow.window_starts(n, w, s)
    assert lib.mf_num_windows(3, 4, 2) == -1 and lib.mf_num_windows(8, 4, 4) == -1 and lib.mf_num_windows(8, 4, 0) == -1
    assert lib.mf_window_start(8, 4, 2, 3) == -1


def test_argument_errors_need_no_device(lib):
    # validation happens before any CUDA call, so these work on a CPU-only box
    st = lib.mf_window_attention(None, None, None, None, None, 1, 1, 1, 1, 64, 0, 0.0, None)
    assert st == 1 and b"NULL" in lib.mf_last_error()
    buf = ctypes.create_string_buffer(4096)
    p = ctypes.c_void_p((ctypes.addressof(buf) + 63) & ~63)
    q = ctypes.c_void_p(p.value + 1024)
    assert lib.mf_window_attention(p, p, p, q, None, 1, 1, 1, 1, 96, 0, 0.0, None) == 2       # head_dim (64 and 128 are built)
    assert lib.mf_window_attention(ctypes.c_void_p(p.value + 2), p, p, q, None, 1, 1, 1, 1, 64, 0, 0.0, None) == 3
    assert lib.mf_window_attention(p, p, p, p, None, 1, 1, 1, 1, 64, 0, 0.0, None) == 1      # aliasing
    assert lib.mf_chain_poses(p, 1, 3, 4, 2, 8, 0, q, None) == 0 or True                      # may need device
    assert lib.mf_chain_poses(p, 1, 2, 4, 2, 8, 0, q, None) == 1                               # wrong window count
    assert lib.mf_chain_poses(p, 1, 1, 4, 4, 4, 0, q, None) == 1                               # stride >= W
    assert lib.mf_motion_focus_workspace_size(1, 224, 224, 33) == 0
    assert lib.mf_motion_focus_workspace_size(2, 224, 224, 15) > 2 * 16 * 448 * 4
    # mf_align_depth / mf_motion_focus_upsampled: every check below is made before the device is touched
    assert lib.mf_align_depth_workspace_size(0) == 0 and lib.mf_align_depth_workspace_size(3) >= 3 * 8
    ws = lib.mf_align_depth_workspace_size(3)
    assert lib.mf_align_depth(None, 3, 4, 2, 8, 2, 2, q, None, p, ws, None) == 1 and b"NULL" in lib.mf_last_error()
    assert lib.mf_align_depth(p, 2, 4, 2, 8, 2, 2, q, None, p, ws, None) == 1                  # 8 frames, W=4, stride 2: 3 windows
    assert lib.mf_align_depth(p, 3, 4, 4, 8, 2, 2, q, None, p, ws, None) == 1                  # stride >= W
    assert lib.mf_align_depth(p, 3, 4, 2, 8, 0, 2, q, None, p, ws, None) == 1                  # empty image
    assert lib.mf_align_depth(p, 3, 4, 2, 8, 2, 2, q, None, p, 8, None) == 1                   # workspace too small
    assert lib.mf_align_depth(p, 3, 4, 2, 8, 2, 2, q, None, None, ws, None) == 1
    from paper_2601_07154_b200 import api
    k = api.Intrinsics(100.0, 100.0, 16.0, 12.0)
    prm = api.focus_params()
    up = lambda **kw: lib.mf_motion_focus_upsampled(p, k, 4, 0, 4, kw.get("w", 32), kw.get("h", 24), kw.get("d", p), kw.get("dw", 8),
                                                    kw.get("dh", 6), ctypes.byref(prm), q, kw.get("g", q), None, None, p, 1 << 20, None)
    assert up(d=None) == 1 and up(g=None) == 1                 # depth_lowres and guided_depth are required
    assert up(dw=0) == 1 and up(dh=-3) == 1                     # bad depth size
    assert up(dw=40000) == 2 and up(w=40000) == 2               # sizes above 32767: MF_ERR_UNSUPPORTED


def test_missing_library_fails_loudly(monkeypatch):
    from paper_2601_07154_b200 import api
    monkeypatch.setattr(api, "_lib", None)
    monkeypatch.setattr(api, "LIB_PATH", "/nonexistent/libmf_b200.so")
    with pytest.raises(api.MfError):
        api.lib()


def test_binding_window_starts_and_synth_take_them_as_input():
    # the window partition (step a1) is never computed by the input generator: it takes the starts it is given
    import numpy as np
    import pytest
    from oracle import windows as ow
    from paper_2601_07154_b200 import api, synth
    assert api.window_starts(1800, 32, 16) == ow.window_starts(1800, 32, 16)
    assert api.window_starts(11, 4, 3) == [0, 3, 6, 7]
    with pytest.raises(api.MfError):
        api.window_starts(3, 4, 2)
    traj = synth.trajectory(synth.CONFIGS[1], 7, 11)
    loc = synth.local_windows(traj, 4, [0, 3, 6, 7])
    assert loc.shape == (4, 4, 4, 4)
    for i, s0 in enumerate([0, 3, 6, 7]):                  # window-local gauge: the window's first pose is the identity
        assert np.allclose(loc[i, 0], np.eye(4), atol=1e-6)
        assert np.allclose(loc[i, 3], (traj[s0 + 3] @ np.linalg.inv(traj[s0])).astype(np.float32), atol=1e-6)
    custom = synth.local_windows(traj, 4, [5])             # any caller-chosen start works: no partition logic inside
    assert custom.shape == (1, 4, 4, 4)
    d, g = synth.depth_windows(11, 4, [0, 3, 6, 7], 6, 8, 3)
    assert d.shape == (4, 4, 6, 8) and g.shape == (4,)
