"""Python binding of include/mf.h: argument marshalling only (ctypes).  Every step of the path
runs in the CUDA library; torch supplies device memory and the current stream.  There is no
fallback: a missing library or a non-sm_100 device raises."""
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmf_b200.so")

ATTN_GLOBAL, ATTN_FRAME = 0, 1
ALIGN_YAW_TRANSLATION, ALIGN_RIGID = 0, 1
VEC_ACCEL, VEC_VELOCITY = 0, 1
MAG_RAW, MAG_UNIT = 0, 1
NORM_MAX, NORM_SUM, NORM_NONE = 0, 1, 2
PTS_CURRENT_FRAME, PTS_OWN_FRAME = 0, 1
ACT_NONE, ACT_GELU = 0, 1

EXPORTS = ["mf_status_string", "mf_last_error", "mf_version", "mf_num_windows", "mf_window_start",
           "mf_window_attention", "mf_chain_poses", "mf_motion_focus_workspace_size", "mf_motion_focus",
           "mf_window_attention_host", "mf_chain_and_focus_host", "mf_linear", "mf_layernorm",
           "mf_block_workspace_size", "mf_block_forward", "mf_chain_state_size", "mf_chain_poses_step", "mf_motion_focus_upsampled",
           "mf_align_depth_workspace_size", "mf_align_depth",
           "mf_align_depth_state_size", "mf_align_depth_step", "mf_window_attention_noalloc"]


class MfError(RuntimeError):
    pass


class Intrinsics(ctypes.Structure):
    _fields_ = [("fx", ctypes.c_double), ("fy", ctypes.c_double), ("cx", ctypes.c_double), ("cy", ctypes.c_double)]


class BlockWeights(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in ("ln1_gamma", "ln1_beta", "w_qkv", "b_qkv", "w_o", "b_o", "ln2_gamma", "ln2_beta",
                                               "w_1", "b_1", "w_2", "b_2")]


class FocusParams(ctypes.Structure):
    _fields_ = [("n_points", ctypes.c_int), ("sigma", ctypes.c_float), ("vec", ctypes.c_int),
                ("mag", ctypes.c_int), ("norm", ctypes.c_int), ("pts", ctypes.c_int), ("eps_z", ctypes.c_double)]


_lib = None


def lib():
    """Loads libmf_b200.so (built by paper_2601_07154_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise MfError(f"{LIB_PATH} not found: run `python -m paper_2601_07154_b200.build` "
                          "(there is no CPU or PyTorch fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cf, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_double
        L.mf_status_string.restype = ctypes.c_char_p
        L.mf_status_string.argtypes = [ci]
        L.mf_last_error.restype = ctypes.c_char_p
        L.mf_version.restype = ci
        L.mf_num_windows.argtypes = [ci, ci, ci]
        L.mf_window_start.argtypes = [ci, ci, ci, ci]
        L.mf_window_attention.argtypes = [vp, vp, vp, vp, vp, ci, ci, ci, ci, ci, ci, cf, vp]
        L.mf_window_attention_noalloc.argtypes = L.mf_window_attention.argtypes
        L.mf_chain_poses.argtypes = [vp, ci, ci, ci, ci, ci, ci, vp, vp]
        L.mf_motion_focus_workspace_size.restype = ctypes.c_size_t
        L.mf_motion_focus_workspace_size.argtypes = [ci, ci, ci, ci]
        L.mf_motion_focus.argtypes = [vp, Intrinsics, ci, ci, ci, ci, ci, vp, ctypes.POINTER(FocusParams),
                                      vp, vp, vp, vp, vp, ctypes.c_size_t, vp]
        L.mf_window_attention_host.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, ci, ci, ci, cf, vp]
        L.mf_chain_and_focus_host.argtypes = [vp, ci, ci, ci, ci, ci, Intrinsics, ci, ci, ci, ci, vp,
                                              ctypes.POINTER(FocusParams), vp, vp, vp, vp, vp, vp]
        L.mf_linear.argtypes = [vp, vp, vp, vp, vp, vp, vp, ci, ci, ci, ci, ci, vp]
        L.mf_layernorm.argtypes = [vp, vp, vp, cf, vp, ci, ci, vp]
        L.mf_block_workspace_size.restype = ctypes.c_size_t
        L.mf_block_workspace_size.argtypes = [ci, ci, ci, ci, ci]
        L.mf_block_forward.argtypes = [vp, ctypes.POINTER(BlockWeights), vp, ci, ci, ci, ci, ci, ci, ci, cf, vp, ctypes.c_size_t, vp]
        L.mf_chain_state_size.restype = ctypes.c_size_t
        L.mf_chain_poses_step.argtypes = [vp, vp, ci, ci, ci, ci, vp, vp]
        L.mf_motion_focus_upsampled.argtypes = [vp, Intrinsics, ci, ci, ci, ci, ci, vp, ci, ci, ctypes.POINTER(FocusParams),
                                                vp, vp, vp, vp, vp, ctypes.c_size_t, vp]
        L.mf_align_depth_workspace_size.restype = ctypes.c_size_t
        L.mf_align_depth_workspace_size.argtypes = [ci]
        L.mf_align_depth.argtypes = [vp, ci, ci, ci, ci, ci, ci, vp, vp, vp, ctypes.c_size_t, vp]
        L.mf_align_depth_state_size.restype = ctypes.c_size_t
        L.mf_align_depth_step.argtypes = [vp, vp, vp, ci, ci, ci, ci, ci, vp, vp]
        _lib = L
    return _lib


def _check(status):
    if status != 0:
        L = lib()
        raise MfError(f"{L.mf_status_string(status).decode()}: {L.mf_last_error().decode()}")


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(0 if t is None else t.data_ptr())


def _dev(t, dtype, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise MfError(f"{name}: expected a contiguous CUDA tensor of {dtype}")
    return t


def num_windows(num_frames, w, stride):
    return lib().mf_num_windows(num_frames, w, stride)


def window_start(num_frames, w, stride, n):
    return lib().mf_window_start(num_frames, w, stride, n)


def window_starts(num_frames, w, stride):
    """[mf_window_start(n) for every window] (host arithmetic of the library, no device needed)."""
    L = lib()
    nw = L.mf_num_windows(num_frames, w, stride)
    if nw < 0:
        raise MfError("window_starts: need num_frames >= W > stride >= 1")
    return [L.mf_window_start(num_frames, w, stride, n) for n in range(nw)]


def window_attention(q, k, v, frames_per_window, tokens_per_frame, mode=ATTN_GLOBAL, softmax_scale=0.0,
                     out=None, return_lse=False, noalloc=False):
    """q,k,v: bf16 CUDA [windows, S, H, D] with S = frames_per_window*tokens_per_frame.  noalloc=True calls
    mf_window_attention_noalloc (static scratch inside the library, include/mf.h); pass `out` as well if this
    binding must not create a tensor either."""
    for name, t in (("q", q), ("k", k), ("v", v)):
        _dev(t, torch.bfloat16, name)
    if q.dim() != 4 or k.shape != q.shape or v.shape != q.shape:
        raise MfError("q, k, v must share the shape [windows, S, H, D]")
    windows, s_len, heads, dim = q.shape
    if s_len != frames_per_window * tokens_per_frame:
        raise MfError("S != frames_per_window * tokens_per_frame")
    if out is None:
        out = torch.empty_like(q)
    _dev(out, torch.bfloat16, "out")
    lse = torch.empty((windows, heads, s_len), device=q.device, dtype=torch.float32) if return_lse else None
    fn = lib().mf_window_attention_noalloc if noalloc else lib().mf_window_attention
    _check(fn(_ptr(q), _ptr(k), _ptr(v), _ptr(out), _ptr(lse), windows, frames_per_window, tokens_per_frame, heads, dim, mode,
              float(softmax_scale), _stream()))
    return (out, lse) if return_lse else out


def chain_poses(local_w2c, stride, num_frames, mode=ALIGN_YAW_TRANSLATION):
    """local_w2c: fp32 CUDA [sequences, num_windows, W, 4, 4] (or 4-D for one sequence) -> fp64 [.., N, 4, 4]."""
    _dev(local_w2c, torch.float32, "local_w2c")
    squeeze = local_w2c.dim() == 4
    x = local_w2c.unsqueeze(0) if squeeze else local_w2c
    if x.dim() != 5 or x.shape[-2:] != (4, 4):
        raise MfError("local_w2c must be [sequences, num_windows, W, 4, 4]")
    seqs, nw, w = x.shape[:3]
    out = torch.empty((seqs, num_frames, 4, 4), device=x.device, dtype=torch.float64)
    _check(lib().mf_chain_poses(_ptr(x), seqs, nw, w, stride, num_frames, mode, _ptr(out), _stream()))
    return out[0] if squeeze else out


def align_depth(depth_local, stride, num_frames, workspace=None, out=None):
    """depth_local: fp32 CUDA [num_windows, W, h, w], each window in its own scale -> (depth fp32 [N, h, w], c_n fp64 [Nw])."""
    _dev(depth_local, torch.float32, "depth_local")
    if depth_local.dim() != 4:
        raise MfError("depth_local must be [num_windows, W, height, width]")
    nw, w, h, wd = depth_local.shape
    need = lib().mf_align_depth_workspace_size(nw)
    if workspace is None:
        workspace = torch.empty((need,), device=depth_local.device, dtype=torch.uint8)
    if out is None:
        out = torch.empty((num_frames, h, wd), device=depth_local.device, dtype=torch.float32)
    else:
        _dev(out, torch.float32, "out")
    scales = torch.empty((nw,), device=depth_local.device, dtype=torch.float64)
    _check(lib().mf_align_depth(_ptr(depth_local), nw, w, stride, num_frames, h, wd, _ptr(out), _ptr(scales), _ptr(workspace),
                                workspace.numel(), _stream()))
    return out, scales


def align_depth_state(device="cuda"):
    """Device-resident state of the streaming depth alignment (mf_align_depth_step)."""
    return torch.zeros((lib().mf_align_depth_state_size(),), device=device, dtype=torch.uint8)


def align_depth_step(cur_window, state, prev_window=None, new_frames=0, first=False, out=None):
    """One window [W, h, w] fp32 through the depth scale chain; returns the emitted frames fp32 [n, h, w]."""
    _dev(cur_window, torch.float32, "cur_window")
    if prev_window is not None:
        _dev(prev_window, torch.float32, "prev_window")
    w, h, wd = cur_window.shape
    n = w if first else new_frames
    if out is None:
        out = torch.empty((max(n, 0), h, wd), device=cur_window.device, dtype=torch.float32)
    _check(lib().mf_align_depth_step(_ptr(prev_window), _ptr(cur_window), _ptr(state), w, new_frames, 1 if first else 0, h, wd,
                                     _ptr(out), _stream()))
    return out


def focus_params(n_points=15, sigma=20.0, vec=VEC_ACCEL, mag=MAG_UNIT, norm=NORM_MAX, pts=PTS_CURRENT_FRAME,
                 eps_z=1e-6):
    return FocusParams(n_points, sigma, vec, mag, norm, pts, eps_z)


def motion_focus(global_w2c, fx, fy, cx, cy, width, height, params=None, depth=None, render_begin=0,
                 render_end=None, want_map=True, want_guided=None, workspace=None, out=None):
    """global_w2c: fp64 CUDA [N,4,4].  Returns dict(focus_map, guided_depth, focus_uv, focus_index)."""
    _dev(global_w2c, torch.float64, "global_w2c")
    n = global_w2c.shape[0]
    render_end = n if render_end is None else render_end
    count = render_end - render_begin
    params = focus_params() if params is None else params
    dev = global_w2c.device
    if depth is not None:
        _dev(depth, torch.float32, "depth")
        if tuple(depth.shape) != (count, height, width):
            raise MfError("depth must be [count, height, width]")
    want_guided = (depth is not None) if want_guided is None else want_guided
    out = {} if out is None else out
    fmap = out.get("focus_map")
    if want_map and fmap is None:
        fmap = torch.empty((max(count, 0), height, width), device=dev, dtype=torch.float32)
    guided = out.get("guided_depth")
    if want_guided and guided is None:
        guided = torch.empty((max(count, 0), height, width), device=dev, dtype=torch.float32)
    uv = torch.empty((max(count, 0), 2), device=dev, dtype=torch.float32)
    idx = torch.empty((max(count, 0),), device=dev, dtype=torch.int32)
    need = lib().mf_motion_focus_workspace_size(count, width, height, params.n_points)
    if workspace is None or workspace.numel() < need:
        workspace = torch.empty((max(need, 16),), device=dev, dtype=torch.uint8)
    _check(lib().mf_motion_focus(_ptr(global_w2c), Intrinsics(fx, fy, cx, cy), n, render_begin, render_end,
                                 width, height, _ptr(depth), ctypes.byref(params), _ptr(fmap), _ptr(guided),
                                 _ptr(uv), _ptr(idx), _ptr(workspace), workspace.numel(), _stream()))
    return {"focus_map": fmap, "guided_depth": guided, "focus_uv": uv, "focus_index": idx,
            "workspace": workspace}


def motion_focus_upsampled(global_w2c, fx, fy, cx, cy, width, height, depth_lowres, params=None, render_begin=0,
                           render_end=None, workspace=None, out=None):
    """mf_motion_focus_upsampled: depth_lowres fp32 CUDA [count, h_lo, w_lo] is interpolated (bilinear, half-pixel centres)
    to width x height inside the render pass.  Returns dict(focus_map, guided_depth, focus_uv, focus_index)."""
    _dev(global_w2c, torch.float64, "global_w2c")
    _dev(depth_lowres, torch.float32, "depth_lowres")
    n = global_w2c.shape[0]
    render_end = n if render_end is None else render_end
    count = render_end - render_begin
    if depth_lowres.dim() != 3 or depth_lowres.shape[0] != count:
        raise MfError("depth_lowres must be [count, h_lo, w_lo]")
    params = focus_params() if params is None else params
    dev = global_w2c.device
    out = {} if out is None else out
    fmap = out.get("focus_map")
    if fmap is None:
        fmap = torch.empty((count, height, width), device=dev, dtype=torch.float32)
    guided = out.get("guided_depth")
    if guided is None:
        guided = torch.empty((count, height, width), device=dev, dtype=torch.float32)
    uv = torch.empty((count, 2), device=dev, dtype=torch.float32)
    idx = torch.empty((count,), device=dev, dtype=torch.int32)
    need = lib().mf_motion_focus_workspace_size(count, width, height, params.n_points)
    if workspace is None or workspace.numel() < need:
        workspace = torch.empty((max(need, 16),), device=dev, dtype=torch.uint8)
    _check(lib().mf_motion_focus_upsampled(_ptr(global_w2c), Intrinsics(fx, fy, cx, cy), n, render_begin, render_end, width,
                                           height, _ptr(depth_lowres), depth_lowres.shape[2], depth_lowres.shape[1],
                                           ctypes.byref(params), _ptr(fmap), _ptr(guided), _ptr(uv), _ptr(idx), _ptr(workspace),
                                           workspace.numel(), _stream()))
    return {"focus_map": fmap, "guided_depth": guided, "focus_uv": uv, "focus_index": idx, "workspace": workspace}


# ---- host-buffer entry points (end-to-end path) ---------------------------------------------------

def _host(t, dtype, name):
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise MfError(f"{name}: expected a contiguous CPU tensor of {dtype}")
    return t


def window_attention_host(q, k, v, frames_per_window, tokens_per_frame, mode=ATTN_GLOBAL, softmax_scale=0.0,
                          out=None, num_layers=1):
    for name, t in (("q", q), ("k", k), ("v", v)):
        _host(t, torch.bfloat16, name)
    windows, s_len, heads, dim = q.shape
    if out is None:
        out = torch.empty_like(q)
    _check(lib().mf_window_attention_host(_ptr(q), _ptr(k), _ptr(v), _ptr(out), windows, frames_per_window,
                                          tokens_per_frame, heads, dim, num_layers, mode, float(softmax_scale),
                                          _stream()))
    return out


def chain_and_focus_host(local_w2c, stride, num_frames, fx, fy, cx, cy, width, height, params=None, depth=None,
                         render_begin=0, render_end=None, align=ALIGN_YAW_TRANSLATION, out=None):
    _host(local_w2c, torch.float32, "local_w2c")
    nw, w = local_w2c.shape[:2]
    render_end = num_frames if render_end is None else render_end
    count = render_end - render_begin
    params = focus_params() if params is None else params
    out = {} if out is None else out
    pin = torch.cuda.is_available()
    mk = lambda shape, dt: torch.empty(shape, dtype=dt, pin_memory=pin)
    poses = out.get("global_w2c") if "global_w2c" in out else mk((num_frames, 4, 4), torch.float64)
    fmap = out.get("focus_map") if "focus_map" in out else mk((count, height, width), torch.float32)
    guided = None
    if depth is not None:
        _host(depth, torch.float32, "depth")
        guided = out.get("guided_depth") if "guided_depth" in out else mk((count, height, width), torch.float32)
    uv = mk((count, 2), torch.float32)
    idx = mk((count,), torch.int32)
    _check(lib().mf_chain_and_focus_host(_ptr(local_w2c), nw, w, stride, num_frames, align,
                                         Intrinsics(fx, fy, cx, cy), render_begin, render_end, width, height,
                                         _ptr(depth), ctypes.byref(params), _ptr(poses), _ptr(fmap), _ptr(guided),
                                         _ptr(uv), _ptr(idx), _stream()))
    return {"global_w2c": poses, "focus_map": fmap, "guided_depth": guided, "focus_uv": uv, "focus_index": idx}


def linear(x, w, bias=None, residual=None, act=ACT_NONE, splits=1, out=None):
    """out = act(x w^T + bias) (+ residual).  x bf16 [M,K], w bf16 [N,K]; `splits` = 1 or 3 output tensors
    [M, N/splits] (3: q | k | v).  Returns a tensor (splits == 1) or a tuple of tensors."""
    _dev(x, torch.bfloat16, "x")
    _dev(w, torch.bfloat16, "w")
    if x.dim() != 2 or w.dim() != 2 or x.shape[1] != w.shape[1]:
        raise MfError("linear: x [M,K] and w [N,K] expected")
    m, k = x.shape
    n = w.shape[0]
    if n % splits:
        raise MfError("linear: N not divisible by splits")
    if bias is not None:
        _dev(bias, torch.float32, "bias")
    if residual is not None:
        _dev(residual, torch.bfloat16, "residual")
    outs = list(out) if out is not None else [torch.empty((m, n // splits), device=x.device, dtype=torch.bfloat16)
                                              for _ in range(splits)]
    for o in outs:
        _dev(o, torch.bfloat16, "out")
    o3 = outs + [None] * (3 - len(outs))
    _check(lib().mf_linear(_ptr(x), _ptr(w), _ptr(bias), _ptr(residual), _ptr(o3[0]), _ptr(o3[1]), _ptr(o3[2]), m, n, k,
                           n // splits, act, _stream()))
    return outs[0] if splits == 1 else tuple(outs)


def layernorm(x, gamma, beta, eps=1e-6, out=None):
    _dev(x, torch.bfloat16, "x")
    _dev(gamma, torch.float32, "gamma")
    _dev(beta, torch.float32, "beta")
    if out is None:
        out = torch.empty_like(x)
    _dev(out, torch.bfloat16, "out")
    _check(lib().mf_layernorm(_ptr(x), _ptr(gamma), _ptr(beta), float(eps), _ptr(out), x.shape[0], x.shape[1], _stream()))
    return out


_BLOCK_KEYS = ("ln1_g", "ln1_b", "w_qkv", "b_qkv", "w_o", "b_o", "ln2_g", "ln2_b", "w_1", "b_1", "w_2", "b_2")


def block_forward(x, wts, windows, frames_per_window, tokens_per_frame, heads, mode=ATTN_GLOBAL, ln_eps=1e-6,
                  out=None, workspace=None):
    """One pre-norm transformer block (mf_block_forward).  x bf16 [windows*W*P, d]; wts: dict with the keys of
    _BLOCK_KEYS (bf16 matrices, fp32 vectors, biases may be None)."""
    _dev(x, torch.bfloat16, "x")
    d = x.shape[1]
    d_hidden = wts["w_1"].shape[0]
    need = lib().mf_block_workspace_size(windows, frames_per_window, tokens_per_frame, d, d_hidden)
    if workspace is None:
        workspace = torch.empty((need,), device=x.device, dtype=torch.uint8)
    if out is None:
        out = torch.empty_like(x)
    bw = BlockWeights(*[0 if wts.get(k) is None else wts[k].data_ptr() for k in _BLOCK_KEYS])
    _check(lib().mf_block_forward(_ptr(x), ctypes.byref(bw), _ptr(out), windows, frames_per_window, tokens_per_frame, heads,
                                  d // heads, d_hidden, mode, float(ln_eps), _ptr(workspace), workspace.numel(), _stream()))
    return out


def chain_state(device="cuda"):
    """Device-resident state of the streaming pose chain (mf_chain_poses_step)."""
    return torch.zeros((lib().mf_chain_state_size(),), device=device, dtype=torch.uint8)


def chain_poses_step(window_local_w2c, state, new_frames=0, first=False, mode=ALIGN_YAW_TRANSLATION, out=None):
    """One window [W,4,4] fp32 through the incremental anchoring; returns the emitted global poses fp64 [n,4,4]."""
    _dev(window_local_w2c, torch.float32, "window_local_w2c")
    w = window_local_w2c.shape[0]
    n = w if first else new_frames
    if out is None:
        out = torch.empty((max(n, 0), 4, 4), device=window_local_w2c.device, dtype=torch.float64)
    _check(lib().mf_chain_poses_step(_ptr(window_local_w2c), _ptr(state), w, int(new_frames), 1 if first else 0, mode, _ptr(out),
                                     _stream()))
    return out
