"""Seeded synthetic inputs shaped like the paper's clips (Table 1) and
BASELINE.json's configs.  This module serves BOTH the oracle-side tests and the
CUDA path's tests/bench; it holds none of the method's arithmetic (no attention,
no anchoring, no projection, no rendering) -- only random tokens, a random
camera trajectory cut into window-local poses, and random depth.

The paper's dataset and DA3's weights are not available; these inputs stand in
for them (recipe in DESIGN.md "Input recipe").
"""
import math

import numpy as np

BASE_SEED = 260107154

# BASELINE.json configs[0..4].  P = tokens/frame, N = frames in the clip.
CONFIGS = [
    dict(name="tiny", W=4, stride=2, N=4, P=256, H=16, D=64, layers=1,
         width=224, height=224, fx=200.0, fy=200.0, cx=112.0, cy=112.0, fps=30,
         step=0.1, step_sd=0.02, rot_sd=0.05, head_yaw_sd=0.0, sigma=20.0),
    dict(name="suburban", W=8, stride=4, N=240, P=777, H=16, D=64, layers=24,
         width=960, height=544, fx=700.0, fy=700.0, cx=480.0, cy=272.0, fps=30,
         step=0.047, step_sd=0.01, rot_sd=0.02, head_yaw_sd=0.05, sigma=20.0),
    dict(name="city", W=16, stride=8, N=600, P=777, H=16, D=64, layers=24,
         width=1920, height=1080, fx=1400.0, fy=1400.0, cx=960.0, cy=540.0, fps=30,
         step=0.047, step_sd=0.01, rot_sd=0.02, head_yaw_sd=0.15, sigma=20.0),
    dict(name="campus", W=32, stride=16, N=1800, P=777, H=16, D=64, layers=24,
         width=1920, height=1080, fx=1400.0, fy=1400.0, cx=960.0, cy=540.0, fps=60,
         step=0.08, step_sd=0.01, rot_sd=0.1, head_yaw_sd=0.0, sigma=20.0),
    dict(name="town", W=64, stride=32, N=720, P=777, H=16, D=64, layers=24,
         width=3840, height=2160, fx=2800.0, fy=2800.0, cx=1920.0, cy=1080.0, fps=30,
         step=0.047, step_sd=0.01, rot_sd=0.02, head_yaw_sd=0.05, sigma=20.0),
    # Not a BASELINE.json config: the shape of the paper's own Table 2 row "DA3 Base, res 504, batch 60" as a second
    # workload.  504 px at 16:9 with 14-px patches -> 36 x 20 = 720 tokens/frame; ViT-B widths
    # (12 heads x 64, 12 blocks) are an ASSUMPTION about DA3 Base, not stated in PAPER.md; overlap W/2 as in BJ.
    dict(name="table2-base-504-b60", W=60, stride=30, N=600, P=720, H=12, D=64, layers=12,
         width=1920, height=1080, fx=1400.0, fy=1400.0, cx=960.0, cy=540.0, fps=30,
         step=0.047, step_sd=0.01, rot_sd=0.02, head_yaw_sd=0.15, sigma=20.0),
]

# The other six rows of the paper's Table 2 as workloads 6..11, same recipe as workload 5.  Resolution 384 at 16:9 with
# 14-px patches -> 27 x 15 = 405 tokens/frame; "DA3 Small" is taken as ViT-S widths (6 heads x 64, 12 blocks): like the ViT-B
# widths of "DA3 Base" an ASSUMPTION, not stated in PAPER.md.  Batch size = window W, overlap W/2.
def _table2(name, w, p, heads):
    return dict(name=name, W=w, stride=w // 2, N=600, P=p, H=heads, D=64, layers=12,
                width=1920, height=1080, fx=1400.0, fy=1400.0, cx=960.0, cy=540.0, fps=30,
                step=0.047, step_sd=0.01, rot_sd=0.02, head_yaw_sd=0.15, sigma=20.0)


CONFIGS += [_table2("table2-base-384-b60", 60, 405, 12), _table2("table2-base-384-b30", 30, 405, 12),
            _table2("table2-small-504-b60", 60, 720, 6), _table2("table2-small-384-b60", 60, 405, 6),
            _table2("table2-small-504-b30", 30, 720, 6), _table2("table2-small-384-b30", 30, 405, 6)]


def seed_for(config_index, stream):
    return BASE_SEED + 1000 * config_index + stream


def qkv(windows, s_len, heads, dim, seed, device="cpu", scale=1.0):
    """Three bf16 tensors [windows, S, H, D] ~ N(0, scale^2), seeded."""
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    out = []
    for _ in range(3):
        t = torch.randn((windows, s_len, heads, dim), generator=g, device=device,
                        dtype=torch.float32)
        out.append((t * scale).to(torch.bfloat16))
    return out


def _rot(axis, a):
    c, s = math.cos(a), math.sin(a)
    if axis == 0:
        return np.array([[1, 0, 0], [0, c, -s], [0, s, c]], dtype=np.float64)
    if axis == 1:
        return np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]], dtype=np.float64)
    return np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]], dtype=np.float64)


def trajectory(cfg, seed, num_frames=None):
    """World->camera poses [N,4,4] fp64 of a walking / riding camera.

    OpenCV axes (x right, y down, z forward).  The body heading is a random walk
    about Y; the camera adds head yaw and pitch/roll noise; each frame advances
    `step + N(0, step_sd)` metres along the body heading (tiny config: along the
    camera's own z axis).
    """
    n = cfg["N"] if num_frames is None else num_frames
    rng = np.random.default_rng(seed)
    pos = np.zeros(3)
    heading = 0.0
    out = np.zeros((n, 4, 4), dtype=np.float64)
    for t in range(n):
        if cfg["name"] == "tiny":
            ax, ay, az = rng.normal(0.0, cfg["rot_sd"], 3)
            r_c2w = _rot(1, ay) @ _rot(0, ax) @ _rot(2, az)
            fwd = r_c2w[:, 2]
        else:
            heading += rng.normal(0.0, 0.02)
            yaw = heading + rng.normal(0.0, cfg["head_yaw_sd"]) + rng.normal(0.0, cfg["rot_sd"])
            pitch, roll = rng.normal(0.0, cfg["rot_sd"], 2)
            r_c2w = _rot(1, yaw) @ _rot(0, pitch) @ _rot(2, roll)
            fwd = _rot(1, heading)[:, 2]
        pos = pos + fwd * (cfg["step"] + rng.normal(0.0, cfg["step_sd"]))
        out[t, :3, :3] = r_c2w.T
        out[t, :3, 3] = -r_c2w.T @ pos
        out[t, 3, 3] = 1.0
    return out


def local_windows(global_w2c, w, starts, seed=None, perturb_rot=0.0, perturb_t=0.0):
    """Cut a trajectory into window-local poses, fp32 [len(starts), W, 4, 4].

    `starts` = the first frame of every window.  The caller supplies it (the window partition is step a1 of the
    method: tests take it from oracle/windows.py, bench.py and smoke() from mf_window_start), so this
    module holds none of the method's arithmetic.

    Window n's local world is its own first camera (6-DoF gauge).  Optional
    per-frame perturbation makes overlapping estimates disagree like a real
    model's would.
    """
    starts = list(starts)
    rng = np.random.default_rng(seed)
    out = np.zeros((len(starts), w, 4, 4), dtype=np.float32)
    for i, s0 in enumerate(starts):
        gauge = np.linalg.inv(global_w2c[s0])
        for k in range(w):
            m = global_w2c[s0 + k] @ gauge
            if perturb_rot > 0.0 or perturb_t > 0.0:
                e = np.eye(4)
                a = rng.normal(0.0, perturb_rot, 3)
                e[:3, :3] = _rot(1, a[1]) @ _rot(0, a[0]) @ _rot(2, a[2])
                e[:3, 3] = rng.normal(0.0, perturb_t, 3)
                m = e @ m
            out[i, k] = m.astype(np.float32)
    return out


def depth(frames, height, width, seed, device="cpu"):
    """fp32 depth ~ Uniform(1, 30) m, [frames, height, width]."""
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return torch.rand((frames, height, width), generator=g, device=device,
                      dtype=torch.float32) * 29.0 + 1.0


def depth_windows(num_frames, w, starts, height, width, seed, gauge_spread=2.0, noise=0.02, invalid=0.0):
    """Window-local depth maps, fp32 numpy [Nw, W, height, width]: one Uniform(1, 30) m stream, cut into windows at the
    caller-supplied `starts` (see local_windows), each window
    divided by its own scale (log-uniform in [1/gauge_spread, gauge_spread]) and multiplied by per-pixel noise
    (1 + noise * N(0,1)), so that overlapping estimates disagree like a model's would.  A fraction `invalid` of the pixels is
    replaced by 0, NaN or inf (sky / holes).  Returns (depth_local, gauges)."""
    rng = np.random.default_rng(seed)
    stream = rng.uniform(1.0, 30.0, (num_frames, height, width))
    starts = list(starts)
    gauges = np.exp(rng.uniform(-np.log(gauge_spread), np.log(gauge_spread), len(starts)))
    out = np.empty((len(starts), w, height, width), dtype=np.float32)
    for i, s0 in enumerate(starts):
        d = stream[s0:s0 + w] / gauges[i] * (1.0 + noise * rng.standard_normal((w, height, width)))
        if invalid > 0.0:
            bad = rng.uniform(size=d.shape) < invalid
            d[bad] = rng.choice(np.array([0.0, np.nan, np.inf, -1.0]), size=int(bad.sum()))
        out[i] = d.astype(np.float32)
    return out, gauges


def tokens(m, d, seed, device="cpu"):
    """Activations ~ N(0,1) rounded to bf16, [m, d]."""
    import torch
    g = torch.Generator(device=device).manual_seed(int(seed))
    return torch.randn((m, d), generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)


def linear_inputs(m, n, k, seed, device="cpu"):
    """Seeded synthetic dense layer: x ~ N(0,1) bf16 [m,k]; w ~ N(0, 1/k) bf16 [n,k] (so x w^T ~ N(0,1)); bias ~ N(0, 0.1) fp32 [n].
    Stand-in for trained weights, which are not available."""
    import torch
    g = torch.Generator(device=device).manual_seed(int(seed))
    x = torch.randn((m, k), generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
    w = (torch.randn((n, k), generator=g, device=device, dtype=torch.float32) / (k ** 0.5)).to(torch.bfloat16)
    b = 0.1 * torch.randn((n,), generator=g, device=device, dtype=torch.float32)
    return x, w, b


def block_weights(d, d_hidden, seed, device="cpu"):
    """Seeded synthetic weights of one pre-norm block (stand-in for trained weights): matrices ~ N(0, 1/fan_in) bf16,
    biases ~ N(0, 0.1) fp32, LayerNorm gamma ~ 1 + N(0, 0.1), beta ~ N(0, 0.1) fp32."""
    import torch
    g = torch.Generator(device=device).manual_seed(int(seed))
    rn = lambda *shape: torch.randn(shape, generator=g, device=device, dtype=torch.float32)
    mat = lambda n, k: (rn(n, k) / (k ** 0.5)).to(torch.bfloat16)
    return dict(ln1_g=1 + 0.1 * rn(d), ln1_b=0.1 * rn(d), w_qkv=mat(3 * d, d), b_qkv=0.1 * rn(3 * d), w_o=mat(d, d),
                b_o=0.1 * rn(d), ln2_g=1 + 0.1 * rn(d), ln2_b=0.1 * rn(d), w_1=mat(d_hidden, d), b_1=0.1 * rn(d_hidden),
                w_2=mat(d, d_hidden), b_2=0.1 * rn(d))
