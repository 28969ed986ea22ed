"""Writes tests/golden/oracle_regression.json from the oracle alone (no CUDA path, no product import).

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import attention as oa          # noqa: E402
from oracle import block as ob              # noqa: E402
from oracle import chain as oc              # noqa: E402
from oracle import depth as od              # noqa: E402
from oracle import points as op             # noqa: E402
from oracle import render as orr            # noqa: E402


def poses_quadratic(n):
    """Camera moving along +z with z_t = 0.05 t^2 + 0.1 t and a slow yaw: world->camera [R | -R p]."""
    out = []
    for t in range(n):
        a = 0.01 * t
        c, s = np.cos(a), np.sin(a)
        r = np.array([[c, 0.0, -s], [0.0, 1.0, 0.0], [s, 0.0, c]])
        p = np.array([0.02 * t, 0.0, 0.05 * t * t + 0.1 * t])
        m = np.eye(4)
        m[:3, :3] = r
        m[:3, 3] = -r @ p
        out.append(m.tolist())
    return out


def build():
    rng = np.random.default_rng(20260107)
    q, k, v = (rng.standard_normal((1, 6, 2, 4)) for _ in range(3))
    o_g, lse_g = oa.window_attention(q, k, v, 2, 3, oa.GLOBAL)
    o_f, _ = oa.window_attention(q, k, v, 2, 3, oa.FRAME)
    poses = poses_quadratic(8)
    frames = op.motion_points(poses, 100.0, 100.0, 16.0, 12.0, 32, 24, 4, 3.0)
    m, g = orr.focus_map(frames[5]["points"], 32, 24, orr.NORM_MAX, np.full((24, 32), 2.0))
    loc = np.stack([np.array(poses[0:4]), np.array(poses[2:6]), np.array(poses[4:8])]).astype(np.float32)
    chained = np.array(oc.chain_poses(loc.tolist(), 4, 2, 8))
    x = rng.standard_normal((3, 8))
    up = orr.upsample_bilinear(rng.uniform(1.0, 9.0, (3, 4)), 10, 7)
    dloc = rng.uniform(1.0, 9.0, (3, 4, 2, 3))
    dloc[1] *= 0.5
    dloc[2] *= 3.0
    d_out, d_scales = od.align_depth(dloc, 4, 2, 8)
    return {
        "attention_global_o": np.round(o_g, 12).tolist(), "attention_global_lse": np.round(lse_g, 12).tolist(),
        "attention_frame_o_row0": np.round(o_f[0, 0], 12).tolist(),
        "focus_index": [f["focus_index"] for f in frames], "focus_uv_frame5": [float(u) for u in frames[5]["focus_uv"]],
        "focus_map_frame5_row12": np.round(m[12], 12).tolist(), "guided_depth_frame5_max": float(np.round(g.max(), 12)),
        "chain_last_pose": np.round(chained[-1], 12).tolist(),
        "gelu": np.round(ob.gelu(x[0]), 12).tolist(),
        "layernorm_row0": np.round(ob.layernorm(x, np.ones(8), np.zeros(8))[0], 12).tolist(),
        "round_bf16": ob.round_bf16(x[1]).tolist(),
        "upsample_bilinear_row3": np.round(up[3], 12).tolist(),
        "align_depth_scales": np.round(d_scales, 12).tolist(), "align_depth_last_frame": np.round(d_out[-1], 12).tolist(),
    }


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    with open(path, "w") as f:
        json.dump(build(), f, indent=1)
    print("wrote", path)
