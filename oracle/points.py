"""Oracle: motion points, Eq. 1-6, and the focus pixel.

  Eq.1  p_t = (T_t^{w->c})^{-1}[1:3,4] = -R_t^T t_t     camera centre
  Eq.2-3  a_w = (p_t - p_{t-1}) - (p_{t-1} - p_{t-2})
  Eq.4  a_c = R_tau a_w
  Eq.6  u = c_x + f_x (a_x / a_z),  v = c_y + f_y (a_y / a_z)
  P:131-137     N motion points per map, spread sigma * s_i (s_i = motion magnitude)

Readings C1-C10: ACCEL is the paper's mode, VELOCITY (P:125's
contrast, a_w := p_t - p_{t-1}) is a flag; the map of frame t aggregates the
trailing n_points frames i = t-n_points+1..t, rotated by R_t (CURRENT_FRAME)
or R_i (OWN_FRAME); a point is invalid when it needs a frame < 0, when
|a_w| < 1e-12 or when |a_z| <= eps_z |a_c|; the focus pixel is
(floor(u+0.5), floor(v+0.5)) of the frame's own point, index y*width + x or -1.

fp64 Python floats, only + - * / sqrt, one rounding per operation, dot products
left to right (shared *convention* with chain.py, which supplies dot3).  The
hand-off values (u, v, sigma_i) are rounded once to fp32 (C-def-8).
TEST INFRASTRUCTURE ONLY.
"""
import math

import numpy as np

from .chain import dot3, from_4x4

ACCEL, VELOCITY = 0, 1
MAG_RAW, MAG_UNIT = 0, 1
PTS_CURRENT_FRAME, PTS_OWN_FRAME = 0, 1
SIGMA_MIN = 1e-3          # reading D6
A_W_MIN = 1e-12           # C-def-6


def centre(pose):
    """Eq. 1: p = -R^T t."""
    r, t = pose
    return [-dot3(r[0][i], r[1][i], r[2][i], t[0], t[1], t[2]) for i in range(3)]


def norm3(a):
    return math.sqrt(((a[0] * a[0]) + (a[1] * a[1])) + (a[2] * a[2]))


def world_vector(centres, i, vec):
    """Eq. 2-3 (ACCEL) or the velocity variant; None if it needs a frame < 0."""
    if vec == ACCEL:
        if i < 2:
            return None
        return [(centres[i][c] - centres[i - 1][c]) - (centres[i - 1][c] - centres[i - 2][c])
                for c in range(3)]
    if i < 1:
        return None
    return [centres[i][c] - centres[i - 1][c] for c in range(3)]


def project(a_w, rot, fx, fy, cx, cy, sigma, mag, eps_z):
    """Eq. 4 + Eq. 6 + spread.  Returns (u, v, sigma_i) in fp64 or None if invalid."""
    if a_w is None:
        return None
    s = norm3(a_w)
    if s < A_W_MIN:
        return None
    a_c = [dot3(rot[i][0], rot[i][1], rot[i][2], a_w[0], a_w[1], a_w[2]) for i in range(3)]
    n_c = norm3(a_c)
    if abs(a_c[2]) <= eps_z * n_c:
        return None
    u = cx + (fx * (a_c[0] / a_c[2]))
    v = cy + (fy * (a_c[1] / a_c[2]))
    sig = (sigma * s) if mag == MAG_RAW else sigma
    if sig < SIGMA_MIN:
        sig = SIGMA_MIN
    return u, v, sig


def motion_points(global_w2c, fx, fy, cx, cy, width, height, n_points, sigma,
                  vec=ACCEL, mag=MAG_UNIT, pts=PTS_CURRENT_FRAME, eps_z=1e-6,
                  render_begin=0, render_end=None):
    """global_w2c: sequence of num_frames 4x4 fp64.

    Returns per rendered frame t a dict:
      points       list of (u, v, sigma_i) np.float32 triples (valid points only,
                   oldest first)
      focus_uv     (np.float32 u, np.float32 v) of the frame's own point, NaN if invalid
      focus_index  int, y*width + x, or -1
      focus_uv64   the same point before rounding to fp32 (Python floats), None if invalid
    """
    sigma = float(np.float32(sigma))                      # the API carries sigma as fp32
    poses = [from_4x4(m) for m in global_w2c]
    centres = [centre(p) for p in poses]
    render_end = len(poses) if render_end is None else render_end
    frames = []
    for t in range(render_begin, render_end):
        pts_t = []
        own = None
        for i in range(t - n_points + 1, t + 1):
            if i < 0:
                continue
            rot = poses[t][0] if pts == PTS_CURRENT_FRAME else poses[i][0]
            pr = project(world_vector(centres, i, vec), rot, fx, fy, cx, cy, sigma, mag, eps_z)
            if i == t:
                own = pr
            if pr is not None:
                pts_t.append((np.float32(pr[0]), np.float32(pr[1]), np.float32(pr[2])))
        if own is None:
            uv = (np.float32("nan"), np.float32("nan"))
            index = -1
        else:
            uv = (np.float32(own[0]), np.float32(own[1]))
            x = math.floor(own[0] + 0.5) if math.isfinite(own[0]) else -1
            y = math.floor(own[1] + 0.5) if math.isfinite(own[1]) else -1
            index = y * width + x if (0 <= x < width and 0 <= y < height) else -1
        frames.append({"points": pts_t, "focus_uv": uv, "focus_index": index,
                       "focus_uv64": None if own is None else (own[0], own[1])})    # unrounded (u, v): near-tie reports only
    return frames
