"""Oracle: focus map, Eq. 7, and motion-guided depth (Fig. 1(iii), Fig. 5).

  M(u,v) = (1/Z) sum_i exp( -((u-u_i)^2 + (v-v_i)^2) / (2 (sigma s_i)^2) )

Brute force over every pixel and every point in fp64 (NOT the separable form a
GPU would use).  Pixel (x, y) is centred at (u, v) = (x, y) (reading C7).
Readings D1-D6: Z = per-frame max over the image's pixels (MAX,
default), sum (SUM) or 1 (NONE); Z = 0 -> M = 0; guided depth G = M * D.
Inputs are the fp32 (u_i, v_i, sigma_i) of points.py promoted exactly.
TEST INFRASTRUCTURE ONLY.
"""
import numpy as np

NORM_MAX, NORM_SUM, NORM_NONE = 0, 1, 2


def unnormalised(points, width, height):
    """U(x,y) = sum_i exp(-((x-u_i)^2+(y-v_i)^2)/(2 sigma_i^2)), fp64 [height, width]."""
    x = np.arange(width, dtype=np.float64)[None, :]
    y = np.arange(height, dtype=np.float64)[:, None]
    u_map = np.zeros((height, width), dtype=np.float64)
    for (u, v, sig) in points:
        u, v, sig = float(u), float(v), float(sig)
        dx = x - u
        dy = y - v
        u_map += np.exp(-((dx * dx) + (dy * dy)) / (2.0 * sig * sig))
    return u_map


def focus_map(points, width, height, norm=NORM_MAX, depth=None):
    """Returns (M, G): fp64 [height, width]; G is None when depth is None."""
    u_map = unnormalised(points, width, height)
    if norm == NORM_MAX:
        z = float(u_map.max()) if len(points) else 0.0
    elif norm == NORM_SUM:
        z = float(u_map.sum())
    else:
        z = 1.0
    m = u_map / z if z > 0.0 else np.zeros_like(u_map)
    g = None if depth is None else m * np.asarray(depth, dtype=np.float64)
    return m, g


def brute_force_pixel(points, x, y):
    """Pure-Python single pixel of U, for the pins."""
    import math
    return sum(math.exp(-(((x - float(u)) ** 2) + ((y - float(v)) ** 2)) / (2.0 * float(s) * float(s)))
               for (u, v, s) in points)


def upsample_bilinear(depth_lo, width, height):
    """Reading F1 (the paper is silent on how the model-resolution depth reaches the focus-map
    resolution, B7/D4): bilinear interpolation with half-pixel centres and edge clamping, i.e. what
    torch.nn.functional.interpolate(mode="bilinear", align_corners=False) computes.  For output column x of `width`
    from an input row of w_lo samples: src = max(0, (x + 1/2) w_lo / width - 1/2), x0 = floor(src),
    x1 = min(x0 + 1, w_lo - 1), lambda = src - x0; the same along y; D = (1-ly)((1-lx) d00 + lx d01) + ly((1-lx) d10 + lx d11).
    depth_lo [h_lo, w_lo] -> fp64 [height, width].  Plain loops over the output axes, no library interpolation."""
    d = np.asarray(depth_lo, dtype=np.float64)
    h_lo, w_lo = d.shape

    def taps(n_out, n_in):
        i0, i1, lam = [], [], []
        for o in range(n_out):
            src = max(0.0, (o + 0.5) * n_in / n_out - 0.5)
            a = int(np.floor(src))
            a = min(a, n_in - 1)
            i0.append(a)
            i1.append(min(a + 1, n_in - 1))
            lam.append(src - a)
        return np.array(i0), np.array(i1), np.array(lam, dtype=np.float64)

    x0, x1, lx = taps(width, w_lo)
    y0, y1, ly = taps(height, h_lo)
    top = d[y0][:, x0] * (1.0 - lx)[None, :] + d[y0][:, x1] * lx[None, :]
    bot = d[y1][:, x0] * (1.0 - lx)[None, :] + d[y1][:, x1] * lx[None, :]
    return top * (1.0 - ly)[:, None] + bot * ly[:, None]
