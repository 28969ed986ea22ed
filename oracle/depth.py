"""Oracle: per-window depth scale alignment on the overlap and depth-stream stitching
(Fig. 3 "Depth alignment"; the emitted frames of P:76).

The paper gives no formula (it states the pose alignment is rigid, "not Sim(3)", and is silent on the depth
scale, reading B7).  Reading F2: every window's depth maps live in the window's own scale; window n >= 1
is brought to the scale of the stream so far by the least-squares factor on the frames it shares with window n-1:

    r_n = argmin_r  sum_{t in overlap, pixels} (r D_n[t] - D_{n-1}[t])^2  =  sum D_{n-1} D_n / sum D_n^2
    c_0 = 1,  c_n = c_{n-1} r_n,         emitted frame t of window n:  D_out[t] = c_n D_n[t - start_n]

over the pixels where both depths are finite and > 0; r_n = 1 when there is no such pixel.  Windows, overlaps and
emitted frames are those of windows.py (reading B6 for the tail).  Plain numpy fp64.  TEST INFRASTRUCTURE ONLY.
"""
import numpy as np

from . import windows as ow


def overlap_ratio(prev_frames, cur_frames):
    """r = sum(a b) / sum(b b) over valid pixels of the shared frames (a: previous window, b: current)."""
    a = np.asarray(prev_frames, dtype=np.float64).ravel()
    b = np.asarray(cur_frames, dtype=np.float64).ravel()
    ok = np.isfinite(a) & np.isfinite(b) & (a > 0) & (b > 0)
    sab = float(np.sum(a[ok] * b[ok]))
    sbb = float(np.sum(b[ok] * b[ok]))
    return sab / sbb if sbb > 0.0 else 1.0


def align_depth(depth_local, w, stride, num_frames):
    """depth_local [Nw, W, h, w_px] -> (depth_out fp64 [N, h, w_px], scales c_n fp64 [Nw])."""
    d = np.asarray(depth_local, dtype=np.float64)
    starts = ow.window_starts(num_frames, w, stride)
    assert d.shape[0] == len(starts) and d.shape[1] == w
    c = [1.0]
    for n in range(1, len(starts)):
        shared = starts[n - 1] + w - starts[n]            # frames [start_n, start_{n-1} + W)
        off = starts[n] - starts[n - 1]
        r = overlap_ratio(d[n - 1, off:off + shared], d[n, 0:shared])
        c.append(c[-1] * r)
    out = np.empty((num_frames,) + d.shape[2:], dtype=np.float64)
    for t, (n, k) in enumerate(ow.owner_of_frames(num_frames, w, stride)):
        out[t] = c[n] * d[n, k]
    return out, np.array(c, dtype=np.float64)
