"""Oracle: window self-attention, the definition written out in fp64.

BJ north_star: "cross-frame global self-attention over all S=W*P patch tokens
of a window, alternating with per-frame attention".  PAPER.md does not describe
the transformer (P:41 only says a foundation model's pose prediction is used),
so the authority is BASELINE.json; readings A1-A7 are listed in DESIGN.md.

    x_j  = scale * sum_d Q[i,d] K[j,d]        scale = 1/sqrt(D)
    m    = max_j x_j ; e_j = exp(x_j - m) ; l = sum_j e_j
    O[i] = sum_j (e_j / l) V[j]               lse = m + log l

Global mode: j ranges over all S tokens of the window.  Frame mode: j ranges
over the tokens of i's own frame (token order is frame-major, s = f*P + p).
A numpy matmul is used as a library step; nothing is blocked, fused or
reordered beyond the formula above.  TEST INFRASTRUCTURE ONLY.
"""
import numpy as np

GLOBAL = 0
FRAME = 1


def _rows(q_rows, k, v, scale):
    """q_rows [R,D], k [J,D], v [J,D] (fp64) -> O [R,D], lse [R]."""
    x = (q_rows @ k.T) * scale
    m = x.max(axis=1, keepdims=True)
    e = np.exp(x - m)
    l = e.sum(axis=1, keepdims=True)
    o = (e / l) @ v
    lse = (m + np.log(l))[:, 0]
    return o, lse


def window_attention(q, k, v, frames_per_window, tokens_per_frame, mode=GLOBAL,
                     scale=None, rows=None):
    """q,k,v: float arrays [windows, S, H, D] (bf16 values promoted exactly).

    rows: optional 1-D int array of query indices s (reading A7: rows are
    independent, so a subset is evaluated exactly).  Returns (O, lse) with
    O [windows, R, H, D] fp64 and lse [windows, H, R] fp64, R = len(rows) or S.
    """
    q = np.asarray(q, dtype=np.float64)
    k = np.asarray(k, dtype=np.float64)
    v = np.asarray(v, dtype=np.float64)
    nw, s_len, heads, d = q.shape
    w, p = frames_per_window, tokens_per_frame
    assert s_len == w * p
    if scale is None or scale <= 0:
        scale = 1.0 / np.sqrt(float(d))
    rows = np.arange(s_len) if rows is None else np.asarray(rows, dtype=np.int64)
    out = np.zeros((nw, len(rows), heads, d), dtype=np.float64)
    lse = np.zeros((nw, heads, len(rows)), dtype=np.float64)
    for n in range(nw):
        for h in range(heads):
            if mode == GLOBAL:
                o, l = _rows(q[n, rows, h, :], k[n, :, h, :], v[n, :, h, :], scale)
                out[n, :, h, :] = o
                lse[n, h, :] = l
            else:
                frame_of = rows // p
                for f in np.unique(frame_of):
                    sel = np.nonzero(frame_of == f)[0]
                    lo, hi = f * p, (f + 1) * p
                    o, l = _rows(q[n, rows[sel], h, :], k[n, lo:hi, h, :],
                                 v[n, lo:hi, h, :], scale)
                    out[n, sel, h, :] = o
                    lse[n, h, sel] = l
    return out, lse


def brute_force_row(q_row, k, v, scale):
    """Pure-Python exp/sum for one query row (tiny inputs only); used by the pins."""
    import math
    xs = [scale * sum(float(q_row[d]) * float(k[j][d]) for d in range(len(q_row)))
          for j in range(len(k))]
    m = max(xs)
    es = [math.exp(x - m) for x in xs]
    l = sum(es)
    return [sum(es[j] / l * float(v[j][d]) for j in range(len(k)))
            for d in range(len(v[0]))], m + math.log(l)
