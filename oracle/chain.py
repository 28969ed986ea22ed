"""Oracle: incremental anchoring of window-local poses into one trajectory.

P:72-74  "For each batch, the model predicts ... camera extrinsics {T_t^{w->c}}
in a local coordinate frame. ... Let t_anchor denote the transition frame
shared by the current and previous windows.  We compute a rigid transformation
to align the current batch's local origin to the terminal pose of the previous
trajectory".  P:76 "we lock the gravity-aligned rotation (pitch and roll) and
propagate only the horizontal yaw and translation across batch boundaries".

The procedure is followed step by step (readings B1-B9 in DESIGN.md):
  anchor    t_a = start_{n-1} + W - 1 (last frame of the previous window)
  boundary  RIGID: B_n = Cp . Tc          Cp = inv(T^{L_{n-1}}_{W-1}), Tc = T^{L_n}_{k_a}
            YAW  : Y = rotation about world Y by the heading of R(Cp) R(Cc)^T's
                   forward axis; B_n = [Y | p(Cp) - Y p(Cc)]
  fold      A_0 = I, A_n = A_{n-1} . B_n  (left fold, in this order)
  apply     T^{G->c}_t = T^{L_n->c}_k . inv(A_n)

Arithmetic is IEEE fp64 on Python floats: only + - * / sqrt, every operation
rounded on its own (no FMA), dot products associated left to right, so a GPU
that performs the same operations in the same order is bit-identical (needed
for the bit-exact focus pixel, BJ north_star).  Poses are (R, t) pairs: R a 3x3
list of rows, t a 3-list; the bottom row of the 4x4 is never read.
TEST INFRASTRUCTURE ONLY.
"""
import math

from . import windows as _win

YAW_TRANSLATION = 0
RIGID = 1


def dot3(a0, a1, a2, b0, b1, b2):
    return ((a0 * b0) + (a1 * b1)) + (a2 * b2)


def mat_mul(a, b):
    return [[dot3(a[i][0], a[i][1], a[i][2], b[0][j], b[1][j], b[2][j]) for j in range(3)]
            for i in range(3)]


def mat_vec(a, x):
    return [dot3(a[i][0], a[i][1], a[i][2], x[0], x[1], x[2]) for i in range(3)]


def transpose(a):
    return [[a[j][i] for j in range(3)] for i in range(3)]


def compose(x, y):
    """(Rx,tx).(Ry,ty) = (Rx Ry, Rx ty + tx)."""
    rx, tx = x
    ry, ty = y
    rt = mat_vec(rx, ty)
    return mat_mul(rx, ry), [rt[i] + tx[i] for i in range(3)]


def inverse(x):
    """Rigid inverse [R^T | -R^T t]."""
    r, t = x
    rt = transpose(r)
    p = mat_vec(rt, t)
    return rt, [-p[0], -p[1], -p[2]]


def identity():
    return [[1.0, 0.0, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]], [0.0, 0.0, 0.0]


def from_4x4(m):
    return ([[float(m[i][j]) for j in range(3)] for i in range(3)],
            [float(m[i][3]) for i in range(3)])


def to_4x4(x):
    r, t = x
    return [r[0] + [t[0]], r[1] + [t[1]], r[2] + [t[2]], [0.0, 0.0, 0.0, 1.0]]


def boundary(prev_last, cur_anchor, mode):
    """B_n from T^{L_{n-1}}_{W-1} and T^{L_n}_{k_a}."""
    cp = inverse(prev_last)
    if mode == RIGID:
        return compose(cp, cur_anchor)
    cc = inverse(cur_anchor)
    r_rel = mat_mul(cp[0], transpose(cc[0]))
    a = r_rel[2][2]
    b = r_rel[0][2]
    r = math.sqrt((a * a) + (b * b))
    if r < 1e-12:
        c, s = 1.0, 0.0
    else:
        c, s = a / r, b / r
    y = [[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]]
    yp = mat_vec(y, cc[1])
    return y, [cp[1][i] - yp[i] for i in range(3)]


def chain_poses(local_w2c, w, stride, num_frames, mode=YAW_TRANSLATION, return_transforms=False):
    """local_w2c: [num_windows][W] of 4x4 (fp32 values) -> list of num_frames 4x4 (fp64)."""
    starts = _win.window_starts(num_frames, w, stride)
    assert len(local_w2c) == len(starts)
    a = [identity()]
    for n in range(1, len(starts)):
        k_a = (starts[n - 1] + w - 1) - starts[n]
        b_n = boundary(from_4x4(local_w2c[n - 1][w - 1]), from_4x4(local_w2c[n][k_a]), mode)
        a.append(compose(a[n - 1], b_n))
    a_inv = [inverse(x) for x in a]
    out = []
    for n, k in _win.owner_of_frames(num_frames, w, stride):
        out.append(to_4x4(compose(from_4x4(local_w2c[n][k]), a_inv[n])))
    if return_transforms:
        return out, [to_4x4(x) for x in a]
    return out
