"""Pins for oracle/attention.py (BJ north_star lists rows-sum-to-1,
frame-permutation equivariance and brute-force softmax).  CPU only."""
import math

import numpy as np
import pytest
import torch
from scipy.special import logsumexp

from oracle import attention as oa


def _rand(shape, seed, scale=1.0):
    return np.random.default_rng(seed).normal(0.0, scale, shape)


def test_brute_force_tiny():
    # S<=8, D<=4: pure-Python exp/sum, no numpy in the reference value
    q, k, v = _rand((1, 8, 2, 4), 1), _rand((1, 8, 2, 4), 2), _rand((1, 8, 2, 4), 3)
    o, lse = oa.window_attention(q, k, v, 2, 4, oa.GLOBAL)
    for h in range(2):
        for i in range(8):
            ref, l = oa.brute_force_row(q[0, i, h], k[0, :, h], v[0, :, h], 0.5)
            assert np.allclose(o[0, i, h], ref, rtol=0, atol=1e-14)
            assert abs(lse[0, h, i] - l) < 1e-13


def test_hand_computed_two_keys():
    # one query, two keys, D=1: weights are the logistic function of scale*(x0-x1)
    q = np.array([[[[2.0]]]])
    k = np.array([[[[1.0]], [[-1.0]]]]).reshape(1, 2, 1, 1)
    v = np.array([[[[10.0]], [[20.0]]]]).reshape(1, 2, 1, 1)
    qq = np.repeat(q, 2, axis=1)
    o, lse = oa.window_attention(qq, k, v, 1, 2, oa.GLOBAL, scale=1.0)
    w0 = 1.0 / (1.0 + math.exp(-4.0))          # x0 - x1 = 2 - (-2)
    assert abs(o[0, 0, 0, 0] - (10.0 * w0 + 20.0 * (1 - w0))) < 1e-13
    assert abs(lse[0, 0, 0] - (2.0 + math.log1p(math.exp(-4.0)))) < 1e-13


def test_default_scale_is_inv_sqrt_d():
    q, k, v = _rand((1, 6, 1, 16), 4), _rand((1, 6, 1, 16), 5), _rand((1, 6, 1, 16), 6)
    o1, _ = oa.window_attention(q, k, v, 1, 6)
    o2, _ = oa.window_attention(q, k, v, 1, 6, scale=0.25)
    o3, _ = oa.window_attention(q, k, v, 1, 6, scale=0.5)
    assert np.array_equal(o1, o2) and not np.allclose(o1, o3)


def test_closed_forms():
    k, v = _rand((1, 12, 2, 8), 7), _rand((1, 12, 2, 8), 8)
    # Q = 0 -> uniform weights -> mean of V, lse = log S
    o, lse = oa.window_attention(np.zeros_like(k), k, v, 3, 4)
    assert np.allclose(o, np.broadcast_to(v.mean(axis=1, keepdims=True), v.shape), atol=1e-14)
    assert np.allclose(lse, math.log(12), atol=1e-14)
    # all keys equal -> mean of V for any Q
    q = _rand((1, 12, 2, 8), 9)
    keq = np.broadcast_to(k[:, :1], k.shape)
    o, _ = oa.window_attention(q, keq, v, 3, 4)
    assert np.allclose(o, np.broadcast_to(v.mean(axis=1, keepdims=True), v.shape), atol=1e-13)
    # one key dominating -> O -> V of that key
    kd = k.copy()
    kd[0, 5] = 0.0
    qd = np.zeros_like(q)
    qd[..., 0] = 1.0
    kd[..., 0] = 0.0
    kd[0, 5, :, 0] = 400.0
    o, _ = oa.window_attention(qd, kd, v, 3, 4)
    assert np.allclose(o, np.broadcast_to(v[:, 5:6], v.shape), atol=1e-30 + 1e-12)


def test_rows_convex_combination():
    q, k, v = _rand((2, 24, 3, 8), 10), _rand((2, 24, 3, 8), 11), _rand((2, 24, 3, 8), 12)
    # V = const 1 -> O = sum of weights = 1 exactly up to rounding
    o, _ = oa.window_attention(q, k, np.ones_like(v), 4, 6)
    assert np.allclose(o, 1.0, atol=1e-14)
    for mode in (oa.GLOBAL, oa.FRAME):
        o, _ = oa.window_attention(q, k, v, 4, 6, mode)
        if mode == oa.GLOBAL:
            lo, hi = v.min(axis=1, keepdims=True), v.max(axis=1, keepdims=True)
            assert (o >= lo - 1e-12).all() and (o <= hi + 1e-12).all()


def test_permutation_equivariance():
    w, p = 4, 5
    q, k, v = _rand((1, 20, 2, 8), 13), _rand((1, 20, 2, 8), 14), _rand((1, 20, 2, 8), 15)
    o, _ = oa.window_attention(q, k, v, w, p)
    # permute frames of Q,K,V -> O permuted the same way (BJ north_star)
    fperm = np.array([2, 0, 3, 1])
    tok = (fperm[:, None] * p + np.arange(p)[None, :]).reshape(-1)
    o2, _ = oa.window_attention(q[:, tok], k[:, tok], v[:, tok], w, p)
    assert np.allclose(o2, o[:, tok], atol=1e-14)
    # frame mode is equivariant under frame permutation too
    of, _ = oa.window_attention(q, k, v, w, p, oa.FRAME)
    of2, _ = oa.window_attention(q[:, tok], k[:, tok], v[:, tok], w, p, oa.FRAME)
    assert np.allclose(of2, of[:, tok], atol=1e-14)
    # permuting only K and V jointly leaves O unchanged
    anyperm = np.random.default_rng(16).permutation(20)
    o3, _ = oa.window_attention(q, k[:, anyperm], v[:, anyperm], w, p)
    assert np.allclose(o3, o, atol=1e-14)


def test_key_shift_invariance():
    q, k, v = _rand((1, 16, 2, 8), 17), _rand((1, 16, 2, 8), 18), _rand((1, 16, 2, 8), 19)
    o, lse = oa.window_attention(q, k, v, 2, 8)
    shift = _rand((1, 1, 2, 8), 20)
    o2, lse2 = oa.window_attention(q, k + shift, v, 2, 8)
    assert np.allclose(o2, o, atol=1e-13)
    assert np.allclose(lse2 - lse, 8 ** -0.5 * np.einsum("nshd,nxhd->nhs", q, shift), atol=1e-12)


def test_frame_mode_reduces_to_global():
    nw, w, p = 2, 3, 7
    q, k, v = (_rand((nw, w * p, 2, 8), s) for s in (21, 22, 23))
    of, lf = oa.window_attention(q, k, v, w, p, oa.FRAME)
    view = lambda a: a.reshape(nw * w, p, 2, 8)
    og, lg = oa.window_attention(view(q), view(k), view(v), 1, p, oa.GLOBAL)
    assert np.array_equal(of.reshape(og.shape), og)
    assert np.array_equal(lf.transpose(0, 2, 1).reshape(nw * w, p, 2).transpose(0, 2, 1), lg)
    # W = 1: the two modes coincide
    o1, _ = oa.window_attention(view(q), view(k), view(v), 1, p, oa.FRAME)
    assert np.array_equal(o1, og)
    # frame mode differs from global mode when W > 1 (block-diagonal is not a no-op)
    ogl, _ = oa.window_attention(q, k, v, w, p, oa.GLOBAL)
    assert not np.allclose(ogl, of)


def test_frame_mode_ignores_other_frames():
    w, p = 3, 4
    q, k, v = (_rand((1, w * p, 1, 4), s) for s in (24, 25, 26))
    o, _ = oa.window_attention(q, k, v, w, p, oa.FRAME)
    k2, v2 = k.copy(), v.copy()
    k2[0, p:2 * p] += 3.0
    v2[0, p:2 * p] -= 5.0
    o2, _ = oa.window_attention(q, k2, v2, w, p, oa.FRAME)
    assert np.array_equal(o2[0, :p], o[0, :p]) and np.array_equal(o2[0, 2 * p:], o[0, 2 * p:])
    assert not np.allclose(o2[0, p:2 * p], o[0, p:2 * p])


@pytest.mark.parametrize("mode", [oa.GLOBAL, oa.FRAME])
def test_library_cross_check_sdpa_and_logsumexp(mode):
    nw, w, p, h, d = 2, 3, 11, 2, 16
    q, k, v = (_rand((nw, w * p, h, d), s) for s in (27, 28, 29))
    o, lse = oa.window_attention(q, k, v, w, p, mode)
    tq, tk, tv = (torch.from_numpy(a).permute(0, 2, 1, 3) for a in (q, k, v))   # [n,h,s,d]
    if mode == oa.FRAME:
        tq, tk, tv = (t.reshape(nw, h, w, p, d) for t in (tq, tk, tv))
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)
    ref = ref.reshape(nw, h, w * p, d).permute(0, 2, 1, 3).numpy()
    assert np.abs(o - ref).max() < 1e-12
    x = np.einsum("nihd,njhd->nhij", q, k) / math.sqrt(d)
    if mode == oa.FRAME:
        f = np.arange(w * p) // p
        x = np.where(f[:, None] == f[None, :], x, -np.inf)
    assert np.abs(lse - logsumexp(x, axis=-1)).max() < 1e-12


def test_row_subset_is_exact():
    q, k, v = (_rand((1, 30, 2, 8), s) for s in (30, 31, 32))
    rows = np.array([0, 7, 29, 13])
    for mode in (oa.GLOBAL, oa.FRAME):
        o, lse = oa.window_attention(q, k, v, 3, 10, mode)
        os_, ls = oa.window_attention(q, k, v, 3, 10, mode, rows=rows)
        assert np.allclose(os_, o[:, rows], atol=1e-15) and np.allclose(ls, lse[:, :, rows], atol=1e-15)


def test_transposed_operand_would_fail():
    # guards against Q/K swapped: attention is not symmetric in (Q, K)
    q, k, v = (_rand((1, 9, 1, 4), s) for s in (33, 34, 35))
    o, _ = oa.window_attention(q, k, v, 1, 9)
    o_sw, _ = oa.window_attention(k, q, v, 1, 9)
    assert not np.allclose(o, o_sw)
