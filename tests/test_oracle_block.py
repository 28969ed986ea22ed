"""Pins for oracle/block.py: closed forms, invariants, library cross-checks."""
import math

import numpy as np
import torch

from oracle import block as ob


def test_linear_against_brute_force_and_torch():
    rng = np.random.default_rng(0)
    x, w, b = rng.standard_normal((5, 7)), rng.standard_normal((3, 7)), rng.standard_normal(3)
    y = ob.linear(x, w, b)
    for i in range(5):
        for n in range(3):
            assert abs(y[i, n] - (sum(x[i, k] * w[n, k] for k in range(7)) + b[n])) < 1e-13
    t = torch.nn.functional.linear(torch.from_numpy(x), torch.from_numpy(w), torch.from_numpy(b)).numpy()
    assert np.abs(y - t).max() < 1e-13
    # a transposed weight (the plausible mistake) must differ
    assert np.abs(ob.linear(x[:, :3], w[:, :3]) - x[:, :3] @ w[:, :3]).max() > 1e-3


def test_linear_identity_and_selection():
    x = np.arange(12.0).reshape(3, 4)
    assert np.array_equal(ob.linear(x, np.eye(4)), x)
    sel = np.zeros((2, 4)); sel[0, 3] = 1.0; sel[1, 0] = -2.0
    assert np.array_equal(ob.linear(x, sel, np.array([1.0, 0.0])), np.stack([x[:, 3] + 1.0, -2.0 * x[:, 0]], axis=1))


def test_gelu_closed_forms():
    assert ob.gelu(0.0) == 0.0
    assert abs(ob.gelu(1.0) - 0.8413447460685429) < 1e-15          # Phi(1)
    assert abs(ob.gelu(-1.0) + 0.15865525393145707) < 1e-15        # -Phi(-1)
    t = np.linspace(-6, 6, 101)
    assert np.abs(ob.gelu(t) - ob.gelu(-t) - t).max() < 1e-14      # x Phi(x) - (-x) Phi(-x) = x
    assert abs(ob.gelu(10.0) - 10.0) < 1e-12 and abs(ob.gelu(-10.0)) < 1e-12
    ref = torch.nn.functional.gelu(torch.from_numpy(t)).numpy()    # erf form in torch
    assert np.abs(ob.gelu(t) - ref).max() < 1e-14
    tanh_form = 0.5 * t * (1 + np.tanh(math.sqrt(2 / math.pi) * (t + 0.044715 * t ** 3)))
    assert np.abs(ob.gelu(t) - tanh_form).max() > 1e-4             # the tanh approximation is NOT what E3 says


def test_layernorm_invariants():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((6, 32)) * 3 + 5
    y = ob.layernorm(x, np.ones(32), np.zeros(32), eps=0.0)
    assert np.abs(y.mean(axis=1)).max() < 1e-14 and np.abs((y ** 2).mean(axis=1) - 1).max() < 1e-13
    # shift and positive scale invariance (eps = 0), affine part applied after normalisation
    assert np.abs(ob.layernorm(2.5 * x + 7, np.ones(32), np.zeros(32), eps=0.0) - y).max() < 1e-13
    g, b = rng.standard_normal(32), rng.standard_normal(32)
    assert np.abs(ob.layernorm(x, g, b, eps=0.0) - (y * g + b)).max() < 1e-13
    ref = torch.nn.functional.layer_norm(torch.from_numpy(x), (32,), torch.from_numpy(g), torch.from_numpy(b), 1e-6).numpy()
    assert np.abs(ob.layernorm(x, g, b) - ref).max() < 1e-12
    # two-element closed form: (a, b) -> (+-1) / sqrt(1 + eps / ((a-b)/2)^2)
    out = ob.layernorm(np.array([[1.0, 3.0]]), np.ones(2), np.zeros(2), eps=1e-6)
    assert np.abs(out - np.array([[-1.0, 1.0]]) / math.sqrt(1 + 1e-6)).max() < 1e-15


def test_split_heads_layout():
    heads, hd = 3, 4
    y = np.arange(2 * 3 * heads * hd, dtype=np.float64).reshape(2, 3 * heads * hd)
    q, k, v = ob.split_heads(y, heads, hd)
    assert q.shape == (2, heads, hd)
    assert q[1, 2, 3] == y[1, 2 * hd + 3] and k[0, 1, 0] == y[0, heads * hd + hd] and v[1, 0, 1] == y[1, 2 * heads * hd + 1]


def test_round_bf16_matches_torch_and_ties_to_even():
    rng = np.random.default_rng(5)
    a = np.concatenate([rng.standard_normal(4096) * 10.0 ** rng.integers(-6, 6, 4096), [0.0, -0.0, 1.0, 65504.0]])
    ref = torch.from_numpy(a).to(torch.float32).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(ob.round_bf16(a), ref)
    # 1 + 2^-8 is exactly half way between 1 and 1 + 2^-7: ties go to the even mantissa
    assert ob.round_bf16(1.0 + 2.0 ** -8) == 1.0 and ob.round_bf16(1.0 + 3 * 2.0 ** -8) == 1.0 + 2.0 ** -6


def test_block_forward_identity_cases():
    from oracle import attention as oa
    rng = np.random.default_rng(6)
    s_len, d, heads = 12, 8, 2
    x = rng.standard_normal((s_len, d))
    z = lambda *shape: np.zeros(shape)
    wts = dict(ln1_g=np.ones(d), ln1_b=z(d), w_qkv=rng.standard_normal((3 * d, d)), b_qkv=z(3 * d), w_o=z(d, d), b_o=z(d),
               ln2_g=np.ones(d), ln2_b=z(d), w_1=rng.standard_normal((4 * d, d)), b_1=z(4 * d), w_2=z(d, 4 * d), b_2=z(d))
    ident = lambda a: a
    # zero output projections: both residual branches vanish, the block is the identity
    assert np.array_equal(ob.block_forward(x, wts, 3, 4, heads, oa.GLOBAL, oa.window_attention, store=ident), x)
    # only biases on the two branches: y = x + b_o + b_2
    wts["b_o"], wts["b_2"] = rng.standard_normal(d), rng.standard_normal(d)
    y = ob.block_forward(x, wts, 3, 4, heads, oa.GLOBAL, oa.window_attention, store=ident)
    assert np.abs(y - (x + wts["b_o"] + wts["b_2"])).max() < 1e-14
    # w_v = I-selecting, w_o = I, uniform attention (w_q = w_k = 0): branch 1 adds the mean over tokens of LN1(x)
    wq = z(3 * d, d); wq[2 * d:] = np.eye(d)
    wts.update(w_qkv=wq, w_o=np.eye(d), b_o=z(d), b_2=z(d))
    y = ob.block_forward(x, wts, 3, 4, heads, oa.GLOBAL, oa.window_attention, store=ident)
    ln = ob.layernorm(x, np.ones(d), z(d))
    assert np.abs(y - (x + ln.mean(axis=0, keepdims=True))).max() < 1e-13
    # frame mode: the mean is taken per frame of 4 tokens
    y = ob.block_forward(x, wts, 3, 4, heads, oa.FRAME, oa.window_attention, store=ident)
    per_frame = np.repeat(ln.reshape(3, 4, d).mean(axis=1), 4, axis=0)
    assert np.abs(y - (x + per_frame)).max() < 1e-13
    # bf16 storage only perturbs the result at the 2^-8 level
    yb = ob.block_forward(x, wts, 3, 4, heads, oa.FRAME, oa.window_attention)
    assert 0 < np.abs(yb - y).max() < 0.05
