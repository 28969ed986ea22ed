"""Oracle: the dense layers around the window attention, in fp64.

PAPER.md treats the transformer as a black box ("an existing foundation model"); BASELINE.json
fixes only the shapes ("24-layer d=1024 H=16 stack", head_dim 64).  The block structure below is therefore a READING
(E1-E4 in DESIGN.md), the standard pre-norm ViT block that DINOv2-style encoders use, with seeded synthetic weights:

    E1  h = x + W_o . Attn(split_heads(W_qkv . LN1(x) + b_qkv)) + b_o
    E2  y = h + W_2 . GELU(W_1 . LN2(h) + b_1) + b_2           hidden width 4 d
    E3  GELU(t) = t/2 (1 + erf(t / sqrt 2))                     (exact, not the tanh form)
    E4  LN(x) = (x - mean) / sqrt(var + 1e-6) * gamma + beta    biased variance over the d channels

Every function is its definition written out with a numpy matmul as the only library step; inputs are the bf16 / fp32
values promoted exactly to fp64.  Parity of the READING is unpinned by the paper (it names no block); the arithmetic of
each function is pinned by tests/test_oracle_block.py.  TEST INFRASTRUCTURE ONLY.
"""
import math

import numpy as np

_erf = np.vectorize(math.erf, otypes=[np.float64])


def linear(x, w, bias=None):
    """x [M,K], w [N,K] (nn.Linear layout: out_features x in_features), bias [N] -> x w^T + bias, [M,N] fp64."""
    y = np.asarray(x, dtype=np.float64) @ np.asarray(w, dtype=np.float64).T
    if bias is not None:
        y = y + np.asarray(bias, dtype=np.float64)[None, :]
    return y


def gelu(t):
    """E3: t/2 (1 + erf(t/sqrt 2))."""
    t = np.asarray(t, dtype=np.float64)
    return 0.5 * t * (1.0 + _erf(t / math.sqrt(2.0)))


def layernorm(x, gamma, beta, eps=1e-6):
    """E4 over the last axis."""
    x = np.asarray(x, dtype=np.float64)
    mean = x.mean(axis=-1, keepdims=True)
    var = ((x - mean) ** 2).mean(axis=-1, keepdims=True)
    return (x - mean) / np.sqrt(var + eps) * np.asarray(gamma, dtype=np.float64) + np.asarray(beta, dtype=np.float64)


def split_heads(y, heads, head_dim):
    """[M, 3*heads*head_dim] (q | k | v, each head-major) -> three [M, heads, head_dim] arrays."""
    m = y.shape[0]
    hd = heads * head_dim
    return tuple(y[:, i * hd:(i + 1) * hd].reshape(m, heads, head_dim) for i in range(3))


def round_bf16(a):
    """E5: every tensor stored between two layers is bf16, rounded to nearest even (BJ: "bf16 tokens").
    fp64 -> fp32 (nearest even) -> keep the top 16 bits with round-to-nearest-even on the dropped 16."""
    f = np.asarray(a, dtype=np.float64).astype(np.float32)
    bits = f.view(np.uint32).astype(np.uint64)
    rounded = ((bits + 0x7FFF + ((bits >> 16) & 1)) >> 16) << 16
    out = rounded.astype(np.uint32).view(np.float32).astype(np.float64)
    return np.where(np.isfinite(f), out, f.astype(np.float64))


def block_forward(x, wts, frames_per_window, tokens_per_frame, heads, mode, attention_fn, store=round_bf16):
    """E1 + E2 for one window: x [S, d] -> y [S, d], S = W*P.  `wts` maps ln1_g, ln1_b, w_qkv, b_qkv, w_o, b_o, ln2_g,
    ln2_b, w_1, b_1, w_2, b_2 to arrays.  `attention_fn(q, k, v, W, P, mode)` is oracle.attention.window_attention
    (passed in so that this module stays a leaf).  `store` is applied to every tensor the method keeps between two
    layers (E5); pass `lambda a: a` for the unrounded mathematical block."""
    x = np.asarray(x, dtype=np.float64)
    s_len, d = x.shape
    hd = d // heads
    a = store(layernorm(x, wts["ln1_g"], wts["ln1_b"]))
    q, k, v = (store(t) for t in split_heads(linear(a, wts["w_qkv"], wts["b_qkv"]), heads, hd))
    o, _ = attention_fn(q[None], k[None], v[None], frames_per_window, tokens_per_frame, mode)
    o = store(o[0].reshape(s_len, d))
    h = store(linear(o, wts["w_o"], wts["b_o"]) + x)
    m = store(layernorm(h, wts["ln2_g"], wts["ln2_b"]))
    u = store(gelu(linear(m, wts["w_1"], wts["b_1"])))
    return store(linear(u, wts["w_2"], wts["b_2"]) + h)
