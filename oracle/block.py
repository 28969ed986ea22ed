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
