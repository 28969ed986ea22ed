"""Differential test of the two head_dim 64 attention kernels.  Sequences below 32 KV tiles run on the persistent kernel
(attention_clc.cu: work items handed out by cluster launch control, many items per CTA), longer ones on the one-item-per-CTA
kernel (attention.cu).  Both run the same tile pipeline in the same order, so on the same inputs their outputs must be
BIT-IDENTICAL.  A second build of the library with the persistent kernel switched off (-DMF_PERSISTENT_BELOW_TILES=0; and
-DMF_NO_SCORE_BOUND, so that the one-item kernel takes its exact online-softmax path like the persistent one) supplies
the other side; seeded random shapes put many items on every CTA, with one to thirty-one KV tiles per item and live / dead second
Q tiles in every order.  (This is how the two deadlocks of the persistent kernel's protocol were found: DESIGN.md 6.1.)
The oracle comparison of both kernels is tests/test_gpu_attention.py; this test is about the pipeline protocol."""
import ctypes
import os
import sys

import numpy as np
import pytest
import torch

from paper_2601_07154_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def libs(tmp_path_factory):
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    from paper_2601_07154_b200 import api, build
    tmp = tmp_path_factory.mktemp("nopersist")
    other = build.build(out=str(tmp / "libmf_nopersist.so"), extra_flags=["-DMF_PERSISTENT_BELOW_TILES=0", "-DMF_NO_SCORE_BOUND"], build_dir=str(tmp / "obj"))
    new = api.lib()
    old = ctypes.CDLL(other)
    old.mf_window_attention.argtypes = new.mf_window_attention.argtypes
    return new, old


def _run(lib, q, k, v, windows, w, p, heads, mode):
    out = torch.full_like(q, float("nan"))
    lse = torch.full((windows, heads, w * p), float("nan"), device="cuda")
    st = lib.mf_window_attention(q.data_ptr(), k.data_ptr(), v.data_ptr(), out.data_ptr(), lse.data_ptr(), windows, w, p, heads, 64, mode,
                                 0.0, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert st == 0
    torch.cuda.synchronize()
    return out, lse


@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_persistent_kernel_equals_one_item_kernel_bit_for_bit(libs, seed):
    new, old = libs
    rng = np.random.default_rng(seed)
    for _ in range(60):
        w, p = int(rng.integers(1, 6)), int(rng.integers(1, 700))
        heads, windows, mode = int(rng.integers(1, 21)), int(rng.integers(1, 120)), int(rng.integers(0, 2))
        if mode == 0 and w * p > 3900:          # (32 KV tiles and more never reach the persistent kernel)
            p = 3900 // w
        case = dict(windows=windows, w=w, p=p, heads=heads, mode=mode)
        q, k, v = synth.qkv(windows, w * p, heads, 64, int(rng.integers(0, 1 << 30)), device="cuda", scale=float(rng.choice([1.0, 2.0, 6.0])))
        a, la = _run(new, q, k, v, windows, w, p, heads, mode)
        b, lb = _run(old, q, k, v, windows, w, p, heads, mode)
        assert torch.isfinite(a.float()).all(), case
        assert torch.equal(a, b) and torch.equal(la, lb), case


@pytest.mark.parametrize("s_len,seqs,heads", [(65, 60, 15), (128, 60, 15), (1, 400, 16), (129, 300, 3), (300, 250, 12), (257, 300, 3)])
def test_persistent_kernel_short_items(libs, s_len, seqs, heads):
    # the shapes on which the protocol bugs showed: one, two and three KV tiles per item, thousands of items
    new, old = libs
    q, k, v = synth.qkv(seqs, s_len, heads, 64, 11 + s_len, device="cuda")
    a, la = _run(new, q, k, v, seqs, 1, s_len, heads, 0)
    b, lb = _run(old, q, k, v, seqs, 1, s_len, heads, 0)
    assert torch.equal(a, b) and torch.equal(la, lb)


@pytest.fixture(scope="module")
def nosplit(tmp_path_factory):
    from paper_2601_07154_b200 import api, build
    tmp = tmp_path_factory.mktemp("nosplit")
    other = build.build(out=str(tmp / "libmf_nosplit.so"), extra_flags=["-DMF_NO_SPLIT"], build_dir=str(tmp / "obj"))
    new = api.lib()
    old = ctypes.CDLL(other)
    old.mf_window_attention.argtypes = new.mf_window_attention.argtypes
    return new, old


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_split_kernel_equals_one_item_kernel_bit_for_bit(nosplit, seed):
    # Long sequences: CTAs whose rows are all within the score bound run on attention_split.cu (each row's 128 scores per KV
    # tile split between two threads), the rest on attention.cu.  A build without the split kernel (-DMF_NO_SPLIT) runs every CTA
    # on attention.cu, where such rows take the same score-bound arithmetic in one thread: outputs and lse must be bit-identical.
    # Random shapes (ragged tails of every chunk count, dead second Q tiles), blocks of rows with larger query scales so that
    # launches mix both kinds of CTA.
    new, old = nosplit
    rng = np.random.default_rng(seed)
    for _ in range(12):
        w, heads, windows, mode = int(rng.integers(1, 4)), int(rng.integers(1, 6)), int(rng.integers(1, 4)), int(rng.integers(0, 2))
        s_target = int(rng.integers(3969, 9000))
        p = s_target if mode == 1 else max(1, s_target // w)
        s_len = w * p
        q, k, v = synth.qkv(windows, s_len, heads, 64, int(rng.integers(0, 1 << 30)), device="cuda")
        f = torch.ones(s_len, device="cuda")
        for _ in range(int(rng.integers(0, 4))):
            i = int(rng.integers(0, s_len))
            f[i:i + int(rng.integers(1, 600))] = 8.0
        q = (q.float() * f[None, :, None, None]).to(torch.bfloat16)
        case = dict(windows=windows, w=w, p=p, heads=heads, mode=mode)
        a, la = _run(new, q, k, v, windows, w, p, heads, mode)
        b, lb = _run(old, q, k, v, windows, w, p, heads, mode)
        assert torch.isfinite(a.float()).all(), case
        assert torch.equal(a, b) and torch.equal(la, lb), case
