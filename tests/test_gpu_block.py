"""GPU parity: mf_linear / mf_layernorm (through the C ABI) vs the fp64 oracle.
Tolerance: outputs are bf16 roundings (half an ulp = 2^-9 relative) of fp32-accumulated sums, so
|d| <= 2^-8 |ref| + 2e-3 elementwise and rel-L2 <= 4e-3."""
import numpy as np
import pytest
import torch

from oracle import block as ob
from paper_2601_07154_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2601_07154_b200 import api as a
    a.lib()
    return a


def _to64(t):
    return t.detach().float().cpu().numpy().astype(np.float64)


def _close(got, ref):
    d = got - ref
    assert np.isfinite(got).all()
    assert (np.abs(d) <= 2.0 ** -8 * np.abs(ref) + 2e-3).all(), float(np.abs(d).max())
    assert np.linalg.norm(d) / max(np.linalg.norm(ref), 1e-30) <= 4e-3


@pytest.mark.parametrize("m,n,k,splits", [
    (128, 256, 64, 1),        # one tile, one k step
    (300, 256, 64, 1),        # ragged M: three row tiles, last one partial
    (129, 512, 192, 1),       # two n tiles, ring partially filled
    (1000, 768, 320, 3),      # q | k | v split, 5 k steps: the 4-stage ring wraps
    (5000, 1024, 1024, 1),    # more tiles than SMs: persistent loop, both accumulators in use
    (1, 256, 64, 1),          # degenerate: a single row
])
@pytest.mark.parametrize("variant", ["plain", "bias", "bias_gelu", "bias_residual"])
def test_linear_shapes(api, m, n, k, splits, variant):
    if variant == "bias_residual" and splits != 1:
        pytest.skip("residual needs a single output")
    x, w, b = synth.linear_inputs(m, n, k, seed=m * 7 + n + k, device="cuda")
    bias = b if variant != "plain" else None
    res = synth.tokens(m, n, seed=99 + m, device="cuda") if variant == "bias_residual" else None
    act = api.ACT_GELU if variant == "bias_gelu" else api.ACT_NONE
    out = api.linear(x, w, bias, res, act, splits)
    torch.cuda.synchronize()
    ref = ob.linear(_to64(x), _to64(w), None if bias is None else _to64(bias))
    if act == api.ACT_GELU:
        ref = ob.gelu(ref)
    if res is not None:
        ref = ref + _to64(res)
    got = _to64(out) if splits == 1 else np.concatenate([_to64(o) for o in out], axis=1)
    _close(got, ref)


def test_qkv_projection_campus_window_sampled_rows(api):
    # one campus-shaped window: 24864 tokens, d = 1024 -> q | k | v [S, 16*64]; the oracle evaluates sampled rows
    s_len, d = 24864, 1024
    x, w, b = synth.linear_inputs(s_len, 3 * d, d, seed=synth.seed_for(3, 5), device="cuda")
    q, k, v = api.linear(x, w, b, splits=3)
    torch.cuda.synchronize()
    rows = np.unique(np.concatenate([np.arange(64), np.arange(s_len - 64, s_len), np.random.default_rng(3).integers(0, s_len, 256)]))
    ref = ob.linear(_to64(x)[rows], _to64(w), _to64(b))
    rq, rk, rv = ob.split_heads(ref, 16, 64)
    idx = torch.from_numpy(rows).cuda()
    for got, r in ((q, rq), (k, rk), (v, rv)):
        _close(_to64(got[idx]), r.reshape(len(rows), d))
    # the three outputs are exactly the [S, H, D] tensors mf_window_attention takes
    o = api.window_attention(q.view(1, s_len, 16, 64), k.view(1, s_len, 16, 64), v.view(1, s_len, 16, 64), 32, 777)
    assert torch.isfinite(o.float()).all()


@pytest.mark.parametrize("m,d", [(1, 256), (77, 512), (300, 768), (4097, 1024)])
def test_layernorm(api, m, d):
    x = (synth.tokens(m, d, seed=m + d, device="cuda").float() * 3 + 1.5).to(torch.bfloat16)
    g = torch.Generator(device="cuda").manual_seed(m)
    gamma = 1 + 0.1 * torch.randn(d, device="cuda", generator=g)
    beta = 0.1 * torch.randn(d, device="cuda", generator=g)
    out = api.layernorm(x, gamma, beta, 1e-6)
    torch.cuda.synchronize()
    ref = ob.layernorm(_to64(x), _to64(gamma), _to64(beta), 1e-6)
    _close(_to64(out), ref)


def test_linear_errors(api):
    x, w, b = synth.linear_inputs(64, 256, 64, seed=1, device="cuda")
    with pytest.raises(api.MfError):
        api.linear(x, w[:, :32].contiguous())                      # K mismatch
    x2, w2, _ = synth.linear_inputs(64, 128, 64, seed=1, device="cuda")
    with pytest.raises(api.MfError):
        api.linear(x2, w2)                                          # n_split % 256 != 0: unsupported
    x3, w3, _ = synth.linear_inputs(64, 256, 48, seed=1, device="cuda")
    with pytest.raises(api.MfError):
        api.linear(x3, w3)                                          # K % 64 != 0


@pytest.mark.parametrize("mode_name", ["global", "frame"])
@pytest.mark.parametrize("windows,w,p,heads,d_hidden,head_dim", [(2, 2, 100, 4, 1024, 64), (1, 3, 77, 8, 768, 64), (1, 2, 150, 4, 1024, 128)])
def test_block_forward_vs_oracle(api, windows, w, p, heads, d_hidden, head_dim, mode_name):
    # whole pre-norm block (E1, E2) with bf16 storage between kernels (E5): 7 launches vs oracle.block.block_forward.
    # Intermediate bf16 tensors may differ from the oracle's by rare 1-ulp rounding flips (fp32 vs fp64 sums landing on
    # either side of a rounding boundary); a flipped h plus y's own rounding is 2 bf16 ulps = 2^-6 |ref| on a few elements.
    from oracle import attention as oa
    mode = oa.GLOBAL if mode_name == "global" else oa.FRAME
    d = heads * head_dim
    s_len = w * p
    x = synth.tokens(windows * s_len, d, seed=7 + windows + heads, device="cuda")
    wts = synth.block_weights(d, d_hidden, seed=11 + heads, device="cuda")
    y = api.block_forward(x, wts, windows, w, p, heads, mode)
    torch.cuda.synchronize()
    w64 = {k: _to64(v) for k, v in wts.items()}
    for n in range(windows):
        ref = ob.block_forward(_to64(x[n * s_len:(n + 1) * s_len]), w64, w, p, heads, mode, oa.window_attention)
        got = _to64(y[n * s_len:(n + 1) * s_len])
        dlt = got - ref
        assert np.isfinite(got).all()
        # (a flip of h is one ulp of |h|, which can exceed |y| where the MLP branch cancels h: hence the max|ref| term)
        assert (np.abs(dlt) <= 2.0 ** -6 * np.abs(ref) + 2.0 ** -7 * np.abs(ref).max()).all(), float(np.abs(dlt).max())
        assert np.linalg.norm(dlt) / np.linalg.norm(ref) <= 4e-3
    # in place (y == x) gives the same bits
    x2 = x.clone()
    api.block_forward(x2, wts, windows, w, p, heads, mode, out=x2)
    assert torch.equal(x2, y)


@pytest.mark.parametrize("mode_name", ["global", "frame"])
@pytest.mark.parametrize("windows,w,p,heads,d_hidden,head_dim", [(2, 2, 100, 4, 1024, 64), (1, 2, 150, 4, 1024, 128)])
def test_block_forward_vs_unrounded_oracle(api, windows, w, p, heads, d_hidden, head_dim, mode_name):
    # The MATHEMATICAL block (oracle.block.block_forward with store = identity: no rounding anywhere, fp64) against the
    # kernels, so that the check does not depend on the oracle imitating where the kernels store bf16 (reading E5).
    # Tolerance: the path stores seven bf16 tensors (LN1 out, q|k|v, attention out, h, LN2 out, GELU out, y),
    # each a relative perturbation of at most u = 2^-9 per element; the synthetic layers are norm-preserving on average
    # (weights ~ N(0, 1/fan_in)), softmax averaging and LN (unit-variance rows) do not amplify, GELU is 1.13-Lipschitz, so
    # to first order  ||y - y_exact|| / ||y_exact|| <= 7 u = 1.37e-2  (expected ~ sqrt(7) u / sqrt(3) = 3e-3),
    # and per element  |d| <= u |ref| (y's own rounding) + 16 u rms(ref) (six propagated roundings, > 6 sigma).
    from oracle import attention as oa
    mode = oa.GLOBAL if mode_name == "global" else oa.FRAME
    d = heads * head_dim
    s_len = w * p
    x = synth.tokens(windows * s_len, d, seed=70 + windows + heads, device="cuda")
    wts = synth.block_weights(d, d_hidden, seed=110 + heads, device="cuda")
    y = api.block_forward(x, wts, windows, w, p, heads, mode)
    torch.cuda.synchronize()
    w64 = {k: _to64(v) for k, v in wts.items()}
    u = 2.0 ** -9
    for n in range(windows):
        ref = ob.block_forward(_to64(x[n * s_len:(n + 1) * s_len]), w64, w, p, heads, mode, oa.window_attention,
                               store=lambda a: a)
        dlt = _to64(y[n * s_len:(n + 1) * s_len]) - ref
        rel = np.linalg.norm(dlt) / np.linalg.norm(ref)
        rms = np.sqrt(np.mean(ref * ref))
        assert rel <= 7 * u, rel
        assert (np.abs(dlt) <= u * np.abs(ref) + 16 * u * rms).all(), float((np.abs(dlt) - u * np.abs(ref)).max() / (u * rms))
