"""mf_window_attention_noalloc (include/mf.h): the attention entry point that allocates nothing -- its score-bound scratch
is a static __device__ array inside the library.  Collected last on purpose (the suite runs with pytest -x).  The new entry
point must give what mf_window_attention gives (same kernels: bit for bit, and within the oracle bars the other attention
tests use) on two calls in a row, the second with smaller keys so that maxima left in the array by the first call would
show; it must perform no device allocation, and must reject sizes beyond the array before enqueuing anything."""
import ctypes

import numpy as np
import pytest
import torch

from oracle import attention as oa
from paper_2601_07154_b200 import synth

pytestmark = pytest.mark.gpu

MAX_ABS, REL_L2 = 2e-2, 1e-2          # BASELINE.json north_star (tests/test_gpu_attention.py)


@pytest.fixture(scope="module")
def api():
    from paper_2601_07154_b200 import api as a
    a.lib()
    return a


def _to64(t):
    return t.detach().float().cpu().numpy().astype(np.float64)


def test_noalloc_matches_the_allocating_path_twice_in_a_row(api):
    s_len, heads = 40 * 128 + 77, 3                        # 41 KV tiles: the one-item kernel with the score bound
    rows = np.unique(np.concatenate([np.arange(48), np.arange(s_len - 150, s_len)]))
    for call, k_scale in enumerate((1.0, 0.25)):           # second call: |k| four times smaller than what the array last held
        q, k, v = synth.qkv(2, s_len, heads, 64, 4100 + call, device="cuda")
        k = (k.float() * k_scale).to(torch.bfloat16)
        want, want_lse = api.window_attention(q, k, v, 1, s_len, oa.GLOBAL, return_lse=True)
        out = torch.full_like(q, float("nan"))
        torch.cuda.synchronize()
        before = torch.cuda.memory_stats()["allocation.all.allocated"], torch.cuda.mem_get_info()[0]
        lse = torch.empty_like(want_lse)
        mid = torch.cuda.memory_stats()["allocation.all.allocated"]
        st = api.lib().mf_window_attention_noalloc(q.data_ptr(), k.data_ptr(), v.data_ptr(), out.data_ptr(), lse.data_ptr(), 2, 1, s_len,
                                                   heads, 64, oa.GLOBAL, 0.0, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert st == 0, api.lib().mf_last_error()
        torch.cuda.synchronize()
        assert torch.cuda.memory_stats()["allocation.all.allocated"] == mid and mid == before[0] + 1      # (the lse tensor above)
        assert torch.cuda.mem_get_info()[0] >= before[1] - lse.numel() * 4 - (4 << 20)                     # no driver-side allocation either
        assert torch.equal(out, want) and torch.equal(lse, want_lse), call
        ref, lse_ref = oa.window_attention(_to64(q), _to64(k), _to64(v), 1, s_len, oa.GLOBAL, rows=rows)
        got = _to64(out)[:, rows]
        for n in range(2):
            d = got[n] - ref[n]
            assert np.abs(d).max() <= MAX_ABS and np.linalg.norm(d) / np.linalg.norm(ref[n]) <= REL_L2
        assert np.abs(lse.cpu().numpy().astype(np.float64)[:, :, rows] - lse_ref).max() <= 4e-3
    # the binding's switch, FRAME mode of a long frame
    q, k, v = synth.qkv(1, 2 * 4200, 2, 64, 4200, device="cuda")
    assert torch.equal(api.window_attention(q, k, v, 2, 4200, oa.FRAME, noalloc=True), api.window_attention(q, k, v, 2, 4200, oa.FRAME))


def test_noalloc_paths_without_scratch_and_limit(api):
    # short sequences (persistent kernel) and head_dim 128 use no scratch: forwarded, same result
    for dim, s_len in ((64, 777), (128, 5000)):
        q, k, v = synth.qkv(2, s_len, 2, dim, 4300 + dim, device="cuda")
        assert torch.equal(api.window_attention(q, k, v, 1, s_len, oa.GLOBAL, noalloc=True), api.window_attention(q, k, v, 1, s_len, oa.GLOBAL))
    # beyond the static array (sequences x heads > 65536 on the long-sequence path): rejected before anything is enqueued,
    # so the pointers are never touched (they are fake: such tensors would take 36 GB each)
    fake = [ctypes.c_void_p(0x10000 * (i + 1)) for i in range(4)]
    st = api.lib().mf_window_attention_noalloc(*fake, None, 17, 1, 4096, 4000, 64, oa.GLOBAL, 0.0, None)
    assert st != 0 and b"static scratch" in api.lib().mf_last_error()
    torch.cuda.synchronize()
    # and bad arguments give mf_window_attention's own errors
    with pytest.raises(api.MfError, match="MF_ERR_UNSUPPORTED"):
        q32 = torch.zeros((1, 8, 1, 32), dtype=torch.bfloat16, device="cuda")
        api.window_attention(q32, q32.clone(), q32.clone(), 1, 8, oa.GLOBAL, noalloc=True)
