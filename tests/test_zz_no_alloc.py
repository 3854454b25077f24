"""crt_radix_sort_pairs_noalloc: the radix sort with the library's static device scratch (no cudaMalloc / cudaFree inside the call), for
callers that cannot allocate (CUDA graph capture, tight serving loops).  Checked against the existing path, crt_radix_sort_pairs with
caller-provided scratch, bit for bit (integer work: the suite's bar is bit-exact), on two calls in a row that share the static array.
This file sorts last in the collection on purpose: the suite runs with pytest -x, and a failure here must not hide the other tests.
"""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def crt():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_2310_07182_b200 as crt
    return crt


def test_noalloc_sort_equals_the_existing_path_on_two_calls_in_a_row(crt):
    import torch
    from paper_2310_07182_b200 import api
    ctx = crt.Context(0)
    lib = api.lib()
    max_n = lib.crt_radix_sort_noalloc_max_n()
    assert max_n == 1 << 21
    rng = np.random.default_rng(11)
    # first call: a large, ragged size with many equal keys (stability matters) and the inactive-ray sentinel; second call: a smaller size with
    # different data, so that stale contents of the shared scratch (histogram rows of 510 blocks, ping-pong buffers) would show
    cases = [(2088960 - 37, 1 << 12), (300001, 1 << 30)]
    for n, key_range in cases:
        k = rng.integers(0, key_range, n, dtype=np.int64).astype(np.uint32)
        k[rng.random(n) < 0.05] = 0xFFFFFFFF
        keys = ctx.upload(k.view(np.int32)); vals = torch.arange(n, dtype=torch.int32, device=ctx.device)
        ref_k, ref_v = ctx.crt_radix_sort_pairs(keys, vals)                     # existing path: scratch allocated by the caller
        out_k, out_v = torch.full_like(keys, -7), torch.full_like(vals, -7)
        free0 = torch.cuda.mem_get_info()[0]
        ctx.crt_radix_sort_pairs_noalloc(keys, vals, out_k, out_v)
        torch.cuda.synchronize()
        assert free0 - torch.cuda.mem_get_info()[0] < (1 << 20)                 # the call took no device memory (its scratch alone would be 17 MB)
        assert torch.equal(out_k, ref_k) and torch.equal(out_v, ref_v)
        order = np.argsort(k, kind="stable")                                    # and both equal the plain definition: a stable sort
        assert np.array_equal(out_v.cpu().numpy(), order.astype(np.int32)) and np.array_equal(out_k.cpu().numpy().view(np.uint32), k[order])
        assert torch.equal(keys.cpu(), torch.from_numpy(k.view(np.int32)))      # inputs left intact
    # the stated limit: one pair more is refused with a clear error, nothing is launched
    n = max_n + 1
    keys = torch.zeros(n, dtype=torch.int32, device=ctx.device); vals = torch.zeros_like(keys)
    with pytest.raises(api.CrtError) as e:
        ctx.crt_radix_sort_pairs_noalloc(keys, vals, torch.empty_like(keys), torch.empty_like(vals))
    assert e.value.status == api.CRT_ERR_UNSUPPORTED and "maximum" in str(e.value)
    # exactly the maximum works
    n = max_n
    k = rng.integers(0, 1 << 32, n, dtype=np.int64).astype(np.uint32)
    keys = ctx.upload(k.view(np.int32)); vals = torch.arange(n, dtype=torch.int32, device=ctx.device)
    out_k, out_v = ctx.crt_radix_sort_pairs_noalloc(keys, vals, torch.empty_like(keys), torch.empty_like(vals))
    ref_k, ref_v = ctx.crt_radix_sort_pairs(keys, vals)
    assert torch.equal(out_k, ref_k) and torch.equal(out_v, ref_v)
    # n == 0 and argument errors
    e0 = torch.empty(0, dtype=torch.int32, device=ctx.device)
    assert lib.crt_radix_sort_pairs_noalloc(ctx.handle, None, None, C.c_int64(0), None, None, None) == 0
    with pytest.raises(api.CrtError):
        ctx.crt_radix_sort_pairs_noalloc(keys, vals, keys, vals)                # in place
    del e0
