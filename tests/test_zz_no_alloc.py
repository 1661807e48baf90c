"""pici_compress_static (include/pici_static.h): the compress entry point that allocates nothing - its scan scratch is
a static device array inside the library.  Its outputs must equal pici_compress's (the existing path, with a
caller-owned workspace) bit for bit - the tolerance of every compress test here: B, I, A are index / byte work - on
calls made back to back, since every call shares the array and finds what the last one left.
This file sorts last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

import workloads as wl


def test_limits_and_rejection_before_any_cuda_call():
    from paper_2607_04676_b200 import static_ws
    L = static_ws.lib()
    max_n, nbytes = static_ws.limits()
    assert max_n == 1 << 28 and nbytes == 796288
    a, b, c, d = 0x10000, 0x20000, 0x30000, 0x40000
    WORKSPACE, CAPACITY, ALIGN, DTYPE = -5, -4, -3, -2
    assert L.pici_compress_static(a, max_n + 1, 0, b, c, d, max_n + 1, None) == WORKSPACE     # beyond the static scratch
    assert L.pici_compress_static(a, 8192, 0, b, c, d, 8191, None) == CAPACITY
    assert L.pici_compress_static(a + 4, 8192, 0, b, c, d, 8192, None) == ALIGN
    assert L.pici_compress_static(a, 8192, 7, b, c, d, 8192, None) == DTYPE


def _equal(got, want):
    assert got.nnz_host() == want.nnz_host()
    for g, w in zip(got.to_host(), want.to_host()):
        assert np.array_equal(g, w)


@pytest.mark.gpu
def test_static_scratch_compress_equals_the_workspace_path_call_after_call():
    from paper_2607_04676_b200 import pici as pk
    from paper_2607_04676_b200 import static_ws
    pk.lib()
    cases = [((1 << 22) + 4097, 0.01, "f32"), (3 * 4096 + 17, 0.5, "f32"), (1 << 28, 0.01, "f32"), (1, 1.0, "f32"),
             ((1 << 20) + 5, 0.1, "bf16"), (70_001, 0.0, "bf16"), ((1 << 22) + 4097, 0.3, "f32")]
    ws = pk.alloc_workspace(1 << 28)
    results = []
    for j, (n, dens, dtype) in enumerate(cases):
        x = wl.sparse_buffer(n, dens, seed=300 + j, dtype=dtype, device="cuda")
        dt = pk.F32 if dtype == "f32" else pk.BF16
        want, got = pk.alloc_pici(n, dt), pk.alloc_pici(n, dt)
        got.B.fill_(-1); got.I.fill_(-1)
        pk.compress(x, want, ws)                      # the existing path
        held = torch.cuda.memory_allocated()
        static_ws.compress(x, got)                    # two calls in a row on the shared array, no sync in between
        static_ws.compress(x, got)
        assert torch.cuda.memory_allocated() == held  # (torch's allocator; the library itself never allocates)
        results.append((got, want))
    torch.cuda.synchronize()
    for got, want in results:
        _equal(got, want)
