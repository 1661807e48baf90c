"""GPU parity of the COO entry points (include/pici_coo.h) against oracle/coo_oracle.c, bit for bit, on the same
seeded inputs; all calls go through the C ABI.  Inputs of decompress / reductions come from the ORACLE's encoder.
Full-size rows (N = 2^28, the crossover sweep's configuration): whole-buffer properties plus sampled windows."""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import coo_oracle as co

pytestmark = pytest.mark.gpu

SIZES = (1, 63, 127, 128, 129, 4095, 4096, 4097, 8192, 3 * 4096 + 17, (1 << 20), (1 << 22) + 123)
DENSITIES = (0.0, 0.0001, 0.01, 0.1, 0.3, 0.5, 1.0)


@pytest.fixture(scope="module")
def ck():
    from paper_2607_04676_b200 import coo
    coo.lib()
    return coo


def _bits(t):
    return t.detach().cpu().contiguous().view(torch.int32).numpy().view(np.uint32)


def _upload(ck, o: co.Coo):
    d = ck.alloc_coo(o.n)
    d.idx.fill_(-1); d.val.fill_(float("nan"))
    if o.nnz:
        d.idx[:o.nnz] = torch.from_numpy(o.idx.view(np.int32)).cuda()
        d.val[:o.nnz] = torch.from_numpy(o.val.view(np.int32)).view(torch.float32).cuda()
    d.nnz.fill_(o.nnz)
    return d


def _assert_equal(got, want: co.Coo):
    assert got.nnz_host() == want.nnz
    gi, gv = got.to_host()
    assert np.array_equal(gi, want.idx), "indices differ"
    assert np.array_equal(gv, want.val), "values differ"


@pytest.mark.parametrize("n", SIZES)
def test_compress_decompress_match_oracle(ck, n):
    ws = ck.alloc_workspace(n)
    for j, dens in enumerate(DENSITIES):
        host = wl.sparse_buffer(n, dens, seed=31 * n + j)
        want = co.compress(_bits(host))
        out = ck.alloc_coo(n)
        out.idx.fill_(-1); out.val.fill_(-7.0); out.nnz.fill_(-1)
        ck.compress(host.cuda(), out, ws)
        _assert_equal(out, want)
        assert int(out.idx[want.nnz:].max().item() if want.nnz < out.idx.numel() else -1) == -1   # nothing past nnz is written
        back = torch.full((n,), 7.0, device="cuda")
        ck.decompress(_upload(ck, want), back, ws)
        assert np.array_equal(_bits(back), co.decompress(want))


def test_special_values(ck):
    n = 4096 + 300
    v = torch.zeros(n)
    v[::5] = torch.randn((n + 4) // 5)
    bits = _bits(v).copy()
    bits[1] = 0x80000000; bits[2] = 0x7FC12345; bits[3] = 0x00000001; bits[4] = 0xFF800000; bits[4097] = 0x80000001
    host = torch.from_numpy(bits.view(np.int32)).view(torch.float32)
    want = co.compress(bits)
    ws = ck.alloc_workspace(n)
    out = ck.alloc_coo(n)
    ck.compress(host.cuda(), out, ws)
    _assert_equal(out, want)
    back = torch.full((n,), 7.0, device="cuda")
    ck.decompress(out, back, ws)
    assert np.array_equal(_bits(back), co.decompress(want))          # -0.0 -> +0.0, NaN payload kept


@pytest.mark.parametrize("n,dx,dy", [(1, 1.0, 1.0), (4097, 0.01, 0.02), (70000, 0.3, 0.0), (70000, 0.0, 0.3), (1 << 20, 0.01, 0.01),
                                     ((1 << 20) + 77, 0.5, 0.5), (1 << 18, 1.0, 1.0), (1 << 20, 0.0001, 0.05)])
def test_reductions_match_oracle(ck, n, dx, dy):
    xh, yh = wl.sparse_buffer(n, dx, seed=5), wl.sparse_buffer(n, dy, seed=6)
    yh[::11] = -xh[::11]                                              # exact cancellations where both have an entry
    X, Y = co.compress(_bits(xh)), co.compress(_bits(yh))
    ws = ck.alloc_workspace(n)
    out = ck.alloc_coo(n)
    for rep in range(3):                                              # the workspace is reused without clearing
        out.idx.fill_(-1); out.val.fill_(-7.0); out.nnz.fill_(-1)
        ck.reduce_ss(_upload(ck, X), _upload(ck, Y), out, ws)
        _assert_equal(out, co.reduce_ss(X, Y))
    acc = yh.clone().cuda()
    ck.reduce_sd(_upload(ck, X), acc)
    want = yh.numpy().copy()
    co.reduce_sd(X, want)
    assert np.array_equal(_bits(acc), want.view(np.uint32))


@pytest.mark.parametrize("sparsity", [0.9, 0.99, 0.9999])
def test_full_size_properties_and_samples(ck, sparsity):
    """N = 2^28 (configs[1] size, the crossover sweep): compress -> decompress is the identity, indices ascend, nnz is
    the dense count, values are the gathered inputs; sampled 2^16-element windows against the oracle; the merge of two
    independent supports equals the dense sum (whole buffer) and the oracle on a sampled window."""
    n = 1 << 28
    x = wl.sparse_buffer(n, 1.0 - sparsity, seed=0, device="cuda")
    ws = ck.alloc_workspace(n)
    cx = ck.alloc_coo(n)
    ck.compress(x, cx, ws)
    k = cx.nnz_host()
    assert k == int((x != 0).sum().item())
    idx = cx.idx[:k].long()
    assert bool((idx[1:] > idx[:-1]).all())
    assert torch.equal(cx.val[:k], x[idx])
    back = torch.empty_like(x)
    ck.decompress(cx, back, ws)
    assert torch.equal(back.view(torch.int32), x.view(torch.int32))
    for lo in (0, 12345 * 4096, n - (1 << 16)):                       # windows that start on a block boundary
        w = co.compress(_bits(x[lo:lo + (1 << 16)]))
        a = int(torch.searchsorted(idx, lo).item())
        gi = (cx.idx[a:a + w.nnz].cpu().numpy().view(np.uint32) - np.uint32(lo))
        assert np.array_equal(gi, w.idx) and np.array_equal(_bits(cx.val[a:a + w.nnz]), w.val)
    del back
    y = wl.sparse_buffer(n, 1.0 - sparsity, seed=1, device="cuda")
    cy, cz = ck.alloc_coo(n), ck.alloc_coo(n)
    ck.compress(y, cy, ws)
    ck.reduce_ss(cx, cy, cz, ws)
    s = x + y
    kz = cz.nnz_host()
    assert kz == int((s != 0).sum().item())
    zi = cz.idx[:kz].long()
    assert bool((zi[1:] > zi[:-1]).all()) and torch.equal(cz.val[:kz].view(torch.int32), s[zi].view(torch.int32))
    lo = 777 * 4096
    wx, wy = co.compress(_bits(x[lo:lo + (1 << 16)])), co.compress(_bits(y[lo:lo + (1 << 16)]))
    wz = co.reduce_ss(wx, wy)
    a = int(torch.searchsorted(zi, lo).item())
    assert np.array_equal(cz.idx[a:a + wz.nnz].cpu().numpy().view(np.uint32) - np.uint32(lo), wz.idx)
    assert np.array_equal(_bits(cz.val[a:a + wz.nnz]), wz.val)
    acc = y.clone()
    ck.reduce_sd(cx, acc)
    assert torch.equal(acc.view(torch.int32), s.view(torch.int32))    # x + y == y + x bit for bit (no NaN here)


def test_mixed_calls_of_many_sizes_share_one_workspace(ck):
    """One workspace, 90 calls of random size and density back to back, no synchronisation: Pici compress (fp32 and
    bf16), Pici reduce_ss, COO compress, COO reduce_ss.  What one call leaves behind (tagged words, the service's done
    words, ticket and exit counters, the epoch) must never be mistaken by the next, whatever its n."""
    from oracle import pici_oracle as po
    from paper_2607_04676_b200 import pici as pk
    rng = np.random.default_rng(77)
    nmax = (1 << 22) + 4097
    ws = ck.alloc_workspace(nmax)
    checks = []
    for j in range(90):
        op = j % 5
        n = int(rng.integers(1, nmax)) if j % 4 else int(rng.integers(1, 24 * 4096))
        dx, dy = (float(rng.choice([0.0, 0.001, 0.01, 0.08, 0.3, 0.6, 1.0])) for _ in range(2))
        x = wl.sparse_buffer(n, dx, seed=500 + 2 * j)
        if op in (0, 1):                                        # Pici compress
            dtype = "f32" if op == 0 else "bf16"
            if op == 1:
                x = wl.sparse_buffer(n, dx, seed=500 + 2 * j, dtype="bf16")
            out = pk.alloc_pici(n, pk.F32 if op == 0 else pk.BF16)
            pk.compress(x.cuda(), out, ws)
            bits = _bits(x) if op == 0 else x.view(torch.int16).numpy().view(np.uint16)
            checks.append(("pici", out, po.compress(bits, dtype)))
        elif op == 2:                                           # Pici reduce_ss
            y = wl.sparse_buffer(n, dy, seed=501 + 2 * j)
            ox, oy = po.compress(_bits(x), "f32"), po.compress(_bits(y), "f32")
            dxp, dyp, out = pk.alloc_pici(n, pk.F32), pk.alloc_pici(n, pk.F32), pk.alloc_pici(n, pk.F32)
            pk.compress(x.cuda(), dxp, ws)
            pk.compress(y.cuda(), dyp, ws)
            pk.reduce_ss(dxp, dyp, out, ws)
            checks.append(("pici", out, po.reduce_ss(ox, oy)))
        elif op == 3:                                           # COO compress
            out = ck.alloc_coo(n)
            ck.compress(x.cuda(), out, ws)
            checks.append(("coo", out, co.compress(_bits(x))))
        else:                                                   # COO reduce_ss
            y = wl.sparse_buffer(n, dy, seed=501 + 2 * j)
            cx, cy, out = ck.alloc_coo(n), ck.alloc_coo(n), ck.alloc_coo(n)
            ck.compress(x.cuda(), cx, ws)
            ck.compress(y.cuda(), cy, ws)
            ck.reduce_ss(cx, cy, out, ws)
            checks.append(("coo", out, co.reduce_ss(co.compress(_bits(x)), co.compress(_bits(y)))))
    for kind, got, want in checks:
        if kind == "coo":
            _assert_equal(got, want)
        else:
            B, I, A = got.to_host()
            Tn = po.num_tiles(want.n)
            assert np.array_equal(I[:Tn + 1], want.I) and np.array_equal(B[:64 * Tn], want.B) and np.array_equal(A, want.A)
