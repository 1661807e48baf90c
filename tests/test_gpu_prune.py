"""GPU parity of prune-and-compress (include/pici_prune.h) against oracle/prune_oracle.c +
oracle/pici_oracle.c: the threshold is bit-exact (an exact selection), the residual and the Pici message are bit-exact
(same two roundings, same compare); several error-feedback iterations are chained so that e carries over."""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import pici_oracle as po
from oracle import prune_oracle as pr

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from paper_2607_04676_b200 import pici, prune
    prune.lib()
    return pici, prune


def _bits(t):
    return t.detach().cpu().contiguous().view(torch.int32).numpy().view(np.uint32)


@pytest.mark.parametrize("n,leak,keep", [(4096, 1.0, 0.01), (4097, 0.5, 0.05), (70_001, 0.9, 0.01), (1 << 20, 0.75, 0.01),
                                         ((1 << 22) + 333, 1.0, 0.001), (1 << 18, 0.0, 0.5)])
def test_prune_compress_matches_oracle(mods, n, leak, keep):
    _run_case(mods, n, leak, keep, None)


def test_prune_calls_of_many_sizes_share_one_workspace(mods):
    """The same cases through ONE workspace (sized for the largest), a plain compress of yet another size in between."""
    pk, pn = mods
    cases = [((1 << 22) + 333, 1.0, 0.001), (4097, 0.5, 0.05), (1 << 20, 0.75, 0.01), (70_001, 0.9, 0.01), (4096, 1.0, 0.01)]
    ws = pn.alloc_workspace(cases[0][0], cases[0][0] // 1000)
    for j, (n, leak, keep) in enumerate(cases):
        _run_case(mods, n, leak, keep, ws)
        nn = 3 * 4096 * (j + 1) + 5
        x = wl.sparse_buffer(nn, 0.1, seed=60 + j)
        o = pk.alloc_pici(nn, pk.F32)
        pk.compress(x.cuda(), o, ws)
        want = po.compress(_bits(x), "f32")
        B, I, A = o.to_host()
        assert np.array_equal(I[:want.I.size], want.I) and np.array_equal(B[:want.B.size], want.B) and np.array_equal(A, want.A)


def _run_case(mods, n, leak, keep, ws):
    pk, pn = mods
    m = max(4, n // 1000)
    k = max(1, int(np.ceil(keep * m)))
    sample_h = torch.from_numpy(np.sort(np.random.default_rng(n).choice(n, size=m, replace=False)).astype(np.int32))
    sample = sample_h.cuda()
    e_h = np.zeros(n, np.float32)
    e_d = torch.zeros(n, device="cuda")
    if ws is None:
        ws = pn.alloc_workspace(n, m)
    d_tau = torch.zeros(1, device="cuda")
    out = pk.alloc_pici(n, pk.F32)
    for it in range(3):                                              # three iterations: the residual carries over
        g_t = wl.values(n, seed=100 * it + 7, dist="normal", scale=0.02)
        if it == 1:
            g_t[5:n:97] = 0.0
            g_t[min(11, n - 1)] = float("nan")
        g_h = g_t.numpy()
        tau = pr.threshold(g_h, e_h, leak, sample_h.numpy().view(np.uint32), k)
        sent, e_new, _ = pr.prune_ef(g_h, e_h, leak, tau)
        want = po.compress(sent.view(np.uint32), "f32")
        g_d = g_t.cuda()
        pn.threshold(g_d, e_d, leak, sample, k, d_tau, ws)
        assert _bits(d_tau)[0] == np.float32(tau).view(np.uint32)
        out.B.fill_(-1); out.I.fill_(-1)
        pn.prune_compress(g_d, e_d, leak, d_tau, out, ws)
        B, I, A = out.to_host()
        T = po.num_tiles(n)
        assert np.array_equal(I[:T + 1], want.I) and np.array_equal(B[:64 * T], want.B) and np.array_equal(A, want.A)
        got_e = _bits(e_d)
        nan = np.isnan(e_new)
        assert np.array_equal(np.isnan(got_e.view(np.float32)), nan) and np.array_equal(got_e[~nan], e_new.view(np.uint32)[~nan])
        e_h = e_new


def test_full_size_properties(mods):
    """N = 2^28, the paper's recipe (sample 0.1 %, keep 1 %): ~99 % message sparsity, sent + e' == acc, the message
    decompresses to `sent`, the threshold is the k-th largest of the sampled magnitudes (torch.topk)."""
    pk, pn = mods
    n = 1 << 28
    g = wl.values(n, seed=3, scale=0.02, device="cuda")
    e = wl.values(n, seed=4, scale=0.01, device="cuda")
    leak = 0.9
    sample = torch.arange(0, n, 1000, device="cuda", dtype=torch.int32)
    m = sample.numel()
    k = -(-m // 100)
    acc = g + (leak * e)                                             # torch fp32: product rounded, then sum rounded
    want_tau = torch.topk(acc[sample.long()].abs(), k).values[-1]
    ws = pn.alloc_workspace(n, m)
    d_tau = torch.zeros(1, device="cuda")
    pn.threshold(g, e, leak, sample, k, d_tau, ws)
    assert d_tau.item() == want_tau.item()
    out = pk.alloc_pici(n, pk.F32)
    e2 = e.clone()
    pn.prune_compress(g, e2, leak, d_tau, out, ws)
    keep = acc.abs() >= d_tau
    nnz = out.nnz_host()
    assert nnz == int(keep.sum().item()) and 0.007 < nnz / n < 0.013
    sent = torch.empty_like(g)
    pk.decompress(out, sent)
    assert torch.equal(sent.view(torch.int32), torch.where(keep, acc, torch.zeros_like(acc)).view(torch.int32))
    assert torch.equal((sent + e2).view(torch.int32), (acc + 0.0).view(torch.int32))
