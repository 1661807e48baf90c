"""GPU parity: every C-ABI entry point of libpici_b200 against the CPU oracle, element by element,
on the same seeded inputs (workloads.py).  Integer / byte / index outputs (B, I, A, nnz, flags) are
bit-exact; fp32 sums are taken in the oracle's operand order so they are bit-exact too (NaN results
compare as "is NaN").  All calls go through the ctypes binding of the C ABI.
"""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import pici_oracle as po

pytestmark = pytest.mark.gpu

SIZES = (1, 63, 64, 65, 4095, 4096, 4097, 8192, 8193, 3 * 4096 + 17, (1 << 20), (1 << 22) + 123)
DENSITIES = (0.0, 0.0001, 0.01, 0.1, 0.5, 1.0)


@pytest.fixture(scope="module")
def pk():
    from paper_2607_04676_b200 import pici
    pici.lib()
    return pici


def _bits(t: torch.Tensor) -> np.ndarray:
    t = t.detach().cpu().contiguous()
    if t.dtype == torch.float32:
        return t.view(torch.int32).numpy().view(np.uint32)
    return t.view(torch.int16).numpy().view(np.uint16)


def _assert_pici_equal(pk, got, want: po.Pici):
    B, I, A = got.to_host()
    T = po.num_tiles(want.n)
    assert np.array_equal(I[:T + 1], want.I), "index array differs"
    assert np.array_equal(B[:64 * T], want.B), "bitvector differs"
    assert got.nnz_host() == want.nnz
    assert np.array_equal(A, want.A), "packed values differ"


def _assert_bits_equal_nan_aware(got_bits, want_bits):
    g, w = got_bits.view(np.float32), want_bits.view(np.float32)
    nan = np.isnan(w)
    assert np.array_equal(np.isnan(g), nan)
    assert np.array_equal(got_bits[~nan], want_bits[~nan])


def _upload(pk, o: po.Pici, device="cuda"):
    """Oracle Pici -> device Pici (inputs for decompress / reductions come from the ORACLE's encoder)."""
    d = pk.alloc_pici(o.n, pk.F32 if o.dtype == "f32" else pk.BF16, device)
    d.B[:o.B.size] = torch.from_numpy(o.B.view(np.int64)).to(device)
    d.I[:o.I.size] = torch.from_numpy(o.I.view(np.int32)).to(device)
    if o.A.size:
        a = torch.from_numpy(o.A.view(np.int32 if o.dtype == "f32" else np.int16))
        d.A[:o.A.size] = a.view(torch.float32 if o.dtype == "f32" else torch.bfloat16).to(device)
    return d


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("n", SIZES)
def test_compress_and_decompress_match_oracle(pk, n, dtype):
    for j, dens in enumerate(DENSITIES):
        host = wl.sparse_buffer(n, dens, seed=17 * n + j, dtype=dtype)
        want = po.compress(_bits(host), dtype)
        dev = host.cuda()
        out = pk.alloc_pici(n, pk.F32 if dtype == "f32" else pk.BF16)
        out.B.fill_(-1); out.I.fill_(-1)
        ws = pk.alloc_workspace(n)
        pk.compress(dev, out, ws)
        _assert_pici_equal(pk, out, want)
        # decompress the ORACLE's encoding on the GPU
        back = torch.full_like(dev, 7.0)
        pk.decompress(_upload(pk, want), back)
        assert np.array_equal(_bits(back), po.decompress(want))


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_special_values_and_negative_zero(pk, dtype):
    n = 4096 * 2 + 100
    sp = wl.special_values_f32()
    host = sp.repeat((n + sp.numel() - 1) // sp.numel())[:n].contiguous()
    if dtype == "bf16":
        host = (host.view(torch.int32) >> 16).to(torch.int16).view(torch.bfloat16).contiguous()
    want = po.compress(_bits(host), dtype)
    out = pk.alloc_pici(n, pk.F32 if dtype == "f32" else pk.BF16)
    pk.compress(host.cuda(), out, pk.alloc_workspace(n))
    _assert_pici_equal(pk, out, want)
    back = torch.empty_like(host, device="cuda")
    pk.decompress(out, back)
    assert np.array_equal(_bits(back), po.decompress(want))   # -0.0 -> +0.0, NaN payloads kept


@pytest.mark.parametrize("n", (1, 4097, 3 * 4096 + 17, 1 << 20))
@pytest.mark.parametrize("dens", (0.0, 0.01, 0.05, 0.3, 1.0))
def test_reduce_sd_matches_oracle(pk, n, dens):
    x = wl.sparse_buffer(n, dens, seed=5 + n)
    local = wl.sparse_buffer(n, 0.5, seed=6 + n)
    local[::7] = -0.0                               # untouched elements must keep their bits
    xo = po.compress(_bits(x), "f32")
    want = local.numpy().copy()
    po.reduce_sd(xo, want)
    xd = _upload(pk, xo)
    got = local.cuda()
    pk.reduce_sd(xd, got)
    assert np.array_equal(_bits(got), want.view(np.uint32))
    out = torch.full((n,), 3.0, device="cuda")
    pk.reduce_sd_out(xd, local.cuda(), out)
    assert np.array_equal(_bits(out), want.view(np.uint32))


def _clustered(n, lo, hi, every, seed):
    """Buffer whose tiles alternate between two densities: every `every`-th tile has density `hi`,
    the others `lo` - the per-tile path decisions (list / lane walk / streaming, span fits / does not)
    all occur inside one launch."""
    a, b = wl.sparse_buffer(n, lo, seed=seed), wl.sparse_buffer(n, hi, seed=seed + 1)
    tile = torch.arange(n) // wl.TILE
    return torch.where(tile % every == every - 1, b, a)


@pytest.mark.parametrize("lo,hi,every", ((0.002, 1.0, 16), (0.0, 0.3, 5), (0.6, 0.0, 2), (0.9, 0.01, 3)))
def test_reduce_sd_mixed_tiles(pk, lo, hi, every):
    n = 37 * wl.TILE + 1234
    x = _clustered(n, lo, hi, every, seed=77)
    local = wl.sparse_buffer(n, 0.5, seed=79)
    xo = po.compress(_bits(x), "f32")
    want = local.numpy().copy()
    po.reduce_sd(xo, want)
    got = local.cuda()
    pk.reduce_sd(_upload(pk, xo), got)
    assert np.array_equal(_bits(got), want.view(np.uint32))


@pytest.mark.parametrize("lo,hi,every", ((0.002, 1.0, 16), (0.0, 0.5, 5), (0.7, 0.0, 2), (0.01, 0.9, 9),
                                         (0.001, 1.0, 64), (0.02, 0.2, 40), (0.0, 0.07, 3)))
def test_reduce_ss_mixed_tiles(pk, lo, hi, every):
    n = 133 * wl.TILE + 77
    x = _clustered(n, lo, hi, every, seed=81)
    y = _clustered(n, lo, hi, every + 1, seed=83)
    xo, yo = po.compress(_bits(x), "f32"), po.compress(_bits(y), "f32")
    want = po.reduce_ss(xo, yo)
    out = pk.alloc_pici(n, pk.F32)
    out.B.fill_(-1); out.I.fill_(-1)
    pk.reduce_ss(_upload(pk, xo), _upload(pk, yo), out, pk.alloc_workspace(n))
    _assert_pici_equal(pk, out, want)


@pytest.mark.parametrize("n", (1, 64, 4097, 3 * 4096 + 17, 1 << 20))
@pytest.mark.parametrize("dx,dy", ((0.0, 0.0), (0.01, 0.01), (0.0, 0.2), (0.3, 0.02), (0.6, 0.6), (1.0, 1.0)))
def test_reduce_ss_matches_oracle(pk, n, dx, dy):
    x = wl.sparse_buffer(n, dx, seed=11 + n)
    y = wl.sparse_buffer(n, dy, seed=12 + n)
    # exact cancellations: wherever both are present on a stride, y = -x (C5: the sum is NOT stored)
    both = (x != 0) & (y != 0)
    sel = both & (torch.arange(n) % 3 == 0)
    y = torch.where(sel, -x, y)
    xo, yo = po.compress(_bits(x), "f32"), po.compress(_bits(y), "f32")
    want = po.reduce_ss(xo, yo)
    out = pk.alloc_pici(n, pk.F32)
    out.B.fill_(-1); out.I.fill_(-1)
    pk.reduce_ss(_upload(pk, xo), _upload(pk, yo), out, pk.alloc_workspace(n))
    _assert_pici_equal(pk, out, want)


@pytest.mark.parametrize("d", (0.26, 0.13, 0.06))
def test_reduce_ss_disjoint_supports(pk, d):
    """Disjoint supports: the union is larger than two independent supports of the same densities would
    give, so a span length chosen from that estimate overflows the output region and the kernel has to fall
    back to the tile-by-tile path on the exact candidate count."""
    n = 300 * wl.TILE + 5
    g = torch.Generator().manual_seed(91)
    u = torch.rand(n, generator=g)
    vx, vy = wl.values(n, 92), wl.values(n, 93)
    x = wl.apply_mask(u < d, vx)
    y = wl.apply_mask((u >= d) & (u < 2 * d), vy)
    xo, yo = po.compress(_bits(x), "f32"), po.compress(_bits(y), "f32")
    want = po.reduce_ss(xo, yo)
    assert want.nnz == xo.nnz + yo.nnz
    out = pk.alloc_pici(n, pk.F32)
    out.B.fill_(-1); out.I.fill_(-1)
    pk.reduce_ss(_upload(pk, xo), _upload(pk, yo), out, pk.alloc_workspace(n))
    _assert_pici_equal(pk, out, want)


@pytest.mark.parametrize("n,dx,dy", ((1, 1.0, 1.0), (3, 0.7, 0.7), (4096 + 3, 0.5, 0.5), (9 * 4096 + 1, 0.02, 0.9),
                                     (40 * 4096, 0.3, 0.3), (700 * 4096 + 5, 0.01, 0.01)))
def test_reduce_ss_is_repeatable(pk, n, dx, dy):
    """The merge kernel hands data between warp roles through mbarriers (staging / walking / scanning): the same
    launch repeated many times, on buffers whose previous contents differ, must give the oracle's result every
    time (a stale shared-memory word shows up as an occasional wrong value, not as a steady one)."""
    x = wl.sparse_buffer(n, dx, seed=31 + n)
    y = wl.sparse_buffer(n, dy, seed=32 + n)
    y = torch.where((x != 0) & (y != 0) & (torch.arange(n) % 2 == 0), -x, y)     # many exact cancellations
    xo, yo = po.compress(_bits(x), "f32"), po.compress(_bits(y), "f32")
    want = po.reduce_ss(xo, yo)
    xd, yd = _upload(pk, xo), _upload(pk, yo)
    ws = pk.alloc_workspace(n)
    out = pk.alloc_pici(n, pk.F32)
    for it in range(40):
        out.B.fill_(it - 3); out.I.fill_(it - 3); out.A.fill_(float(it))
        pk.reduce_ss(xd, yd, out, ws)
        _assert_pici_equal(pk, out, want)


def test_reduce_ss_special_values(pk):
    n = 4096 + 50
    sp = wl.special_values_f32()
    x = sp.repeat((n + sp.numel() - 1) // sp.numel())[:n].contiguous()
    y = torch.roll(x, 5).contiguous()
    xo, yo = po.compress(_bits(x), "f32"), po.compress(_bits(y), "f32")
    want = po.reduce_ss(xo, yo)
    out = pk.alloc_pici(n, pk.F32)
    pk.reduce_ss(_upload(pk, xo), _upload(pk, yo), out, pk.alloc_workspace(n))
    B, I, A = out.to_host()
    assert np.array_equal(B[:want.B.size], want.B) and np.array_equal(I[:want.I.size], want.I)
    _assert_bits_equal_nan_aware(A, want.A)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("n", (1, 4097, (1 << 20) + 3))
def test_nnz_and_maybe_densify(pk, n, dtype):
    host = wl.sparse_buffer(n, 0.03, seed=n, dtype=dtype)
    want = po.compress(_bits(host), dtype)
    dev = host.cuda()
    cnt = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    pk.nnz_dense(dev, cnt)
    assert int(cnt.item()) == want.nnz == po.nnz_dense(_bits(host), dtype)
    xd = _upload(pk, want)
    cnt.fill_(-1)
    pk.nnz(xd, cnt)
    assert int(cnt.item()) == po.nnz_pici(want)
    for nnz_switch in (0, want.nnz, want.nnz + 1, n + 1):
        flag = torch.full((1,), -7, dtype=torch.int32, device="cuda")
        out = torch.full_like(dev, 9.0)
        pk.maybe_densify(xd, nnz_switch, out, flag)
        switched = want.nnz >= nnz_switch
        assert int(flag.item()) == int(switched)
        if switched:
            assert np.array_equal(_bits(out), po.decompress(want))
        else:
            assert bool((out == 9.0).all())        # untouched


def test_gates_leave_outputs_untouched(pk):
    n = 8192
    host = wl.sparse_buffer(n, 0.1, seed=3)
    dev = host.cuda()
    gate = torch.tensor([1], dtype=torch.int32, device="cuda")
    out = pk.alloc_pici(n, pk.F32)
    out.B.fill_(-1); out.I.fill_(-1)
    ws = pk.alloc_workspace(n)
    pk.compress(dev, out, ws, gate=gate, gate_value=0)          # closed
    assert bool((out.I == -1).all()) and bool((out.B == -1).all())
    pk.compress(dev, out, ws, gate=gate, gate_value=1)          # open
    _assert_pici_equal(pk, out, po.compress(_bits(host), "f32"))
    d = torch.full((n,), 5.0, device="cuda")
    pk.decompress(out, d, gate=gate, gate_value=0)
    assert bool((d == 5.0).all())
    pk.dense_add(dev, dev, d, gate=gate, gate_value=0)
    assert bool((d == 5.0).all())
    pk.dense_add(dev, dev, d, gate=gate, gate_value=1)
    assert np.array_equal(_bits(d), po.dense_add(host.numpy(), host.numpy()).view(np.uint32))


def test_errors_are_codes_not_crashes(pk):
    n = 4096
    dev = torch.zeros(n, device="cuda")
    out = pk.alloc_pici(n, pk.F32)
    ws = pk.alloc_workspace(n)
    with pytest.raises(pk.PiciError) as e:
        pk.compress(dev, out, ws[:16])
    assert e.value.code == -5
    with pytest.raises(pk.PiciError) as e:
        pk.compress(torch.zeros(n + 1, device="cuda")[1:], out, ws)       # 4-byte offset pointer
    assert e.value.code == -3
    small = pk.alloc_pici(n, pk.F32)
    small.A = small.A[: n // 2]
    with pytest.raises(pk.PiciError) as e:
        pk.compress(dev, small, ws)
    assert e.value.code == -4


def test_host_end_to_end_forms(pk):
    n = (1 << 18) + 77
    host = wl.sparse_buffer(n, 0.02, seed=9).pin_memory()
    want = po.compress(_bits(host), "f32")
    h = pk.alloc_host_pici(n, pk.F32)
    scratch = pk.alloc_pici(n, pk.F32)
    d_dense = torch.empty(n, device="cuda")
    pk.compress_host(host, h, d_dense, scratch, pk.alloc_workspace(n))
    assert h.nnz == want.nnz
    assert np.array_equal(h.I.numpy().view(np.uint32)[:want.I.size], want.I)
    assert np.array_equal(h.B.numpy().view(np.uint64)[:want.B.size], want.B)
    assert np.array_equal(_bits(h.A[:h.nnz]), want.A)
    back = torch.empty(n).pin_memory()
    pk.decompress_host(h, back, scratch, d_dense)
    assert np.array_equal(_bits(back), po.decompress(want))


def test_probe_random_rmw_adds_one_at_the_indices(pk):
    """The measurement aid bench.py times beside reduce_sd (pici_probe_random_rmw): dense[idx[i]] += 1.0f."""
    n = 5 * wl.TILE + 17
    x = wl.sparse_buffer(n, 0.01, seed=3)
    idx = torch.nonzero(x).flatten().to(torch.int32).cuda()
    d = wl.sparse_buffer(n, 0.5, seed=4)
    got = d.cuda()
    pk.probe_random_rmw(idx, got)
    want = d.clone()
    want[idx.cpu().long()] += 1.0
    assert torch.equal(got.cpu().view(torch.int32), want.view(torch.int32))


@pytest.mark.parametrize("n,dens", [(4096, 0.5), (4097, 0.01), (70001, 0.3), ((1 << 20) + 5, 0.02), (1 << 20, 1.0), (1 << 18, 0.0)])
def test_bf16_reductions_match_oracle(pk, n, dens):
    """bf16 reduce_sd (in place and with a separate output) and dense add: widened to fp32, one add, rounded to nearest
    even - bit-exact with the oracle (which is pinned to torch's bf16 addition); untouched elements keep their bits."""
    xh = wl.sparse_buffer(n, dens, seed=n + 3, dtype="bf16")
    yh = wl.sparse_buffer(n, 0.7, seed=n + 4, dtype="bf16")
    yh[::9] = -xh[::9]
    yb = _bits(yh).copy()
    yb[1::13] = 0x8000                                              # -0.0 in the dense operand survives where x has no value
    yh = torch.from_numpy(yb.view(np.int16)).view(torch.bfloat16)
    xo = po.compress(_bits(xh), "bf16")
    want = yb.copy()
    po.reduce_sd(xo, want)
    acc = yh.clone().cuda()
    pk.reduce_sd(_upload(pk, xo), acc)
    assert np.array_equal(_bits(acc), want)
    out = torch.full((n,), 7.0, dtype=torch.bfloat16, device="cuda")
    pk.reduce_sd_out(_upload(pk, xo), yh.cuda(), out)
    assert np.array_equal(_bits(out), want)
    got = torch.empty(n, dtype=torch.bfloat16, device="cuda")
    pk.dense_add(xh.cuda(), yh.cuda(), got)
    assert np.array_equal(_bits(got), po.dense_add(_bits(xh), yb))


def test_bf16_reduce_sd_full_size(pk):
    """N = 2^28 bf16: the scatter-add equals torch's bf16 addition on the whole buffer."""
    n = 1 << 28
    x = wl.sparse_buffer(n, 0.05, seed=0, dtype="bf16", device="cuda")
    y = wl.sparse_buffer(n, 0.5, seed=1, dtype="bf16", device="cuda")
    px = pk.alloc_pici(n, pk.BF16)
    pk.compress(x, px, pk.alloc_workspace(n))
    acc = y.clone()
    pk.reduce_sd(px, acc)
    assert torch.equal(acc.view(torch.int16), (x + y).view(torch.int16))


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_compress_random_sizes_share_one_workspace(pk, dtype):
    """The scan service under many launch shapes: 120 random (n, density) pairs - sizes from one tile to 2^23 + tail,
    densities from empty to full, including mixed tiles - compressed back to back through ONE workspace (the launch
    epoch is all that separates them) and compared with the oracle bit for bit."""
    rng = np.random.default_rng(2024 if dtype == "f32" else 2025)
    nmax = (1 << 23) + 4097
    ws = pk.alloc_workspace(nmax)
    dt = pk.F32 if dtype == "f32" else pk.BF16
    cases = []
    for j in range(120):
        n = int(rng.integers(1, nmax)) if j % 3 else int(rng.integers(1, 40 * 4096))
        dens = float(rng.choice([0.0, 0.0005, 0.01, 0.05, 0.12, 0.3, 0.5, 0.7, 1.0]))
        host = wl.sparse_buffer(n, dens, seed=9000 + j, dtype=dtype)
        if j % 5 == 0 and n > 3 * 4096:      # a dense stretch inside a sparse buffer: wide tiles among narrow ones
            lo = int(rng.integers(0, n - 2 * 4096))
            host[lo:lo + 2 * 4096 + 17] = 1.0
        out = pk.alloc_pici(n, dt)
        pk.compress(host.cuda(), out, ws)     # no synchronisation between the launches
        cases.append((host, out))
    for host, out in cases:
        _assert_pici_equal(pk, out, po.compress(_bits(host), dtype))


def test_launch_epoch_wraps(pk):
    """The 30-bit launch epoch that tags every scan word wraps after 2^30 launches.  White box: the epoch word (the
    first 4 bytes of the workspace) is set to three launches before the wrap; a large call, small calls across the
    wrap and the large call again must all match the oracle - the wrap clears every word the workspace has ever
    tagged, not only the current call's."""
    n_big, n_small = (1 << 21) + 77, 5 * 4096 + 3
    ws = pk.alloc_workspace(n_big)
    ws[:4].view(torch.int32).fill_(0x3FFFFFFF - 3)
    big = wl.sparse_buffer(n_big, 0.05, seed=41)
    small = wl.sparse_buffer(n_small, 0.3, seed=42)
    want_big, want_small = po.compress(_bits(big), "f32"), po.compress(_bits(small), "f32")
    want_sum = po.reduce_ss(want_small, want_small)
    dbig, dsmall = big.cuda(), small.cuda()
    outs = []
    for step in range(12):                      # the epoch passes 0x3FFFFFFF at the fourth launch
        if step in (0, 7, 11):
            o = pk.alloc_pici(n_big, pk.F32)
            pk.compress(dbig, o, ws)
            outs.append((o, want_big))
        elif step % 2:
            o = pk.alloc_pici(n_small, pk.F32)
            pk.compress(dsmall, o, ws)
            outs.append((o, want_small))
        else:
            o = pk.alloc_pici(n_small, pk.F32)
            pk.reduce_ss(outs[-1][0], outs[-1][0], o, ws) if outs[-1][1] is want_small else pk.compress(dsmall, o, ws)
            outs.append((o, want_sum if outs[-1][1] is want_small else want_small))
    torch.cuda.synchronize()
    assert int(ws[:4].view(torch.int32).item()) < 16, "the epoch has wrapped"
    for o, want in outs:
        _assert_pici_equal(pk, o, want)


def test_concurrent_streams_with_their_own_workspaces(pk):
    """Three streams, each with its own workspace, launch compress / reduce_ss at the same time: every launch is sized
    for a full resident wave, so the launches share the SMs and each runs partly resident - the kernels' waits (scan
    service, tickets, flushers) must only ever be on work that is already running."""
    n = (1 << 23) + 4097
    streams = [torch.cuda.Stream() for _ in range(3)]
    xs = [wl.sparse_buffer(n, d, seed=70 + i) for i, d in enumerate((0.01, 0.1, 0.5))]
    wants = [po.compress(_bits(x), "f32") for x in xs]
    want_ss = [po.reduce_ss(w, w) for w in wants]
    dev = [x.cuda() for x in xs]
    ws = [pk.alloc_workspace(n) for _ in streams]
    outs = [[] for _ in streams]
    torch.cuda.synchronize()
    for rep in range(6):
        for i, st in enumerate(streams):
            with torch.cuda.stream(st):
                o = pk.alloc_pici(n, pk.F32)
                pk.compress(dev[i], o, ws[i], stream=st)
                s = pk.alloc_pici(n, pk.F32)
                pk.reduce_ss(o, o, s, ws[i], stream=st)
                outs[i].append((o, s))
    torch.cuda.synchronize()
    for i in range(3):
        for o, s in outs[i][::2]:
            _assert_pici_equal(pk, o, wants[i])
            _assert_pici_equal(pk, s, want_ss[i])
