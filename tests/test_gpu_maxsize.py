"""GPU parity at the LARGEST size the C ABI accepts: n = 2^32 - 1 fp32 elements (pici.h: 0 <= n < 2^32), i.e.
T = 2^20 tiles with a ragged last tile of 4095 elements - the sizes the workspace layout is cut for.  The oracle
cannot run 16 GiB in seconds, so: sampled tiles (first, last, around the 2^30 boundaries, dense ones, random ones)
are compressed one by one by the oracle and compared bit for bit; everything else through properties that hold at
any size (counts, monotone I, exact round trips, sums against one fp32 addition per element)."""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import coo_oracle as co
from oracle import pici_oracle as po

pytestmark = pytest.mark.gpu

N = (1 << 32) - 1
TILE = 4096
T = (N + TILE - 1) // TILE
DENSE_TILES = (0, 7, 12345, (1 << 19) + 1, T - 2, T - 1)


@pytest.fixture(scope="module")
def mods():
    from paper_2607_04676_b200 import coo, pici
    pici.lib()
    coo.lib()
    if torch.cuda.mem_get_info()[0] < 130 * (1 << 30):
        pytest.skip("needs 130 GiB of free device memory")
    return pici, coo


def _sample_tiles(seed: int) -> list[int]:
    rng = np.random.default_rng(seed)
    fixed = list(DENSE_TILES) + [1, T - 3] + [(b >> 12) + d for b in (1 << 30, 2 << 30, 3 << 30) for d in (-1, 0)]
    return sorted(set(fixed + [int(v) for v in rng.integers(0, T, 48)]))


def _tile_bits(x: torch.Tensor, t: int) -> np.ndarray:
    return x[t * TILE:min(N, (t + 1) * TILE)].cpu().view(torch.int32).numpy().view(np.uint32)


def _check_pici_tiles(p, dense: torch.Tensor, tiles):
    """B words, count and packed values of the sampled tiles against the oracle's compress of that tile alone."""
    I = p.I[:T + 1].cpu().numpy().view(np.uint32).astype(np.int64)
    assert I[0] == 0 and np.all(np.diff(I) >= 0) and np.all(np.diff(I) <= TILE)
    for t in tiles:
        want = po.compress(_tile_bits(dense, t), "f32")
        B = p.B[64 * t:64 * (t + 1)].cpu().numpy().view(np.uint64)
        assert np.array_equal(B, want.B), f"tile {t}: bitvector"
        assert I[t + 1] - I[t] == want.nnz, f"tile {t}: count"
        A = p.A[int(I[t]):int(I[t + 1])].cpu().view(torch.int32).numpy().view(np.uint32)
        assert np.array_equal(A, want.A), f"tile {t}: values"
    return I


def test_pici_at_max_n(mods):
    pk, _ = mods
    x = wl.scattered_buffer(N, 40_000_000, seed=0, dense_tiles=DENSE_TILES)
    y = wl.scattered_buffer(N, 25_000_000, seed=1, dense_tiles=(7, 99, T - 1))
    ws = pk.alloc_workspace(N)
    px, py = pk.alloc_pici(N, pk.F32), pk.alloc_pici(N, pk.F32)
    pk.compress(x, px, ws)
    pk.compress(y, py, ws)
    nx, ny = int(torch.count_nonzero(x)), int(torch.count_nonzero(y))
    assert px.nnz_host() == nx and py.nnz_host() == ny
    tiles = _sample_tiles(3)
    I = _check_pici_tiles(px, x, tiles)
    assert I[T] == nx
    d_nnz = torch.zeros(1, dtype=torch.int64, device="cuda")
    pk.nnz_dense(x, d_nnz)
    assert int(d_nnz) == nx

    out = torch.empty_like(x)
    out.fill_(float("nan"))
    pk.decompress(px, out)
    assert torch.equal(out.view(torch.int32), x.view(torch.int32))

    # reduce_ss: O = compress(X + Y); checked tile by tile against the oracle's compress of the sum and, whole, through
    # its decompression (one fp32 addition per element; no -0 / NaN in these inputs)
    s = x + y
    del x
    po_ = pk.alloc_pici(N, pk.F32)
    pk.reduce_ss(px, py, po_, ws)
    ns = int(torch.count_nonzero(s))
    assert po_.nnz_host() == ns
    _check_pici_tiles(po_, s, tiles)
    out.fill_(float("nan"))
    pk.decompress(po_, out)
    assert torch.equal(out.view(torch.int32), s.view(torch.int32))
    del po_, out

    # reduce_sd in place (y += X) and the workspace reused by a second compress
    pk.reduce_sd(px, y)
    assert torch.equal(y.view(torch.int32), s.view(torch.int32))
    pk.compress(s, py, ws)
    assert py.nnz_host() == ns
    _check_pici_tiles(py, s, tiles[::4])


def test_coo_at_max_n(mods):
    _, ck = mods
    x = wl.scattered_buffer(N, 40_000_000, seed=2, dense_tiles=DENSE_TILES)
    ws = ck.alloc_workspace(N)
    cx = ck.alloc_coo(N)
    ck.compress(x, cx, ws)
    nx = int(torch.count_nonzero(x))
    assert cx.nnz_host() == nx
    pos = cx.idx[:nx].to(torch.int64) & 0xFFFFFFFF          # idx holds uint32 bit patterns
    assert bool(torch.all(pos[1:] > pos[:-1])), "indices ascending and distinct"
    assert torch.equal(x[pos].view(torch.int32), cx.val[:nx].view(torch.int32))
    for t in _sample_tiles(5)[::3]:           # the entries of a tile against the oracle's compress of that tile
        want = co.compress(_tile_bits(x, t))
        lo = int(torch.searchsorted(pos, t * TILE))
        got_i = (pos[lo:lo + want.nnz] - t * TILE).cpu().numpy().astype(np.uint32)
        got_v = cx.val[lo:lo + want.nnz].cpu().view(torch.int32).numpy().view(np.uint32)
        assert np.array_equal(got_i, want.idx) and np.array_equal(got_v, want.val), f"tile {t}"
    del pos
    out = torch.empty_like(x)
    out.fill_(float("nan"))
    ck.decompress(cx, out, ws)
    assert torch.equal(out.view(torch.int32), x.view(torch.int32))
    del out
    acc = torch.ones_like(x)
    ck.reduce_sd(cx, acc)
    x += 1.0
    assert torch.equal(acc.view(torch.int32), x.view(torch.int32))
    del acc, x
    # the merge at this size: X + X (every entry has a partner, nothing cancels) = the same indices, doubled values
    co_ = ck.alloc_coo(N)
    ck.reduce_ss(cx, cx, co_, ws)
    assert co_.nnz_host() == nx
    assert torch.equal(co_.idx[:nx], cx.idx[:nx])
    assert torch.equal(co_.val[:nx], cx.val[:nx] * 2.0)


def test_pici_bf16_at_max_n(mods):
    pk, _ = mods
    x = wl.scattered_buffer(N, 30_000_000, seed=4, dense_tiles=DENSE_TILES).to(torch.bfloat16)
    ws = pk.alloc_workspace(N)
    px = pk.alloc_pici(N, pk.BF16)
    pk.compress(x, px, ws)
    nx = int(torch.count_nonzero(x))
    assert px.nnz_host() == nx
    I = px.I[:T + 1].cpu().numpy().view(np.uint32).astype(np.int64)
    assert I[0] == 0 and I[T] == nx and np.all(np.diff(I) >= 0) and np.all(np.diff(I) <= TILE)
    for t in _sample_tiles(6):
        bits = x[t * TILE:min(N, (t + 1) * TILE)].cpu().view(torch.int16).numpy().view(np.uint16)
        want = po.compress(bits, "bf16")
        assert np.array_equal(px.B[64 * t:64 * (t + 1)].cpu().numpy().view(np.uint64), want.B), f"tile {t}: bitvector"
        A = px.A[int(I[t]):int(I[t + 1])].cpu().view(torch.int16).numpy().view(np.uint16)
        assert np.array_equal(A, want.A), f"tile {t}: values"
    out = torch.full_like(x, float("nan"))
    pk.decompress(px, out)
    assert torch.equal(out.view(torch.int16), x.view(torch.int16))
    y = torch.ones_like(x)
    pk.reduce_sd(px, y)
    assert torch.equal(y.view(torch.int16), (x + 1.0).view(torch.int16))
