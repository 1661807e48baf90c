"""Seeded synthetic inputs for the Pici hot path (shared by oracle/ tests and the CUDA path).

This module holds NONE of the method's arithmetic: it only draws sparse dense-format buffers
with the shapes, sizes, value distributions and support structure of the paper's workloads
(SVI-A: "Each element is independently selected to be nonzero with
probability equal to 1 - sigma. Each process uses a distinct pseudorandom seed"), and of
BASELINE.json's five configs as concretised in SURVEY.md S8(d).  Both the CPU oracle and the
CUDA path are handed the SAME bytes produced here.

Rules:
  * always ``where(mask, value, +0.0)`` - never ``value * mask`` (that would create -0.0);
  * stream seed for logical rank r of a config with seed S: ``S*1000 + r``; a mask shared by
    all ranks uses ``S*1000 + 999``;
  * bf16: values are N(0,1) rounded to bf16 (RNE) first, the mask is applied after rounding.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import torch

TILE = 4096  # k = 4096 = 64 x 64 virtual tile

_DTYPES = {"f32": torch.float32, "bf16": torch.bfloat16}


def stream_seed(config_seed: int, rank: int) -> int:
    return config_seed * 1000 + rank


def shared_seed(config_seed: int) -> int:
    return config_seed * 1000 + 999


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def bernoulli_mask(n: int, density: float, seed: int, device="cpu") -> torch.Tensor:
    """Boolean support, each position i.i.d. Bernoulli(density)."""
    g = _gen(seed, device)
    out = torch.empty(n, dtype=torch.bool, device=device)
    step = 1 << 26  # bound the fp32 temporary
    for lo in range(0, n, step):
        hi = min(n, lo + step)
        out[lo:hi] = torch.rand(hi - lo, generator=g, device=device, dtype=torch.float32) < density
    return out


def values(n: int, seed: int, dist: str = "normal", scale: float = 1.0, dtype: str = "f32",
           device="cpu") -> torch.Tensor:
    """Dense value field: 'normal' = N(0, scale^2), 'uniform' = U(-scale, scale)."""
    g = _gen(seed + 7_000_003, device)
    out = torch.empty(n, dtype=_DTYPES[dtype], device=device)
    step = 1 << 26
    for lo in range(0, n, step):
        hi = min(n, lo + step)
        if dist == "normal":
            v = torch.randn(hi - lo, generator=g, device=device, dtype=torch.float32) * scale
        elif dist == "uniform":
            v = (torch.rand(hi - lo, generator=g, device=device, dtype=torch.float32) * 2.0 - 1.0) * scale
        else:
            raise ValueError(dist)
        out[lo:hi] = v.to(_DTYPES[dtype])
    return out


def apply_mask(mask: torch.Tensor, vals: torch.Tensor) -> torch.Tensor:
    """where(mask, value, +0.0): zeros are exact +0.0."""
    return torch.where(mask, vals, torch.zeros((), dtype=vals.dtype, device=vals.device))


def sparse_buffer(n: int, density: float, seed: int, dtype: str = "f32", dist: str = "normal",
                  scale: float = 1.0, device="cpu") -> torch.Tensor:
    """One dense-format buffer with unstructured Bernoulli(density) support (config 2 recipe)."""
    return apply_mask(bernoulli_mask(n, density, seed, device),
                      values(n, seed, dist, scale, dtype, device))


def overlapped_rank_buffers(n: int, ranks: int, common_density: float, private_density: float,
                            config_seed: int, dist: str, scale: float, dtype: str = "f32",
                            device="cpu") -> list[torch.Tensor]:
    """P buffers whose support = (mask shared by all ranks) U (private per-rank mask); values are
    independent per rank (configs 4 and 5)."""
    common = bernoulli_mask(n, common_density, shared_seed(config_seed), device) \
        if common_density > 0 else torch.zeros(n, dtype=torch.bool, device=device)
    out = []
    for r in range(ranks):
        s = stream_seed(config_seed, r)
        m = bernoulli_mask(n, private_density, s, device) | common
        out.append(apply_mask(m, values(n, s, dist, scale, dtype, device)))
    return out


# --------------------------------------------------------------------------------------------
# BASELINE.json configs (SURVEY.md S8(d) "Concrete synthetic inputs")
# --------------------------------------------------------------------------------------------

CONFIG2_SPARSITIES = (0.50, 0.75, 0.90, 0.95, 0.99, 0.999, 0.9999)
CONFIG2_SEEDS = (0, 1, 2, 3, 4)
CONFIG2_N = 1 << 28


@dataclass(frozen=True)
class RingConfig:
    name: str
    ranks: int
    n_per_rank: int          # N: elements in each logical rank's buffer
    common_density: float
    private_density: float
    dist: str
    scale: float
    seed: int = 0

    @property
    def chunk(self) -> int:  # n = N / P, must be a multiple of 4096
        assert self.n_per_rank % (self.ranks * TILE) == 0
        return self.n_per_rank // self.ranks

    def expected_density(self, k: int) -> float:
        """Density of the union of k ranks' supports (Eq. 7 generalised to a shared part)."""
        return 1.0 - (1.0 - self.common_density) * (1.0 - self.private_density) ** k

    def buffers(self, device="cpu", n_per_rank: int | None = None) -> list[torch.Tensor]:
        n = self.n_per_rank if n_per_rank is None else n_per_rank
        return overlapped_rank_buffers(n, self.ranks, self.common_density, self.private_density,
                                       self.seed, self.dist, self.scale, "f32", device)


def config1() -> RingConfig:
    """P=4, fp32, N=2^20 per rank, 99% sparsity independent per rank, N(0,1), seed 0."""
    return RingConfig("config1", 4, 1 << 20, 0.0, 0.01, "normal", 1.0, 0)


def config3(density: float = 0.01) -> RingConfig:
    """P=8, fp32, N=2^26 per rank, independent supports, N(0,1)."""
    return RingConfig("config3", 8, 1 << 26, 0.0, density, "normal", 1.0, 0)


def config4() -> RingConfig:
    """P=8, fp32, N=2^27 per rank, 10% density = 5% shared U private p' = 1 - 0.90/0.95, U(-1,1)."""
    return RingConfig("config4", 8, 1 << 27, 0.05, 1.0 - 0.90 / 0.95, "uniform", 1.0, 0)


CONFIG5_TENSOR_SHAPES = ((4096, 4096),) * 4 + ((4096, 11008),) * 3
CONFIG5_BUCKET = sum(a * b for a, b in CONFIG5_TENSOR_SHAPES)  # 202_375_168 elements
CONFIG5_LAYERS = 8


def config5(layer: int = 0) -> RingConfig:
    """One per-layer gradient bucket (772 MiB fp32), P=8, 5% density with 70% mask overlap:
    shared Bernoulli(0.035) U private Bernoulli(1 - 0.95/0.965), values N(0, 0.02^2).
    i.i.d. positions per tensor concatenated == i.i.d. positions over the bucket."""
    return RingConfig(f"config5.layer{layer}", 8, CONFIG5_BUCKET, 0.035, 1.0 - 0.95 / 0.965,
                      "normal", 0.02, 100 + layer)


def nnz_switch_from_permille(n: int, permille: int) -> int:
    """nnz_switch = ceil(theta * n) with theta in per-mille, integers only."""
    return (n * permille + 999) // 1000


def special_values_f32() -> torch.Tensor:
    """Edge-case payload: +-Inf, NaNs with payloads, subnormals, -0.0, +0.0 (as raw bits)."""
    bits = [0x7F800000, 0xFF800000, 0x7FC00001, 0xFFC12345, 0x7F800001, 0x00000001, 0x807FFFFF,
            0x80000000, 0x00000000, 0x3F800000, 0xBF800000, 0x00800000]
    return torch.tensor([b - (1 << 32) if b >= (1 << 31) else b for b in bits],
                        dtype=torch.int32).view(torch.float32)


def edge_sizes() -> tuple[int, ...]:
    return (0, 1, 63, 64, 65, 4095, 4096, 4097, 8192, 8193, 3 * 4096 + 17)


assert math.isclose(config4().expected_density(1), 0.10, rel_tol=1e-12)


def scattered_buffer(n: int, k: int, seed: int, dense_tiles: tuple[int, ...] = (), tile: int = 4096,
                     device="cuda") -> torch.Tensor:
    """fp32 buffer for the maximum-size cases (n up to 2^32 - 1, where a Bernoulli mask would cost 4 more
    buffers of n): zeros, k values N(0, 1) scattered at uniformly drawn positions (collisions overwrite), the first
    and last element and the elements around every 2^30 boundary set, and the listed tiles filled completely."""
    g = _gen(seed + 11_000_027, device)
    out = torch.zeros(n, dtype=torch.float32, device=device)
    step = 1 << 24
    for lo in range(0, k, step):
        c = min(step, k - lo)
        idx = torch.randint(0, n, (c,), generator=g, device=device, dtype=torch.int64)
        out[idx] = torch.randn(c, generator=g, device=device, dtype=torch.float32)
    edges = [0, n - 1] + [b + d for b in range(1 << 30, n, 1 << 30) for d in (-1, 0, 1) if 0 <= b + d < n]
    out[torch.tensor(edges, device=device)] = 1.5
    for t in dense_tiles:
        lo, hi = t * tile, min(n, (t + 1) * tile)
        if lo < n:
            out[lo:hi] = torch.randn(hi - lo, generator=g, device=device, dtype=torch.float32) + 4.0   # no zeros
    return out
