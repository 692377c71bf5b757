"""Seeded synthetic SLA workloads (the five BASELINE.json configs + edge-case layouts).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's tests/bench.
It holds none of the method's arithmetic: it only draws window lengths and N(0,1) tensors and
rounds them to the I/O dtype.  Recipes follow SURVEY.md §8(d); the paper's own workloads (Waymo
Open Dataset, 0.32 m voxels, 12x12 windows; nuScenes, 20x20 windows -- PAPER.md:137-147) are not in
the container, these scenes take their *shapes* and stand in for them.

All randomness is numpy's PCG64 with fixed seeds (`912000 + c` for the lengths of config c,
`seed*10 + {1:Q,2:K,3:V,4:dO}` for tensors), so both sides see bit-identical inputs.
Everything returned is numpy; torch is not imported here.
"""
from __future__ import annotations

import dataclasses
import numpy as np

SEED_BASE = 912000
DTYPES = ("f32", "f16", "bf16")


@dataclasses.dataclass
class Scene:
    name: str
    lengths: np.ndarray          # int64 [W] window lengths (zeros allowed)
    H: int
    d_h: int
    dtype: str                   # "f32" | "f16" | "bf16"
    scale: float
    seed: int

    @property
    def N(self) -> int:
        return int(self.lengths.sum())

    @property
    def W(self) -> int:
        return int(self.lengths.shape[0])

    @property
    def offsets(self) -> np.ndarray:
        off = np.zeros(self.W + 1, dtype=np.int64)
        np.cumsum(self.lengths, out=off[1:])
        assert off[-1] < 2**31
        return off.astype(np.int32)

    @property
    def window_ids(self) -> np.ndarray:
        return np.repeat(np.arange(self.W, dtype=np.int32), self.lengths)

    def tensor(self, which: str) -> np.ndarray:
        """Draw tensor `which` in {"q","k","v","do"}: float32 values already rounded to self.dtype
        (so float64(oracle input) == exactly what the GPU reads)."""
        idx = {"q": 1, "k": 2, "v": 3, "do": 4}[which]
        rng = np.random.Generator(np.random.PCG64(self.seed * 10 + idx))
        x = rng.standard_normal((self.N, self.H, self.d_h), dtype=np.float32)
        if self.scale != 1.0:
            x *= np.float32(self.scale)
        return round_to_dtype(x, self.dtype)


def round_to_dtype(x: np.ndarray, dtype: str) -> np.ndarray:
    """Round float32 array to the I/O dtype (RNE) and return it widened back to float32."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    if dtype == "f32":
        return x
    if dtype == "f16":
        return x.astype(np.float16).astype(np.float32)
    if dtype == "bf16":
        return bf16_bits_to_f32(f32_to_bf16_bits(x))
    raise ValueError(dtype)


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even; NaN kept quiet."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = (u + np.uint32(0x7FFF) + lsb) >> np.uint32(16)
    nan = np.isnan(x)
    r = np.where(nan, np.uint32(0x7FC0), r)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def _fix_residual(lengths: np.ndarray, total: int, lo: int, hi: int) -> np.ndarray:
    """Add/subtract 1 on the longest windows (that stay inside [lo,hi]) until sum == total."""
    lengths = lengths.astype(np.int64).copy()
    diff = total - int(lengths.sum())
    order = np.argsort(-lengths, kind="stable")
    guard = 0
    while diff != 0:
        step = 1 if diff > 0 else -1
        moved = False
        for i in order:
            if diff == 0:
                break
            nv = lengths[i] + step
            if lo <= nv <= hi:
                lengths[i] = nv
                diff -= step
                moved = True
        guard += 1
        if not moved or guard > 1_000_000:
            raise RuntimeError("cannot fix residual")
    return lengths


def lengths_config0(seed: int = SEED_BASE + 0, N: int = 2000, W: int = 64) -> np.ndarray:
    """Geometric lengths, mean ~31, min 1, re-normalised to sum N (BASELINE.json configs[0])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    p = 1.0 / 31.25
    u = rng.random(W)
    g = 1 + np.floor(np.log(u) / np.log(1.0 - p))
    ln = np.maximum(1, np.rint(g * N / g.sum())).astype(np.int64)
    return _fix_residual(ln, N, 1, N)


def lengths_waymo_like(seed: int, N: int = 60000, grid: int = 39, cap: int = 144,
                       r0: float = 2.6, sigma: float = 0.5) -> np.ndarray:
    """39x39 grid of 12x12-cell windows over a 468x468 BEV grid; occupancy ∝ exp(-r/r0) with
    lognormal jitter, capped at 144; empty windows dropped; row-major window order
    (BASELINE.json configs[1])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    c = (grid - 1) / 2.0
    yy, xx = np.meshgrid(np.arange(grid), np.arange(grid), indexing="ij")
    r = np.sqrt((yy - c) ** 2 + (xx - c) ** 2).ravel()
    n = rng.standard_normal(grid * grid)
    shape = np.exp(-r / r0 + sigma * n)

    def occ(A):
        return np.minimum(cap, np.floor(A * shape)).astype(np.int64)

    lo, hi = 1.0, 1e9
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if occ(mid).sum() >= N:
            hi = mid
        else:
            lo = mid
    ln = occ(hi)
    excess = int(ln.sum()) - N
    assert excess >= 0
    # trim excess by -1 on the largest sub-cap windows
    while excess > 0:
        cand = np.where((ln < cap) & (ln > 1))[0]
        cand = cand[np.argsort(-ln[cand], kind="stable")]
        take = cand[:excess]
        ln[take] -= 1
        excess -= len(take)
    ln = ln[ln > 0]
    assert ln.sum() == N
    return ln


def coords_waymo_like(seed: int, N: int = 60000, batch: int = 1, grid_hw: int = 468, win: int = 12, nz: int = 32,
                      r0: float = 2.6, sigma: float = 0.5, n_outside: int = 0) -> np.ndarray:
    """Voxel coordinates int32[N,4], rows (b, z, y, x), for the sequence preparation: per
    sample, N/batch distinct cells of a grid_hw x grid_hw ground-plane grid, drawn without replacement with
    probability ~ exp(-r/r0) (r = distance of the cell's win x win window from the centre, in windows) times a
    lognormal jitter per window -- the density model of lengths_waymo_like -- then shuffled: a voxeliser emits
    voxels in no particular order.  z is uniform in [0, nz).  The last n_outside rows are moved off the grid
    (b, y or x out of range, both sides), then everything is shuffled again."""
    rng = np.random.Generator(np.random.PCG64(seed))
    g = -(-grid_hw // win)
    c = (g - 1) / 2.0
    yy, xx = np.meshgrid(np.arange(grid_hw), np.arange(grid_hw), indexing="ij")
    wy, wx = yy // win, xx // win
    out = []
    per = [N // batch + (1 if b < N % batch else 0) for b in range(batch)]
    for b in range(batch):
        jitter = np.exp(sigma * rng.standard_normal((g, g)))
        r = np.sqrt((wy - c) ** 2 + (wx - c) ** 2)
        p = (np.exp(-r / r0) * jitter[wy, wx]).ravel()
        p /= p.sum()
        cells = rng.choice(grid_hw * grid_hw, size=per[b], replace=False, p=p)
        co = np.empty((per[b], 4), dtype=np.int32)
        co[:, 0] = b
        co[:, 1] = rng.integers(0, nz, per[b])
        co[:, 2] = cells // grid_hw
        co[:, 3] = cells % grid_hw
        out.append(co)
    co = np.concatenate(out, axis=0) if out else np.empty((0, 4), np.int32)
    co = co[rng.permutation(co.shape[0])]
    for j in range(min(n_outside, co.shape[0])):
        row = co.shape[0] - 1 - j
        col, val = [(0, batch), (0, -1), (2, grid_hw), (2, -1), (3, grid_hw + 7), (3, -2)][j % 6]
        co[row, col] = val
    return np.ascontiguousarray(co[rng.permutation(co.shape[0])])


def lengths_config2(seed: int = SEED_BASE + 2, N: int = 200000, W: int = 4000) -> np.ndarray:
    """Lognormal(3.5, 1.2) lengths clipped to [1,2000], rescaled to sum N."""
    rng = np.random.Generator(np.random.PCG64(seed))
    x = np.exp(3.5 + 1.2 * rng.standard_normal(W))
    s = N / np.clip(np.rint(x), 1, 2000).sum()
    ln = np.clip(np.rint(s * x), 1, 2000).astype(np.int64)
    return _fix_residual(ln, N, 1, 2000)


def lengths_config3(seed: int = SEED_BASE + 3, N: int = 150000, n_small: int = 20000,
                    n_big: int = 4) -> np.ndarray:
    """20 000 windows of length U{1,2,3} + 4 windows sharing the rest; shuffled."""
    rng = np.random.Generator(np.random.PCG64(seed))
    small = rng.integers(1, 4, size=n_small).astype(np.int64)
    rest = N - int(small.sum())
    big = np.full(n_big, rest // n_big, dtype=np.int64)
    big[: rest % n_big] += 1
    ln = np.concatenate([small, big])
    rng.shuffle(ln)
    assert ln.sum() == N
    return ln


def make_config(c: int) -> Scene:
    """The five BASELINE.json configs (0-based)."""
    s = SEED_BASE + c
    if c == 0:
        return Scene("config0_tiny_f32", lengths_config0(s), H=4, d_h=32, dtype="f32", scale=1.0, seed=s)
    if c == 1:
        return Scene("config1_waymo_f16", lengths_waymo_like(s, 60000), H=8, d_h=16, dtype="f16",
                     scale=1.0, seed=s)
    if c == 2:
        return Scene("config2_largewin_bf16", lengths_config2(s), H=8, d_h=32, dtype="bf16",
                     scale=1.0, seed=s)
    if c == 3:
        return Scene("config3_skewed_f16", lengths_config3(s), H=8, d_h=16, dtype="f16", scale=3.0, seed=s)
    if c == 4:
        ln = np.concatenate([lengths_waymo_like(s, 60000), lengths_waymo_like(s + 1, 60000)])
        return Scene("config4_train_f16", ln, H=8, d_h=16, dtype="f16", scale=1.0, seed=s)
    raise ValueError(c)


def make_scene(lengths, H: int, d_h: int, dtype: str, seed: int, scale: float = 1.0,
               name: str = "custom") -> Scene:
    return Scene(name, np.asarray(lengths, dtype=np.int64), H, d_h, dtype, scale, seed)


def shard_windows(lengths: np.ndarray, world: int) -> list[tuple[int, int]]:
    """Partition windows into `world` contiguous ranges balanced by voxel count (SURVEY.md §8e:
    windows are independent, Eq. 2, so sharding needs no collective).
    Returns [(w_begin, w_end)) per rank."""
    off = np.concatenate([[0], np.cumsum(np.asarray(lengths, dtype=np.int64))])
    N = int(off[-1])
    cuts = [0]
    for r in range(1, world):
        target = N * r / world
        w = int(np.searchsorted(off, target, side="left"))
        w = min(max(w, cuts[-1]), len(lengths))
        cuts.append(w)
    cuts.append(len(lengths))
    return [(cuts[i], cuts[i + 1]) for i in range(world)]
