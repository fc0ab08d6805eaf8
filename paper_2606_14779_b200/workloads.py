"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NO arithmetic of the method (no placement ratios, counts, round-robin,
gather or scatter): only shapes, sizes, block tables and KV bit patterns.  It imports neither
`oracle/` nor the CUDA binding, so both sides can draw identical inputs from it.

The five configurations are the ones BASELINE.json lists (recipe: SURVEY.md §8(d), restated in
DESIGN.md §5).  They stand in for the paper's Long Doc QA runs (ref. [19]): the hot
path sees only KV *shapes* and context lengths, never prompt content, so no item of that suite is
needed or reproduced.

KV values are a counter-based stream so that any block can be regenerated on its own, on the CPU
(numpy) or on the GPU (torch), bit-identically:

    word w (64-bit index within a layer plane-pair)  ->  splitmix64(w + layer_seed)  ->  4 x 16-bit
    indices  ->  table lookup in a 65536-entry table of N(0,1) quantiles rounded to bf16.

So the values are N(0,1) distributed (quantised to 2^16 equiprobable quantiles), as the configs ask,
and are compared as raw 16-bit patterns, never as floats.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

BASE_SEED = 14779
POISON_BITS = 0x7FC1          # a bf16 NaN pattern; unused blocks and retrieve destinations
BLOCK_TOKENS = 16
SLIDING_WINDOW_TOKENS = 128   # GPT-OSS-style alternating layers keep only the last 128 tokens

_M64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
_MIX1 = 0xBF58476D1CE4E5B9
_MIX2 = 0x94D049BB133111EB


# ----------------------------------------------------------------------------------------------
# geometry and configurations
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Geometry:
    n_layers: int
    n_kv_heads: int
    head_dim: int
    block_tokens: int = BLOCK_TOKENS
    elem_bytes: int = 2

    @property
    def kvb(self) -> int:
        """Bytes of one K (or one V) block of one layer."""
        return self.block_tokens * self.n_kv_heads * self.head_dim * self.elem_bytes

    @property
    def payload(self) -> int:
        """P: pool payload of one (layer, block) = K block then V block."""
        return 2 * self.kvb


@dataclass
class Request:
    """One request: its logical->physical block table and what part of it is offloaded."""
    table: np.ndarray                 # int32[n_blocks], logical -> physical
    retained_prefix: int = 0          # first blocks stay in HBM (cfg 5)

    @property
    def n_blocks(self) -> int:
        return int(self.table.shape[0])


@dataclass
class Workload:
    cfg: int
    name: str
    geom: Geometry
    context_tokens: Sequence[int]
    nphys: int
    requests: List[Request]
    n_pool_devices: int
    weights: Optional[Tuple[float, ...]]     # None -> measured per-buffer bandwidth (bench) / equal (parity)
    sliding_layers: Tuple[int, ...] = field(default_factory=tuple)
    n_streams: int = 1

    # what a layer moves for a request: (first logical block, number of blocks)
    def layer_span(self, req: int, layer: int) -> Tuple[int, int]:
        r = self.requests[req]
        if layer in self.sliding_layers:
            k = min(SLIDING_WINDOW_TOKENS // self.geom.block_tokens, r.n_blocks)
            return r.n_blocks - k, k
        return r.retained_prefix, r.n_blocks - r.retained_prefix

    def blocks_per_layer(self, req: int) -> np.ndarray:
        return np.array([self.layer_span(req, l)[1] for l in range(self.geom.n_layers)], dtype=np.uint32)

    def layer_table(self, req: int, layer: int) -> np.ndarray:
        s, k = self.layer_span(req, layer)
        return self.requests[req].table[s:s + k]

    def moved_bytes(self) -> int:
        return sum(int(self.blocks_per_layer(r).sum()) for r in range(len(self.requests))) * self.geom.payload

    def plane_bytes(self) -> int:
        """Bytes of one K (or V) plane of one layer: nphys blocks."""
        return self.nphys * self.geom.kvb

    def default_weights(self) -> Tuple[float, ...]:
        return self.weights if self.weights is not None else tuple([1.0] * self.n_pool_devices)


LLAMA_8B = Geometry(n_layers=32, n_kv_heads=8, head_dim=128)
GPT_OSS_20B = Geometry(n_layers=24, n_kv_heads=8, head_dim=64)
QWEN3_30B = Geometry(n_layers=48, n_kv_heads=4, head_dim=128)


def _rng(cfg: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(BASE_SEED + cfg))


def make_workload(cfg: int, *, scale: float = 1.0, n_layers: Optional[int] = None) -> Workload:
    """Build configuration `cfg` (1..5 = BASELINE.json configs[0..4]; 6 = LLaMA-8B alone at 128K).

    `scale` < 1 shrinks the context (and the physical pool with it) for tests that need the same
    structure at a size the CPU oracle finishes in seconds; `n_layers` truncates the layer count.
    Neither changes any seed, so the scaled tables are prefixes-in-distribution, not prefixes in value.
    """
    def blocks(tokens: int) -> int:
        return max(1, int(round(tokens * scale)) // BLOCK_TOKENS)

    def geom(g: Geometry) -> Geometry:
        return g if n_layers is None else Geometry(n_layers, g.n_kv_heads, g.head_dim, g.block_tokens, g.elem_bytes)

    rng = _rng(cfg)
    if cfg == 1:
        nb = blocks(1024)
        return Workload(1, "llama3.1-8b@1K", geom(LLAMA_8B), (1024,), nb,
                        [Request(rng.permutation(nb).astype(np.int32))], 2, (2.0, 1.0))
    if cfg == 2:
        nb = blocks(32 * 1024)
        nphys = 2 * nb
        return Workload(2, "llama3.1-8b@32K", geom(LLAMA_8B), (32768,), nphys,
                        [Request(rng.permutation(nphys)[:nb].astype(np.int32))], 4, None)
    if cfg == 3:
        nb = blocks(128 * 1024)
        g = geom(GPT_OSS_20B)
        return Workload(3, "gpt-oss-20b@128K", g, (131072,), nb + nb // 8,
                        [Request(rng.permutation(nb + nb // 8)[:nb].astype(np.int32))], 4, None,
                        sliding_layers=tuple(range(0, g.n_layers, 2)))
    if cfg == 4:
        nb = blocks(128 * 1024)
        nphys = nb + nb // 2
        return Workload(4, "qwen3-30b-a3b@128K", geom(QWEN3_30B), (131072,), nphys,
                        [Request(rng.permutation(nphys)[:nb].astype(np.int32))], 6,
                        (4.0, 4.0, 2.0, 2.0, 1.0, 1.0))
    if cfg == 5:
        ctx = (32768, 65536, 98304, 131072)
        need = [blocks(c) for c in ctx]
        total = sum(need)
        nphys = total + total // 5
        perm = rng.permutation(nphys).astype(np.int32)
        tables: List[List[int]] = [[] for _ in need]
        it = 0
        # deal one physical block at a time, round-robin over the requests that still need blocks
        while any(len(t) < n for t, n in zip(tables, need)):
            for t, n in zip(tables, need):
                if len(t) < n:
                    t.append(int(perm[it]))
                    it += 1
        reqs = [Request(np.array(t, dtype=np.int32), retained_prefix=len(t) // 4) for t in tables]
        return Workload(5, "llama3.1-8b@4x(32K..128K)", geom(LLAMA_8B), ctx, nphys, reqs, 8, None, n_streams=4)
    if cfg == 6:
        nb = blocks(128 * 1024)
        nphys = nb + nb // 2
        return Workload(6, "llama3.1-8b@128K", geom(LLAMA_8B), (131072,), nphys,
                        [Request(rng.permutation(nphys)[:nb].astype(np.int32))], 4, None)
    raise ValueError(f"unknown config {cfg}")


# ----------------------------------------------------------------------------------------------
# counter-based KV values
# ----------------------------------------------------------------------------------------------
_QUANTILES: Optional[np.ndarray] = None


def normal_quantile_table() -> np.ndarray:
    """uint16[65536]: bf16 bit pattern (round-to-nearest-even) of Phi^-1((i + 0.5) / 65536)."""
    global _QUANTILES
    if _QUANTILES is None:
        from scipy.special import ndtri
        q = ndtri((np.arange(65536, dtype=np.float64) + 0.5) / 65536.0).astype(np.float32)
        u = q.view(np.uint32).astype(np.uint64)
        u = (u + 0x7FFF + ((u >> 16) & 1)) >> 16          # fp32 -> bf16, round to nearest even
        _QUANTILES = u.astype(np.uint16)
    return _QUANTILES


def layer_seed(cfg: int, layer: int) -> int:
    return BASE_SEED + 1000 * cfg + layer


def kv_words_numpy(cfg: int, layer: int, first_word: int, n_words: int) -> np.ndarray:
    """uint16[4*n_words]: the KV bit patterns of 64-bit words [first_word, first_word+n_words) of a layer.

    A layer's K plane then V plane, `[2, nphys, T, H, D]`, is one flat array of 16-bit elements; word w
    covers elements 4w..4w+3.
    """
    with np.errstate(over="ignore"):
        z = np.arange(first_word, first_word + n_words, dtype=np.uint64)
        z = z + np.uint64((layer_seed(cfg, layer) * _GOLDEN) & _M64)
        z ^= z >> np.uint64(30)
        z *= np.uint64(_MIX1)
        z ^= z >> np.uint64(27)
        z *= np.uint64(_MIX2)
        z ^= z >> np.uint64(31)
    idx = np.stack([(z >> np.uint64(16 * k)) & np.uint64(0xFFFF) for k in range(4)], axis=1).reshape(-1)
    return normal_quantile_table()[idx.astype(np.int64)]


def kv_block_numpy(wl: Workload, layer: int, plane: int, phys: int) -> np.ndarray:
    """uint16[kvb/2]: bit patterns of physical block `phys` of plane 0 (K) or 1 (V)."""
    elems = wl.geom.kvb // 2
    first_elem = (plane * wl.nphys + phys) * elems
    assert first_elem % 4 == 0 and elems % 4 == 0
    return kv_words_numpy(wl.cfg, layer, first_elem // 4, elems // 4)


def kv_layer_numpy(wl: Workload, layer: int) -> np.ndarray:
    """uint16[2, nphys, kvb/2] — the whole layer (small configs only)."""
    elems = wl.geom.kvb // 2
    n = 2 * wl.nphys * elems
    return kv_words_numpy(wl.cfg, layer, 0, n // 4).reshape(2, wl.nphys, elems)


def kv_layer_torch(wl: Workload, layer: int, device, out=None):
    """int16 tensor [2, nphys, kvb/2] on `device`, bit-identical to kv_layer_numpy."""
    import torch

    elems = wl.geom.kvb // 2
    n_words = 2 * wl.nphys * elems // 4
    if out is None:
        out = torch.empty((2, wl.nphys, elems), dtype=torch.int16, device=device)
    flat = out.view(-1)
    qt = torch.from_numpy(normal_quantile_table().view(np.int16)).to(device)

    def s64(x: int) -> int:          # python int -> signed 64-bit two's complement
        x &= _M64
        return x - (1 << 64) if x >= (1 << 63) else x

    add = s64(layer_seed(wl.cfg, layer) * _GOLDEN)
    step = 1 << 22                   # words per slab: bounds the int64 temporaries
    for w0 in range(0, n_words, step):
        w1 = min(n_words, w0 + step)
        z = torch.arange(w0, w1, dtype=torch.int64, device=device) + add
        z = z ^ ((z >> 30) & ((1 << 34) - 1))
        z = z * s64(_MIX1)
        z = z ^ ((z >> 27) & ((1 << 37) - 1))
        z = z * s64(_MIX2)
        z = z ^ ((z >> 31) & ((1 << 33) - 1))
        idx = torch.stack([(z >> (16 * k)) & 0xFFFF for k in range(4)], dim=1).reshape(-1)
        flat[4 * w0:4 * w1] = qt[idx]
    return out


def poison_torch(shape, device):
    import torch
    return torch.full(shape, np.int16(np.uint16(POISON_BITS).view(np.int16)).item(), dtype=torch.int16, device=device)


def poison_numpy(shape) -> np.ndarray:
    return np.full(shape, POISON_BITS, dtype=np.uint16)
