"""Helpers for the GPU parity tests: run one workload through the C ABI and through the oracle on the same
seeded inputs and compare placement, stripe bytes and the retrieved paged tensors bit for bit."""
from __future__ import annotations

from typing import List, Optional, Sequence

import numpy as np
import torch

import oracle
from paper_2606_14779_b200 import binding as kv
from paper_2606_14779_b200 import workloads as W


def make_pool(wl: W.Workload, bandwidth: Optional[Sequence[float]] = None, slack: float = 1.25,
              dev_flags: Optional[Sequence[int]] = None, link_groups: Optional[Sequence[int]] = None,
              gpus: Optional[Sequence[int]] = None) -> kv.KvPool:
    bw = list(bandwidth) if bandwidth is not None else list(wl.default_weights())
    total = wl.moved_bytes()
    share = np.array(bw) / np.sum(bw)
    # each buffer: its bandwidth share of the bytes plus slack for per-layer rounding and 4 KiB stripe alignment
    caps = [int(total * s * slack) + (wl.geom.n_layers * len(wl.requests) + 4) * (wl.geom.payload + 4096) for s in share]
    g = wl.geom
    return kv.KvPool(bw, caps, n_layers=g.n_layers, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim,
                     block_tokens=g.block_tokens, elem_bytes=g.elem_bytes, dev_flags=dev_flags, link_groups=link_groups, gpus=gpus)


def check_placement(pl: kv.Placement, opl: List[oracle.LayerPlacement]) -> None:
    for l, o in enumerate(opl):
        assert np.array_equal(pl.counts(l), o.counts), f"counts differ at layer {l}"
        dev, slot = pl.layer_map(l)
        assert np.array_equal(dev.astype(np.uint32), o.dev), f"dev[] differs at layer {l}"
        assert np.array_equal(slot, o.slot), f"slot[] differs at layer {l}"


def check_glt(pl: kv.Placement, opl: List[oracle.LayerPlacement], payload: int, sample: int = 64) -> None:
    """Table I: (device_id, type, location) of sampled blocks; location == stripe base + slot*P."""
    rng = np.random.default_rng(0)
    for l, o in enumerate(opl):
        K = len(o.dev)
        for j in ([0, K - 1] + list(rng.integers(0, K, size=min(sample, K)))) if K else []:
            d, t, s, ptr = pl.lookup(l, int(j))
            assert (d, t, s) == (int(o.dev[j]), pl.pool.device_type(d)[0], int(o.slot[j]))
            assert ptr == pl.stripe_location(l, d)[0] + s * payload


def run_parity(wl: W.Workload, *, path: int, kernel: int, bandwidth=None, tuning: Optional[dict] = None,
               interleaved_layout: bool = False, streams: int = 1, dev_flags: Optional[Sequence[int]] = None,
               profiling: bool = False, link_groups: Optional[Sequence[int]] = None, gpus: Optional[Sequence[int]] = None) -> dict:
    """Offload every layer of every request, compare stripes with the oracle, retrieve into a poisoned pool,
    compare with the oracle's retrieve and with the source.  Returns a few counters."""
    dev = torch.device("cuda:0")
    g = wl.geom
    elems = g.kvb // 2
    bw = list(bandwidth) if bandwidth is not None else list(wl.default_weights())
    pool = make_pool(wl, bw, dev_flags=dev_flags, link_groups=link_groups, gpus=gpus)
    try:
        pool.set_path(path)
        pool.set_tuning(kernel=kernel, link_kernel=kernel, **(tuning or {}))
        pool.set_profiling(profiling)
        cuda_streams = [torch.cuda.Stream(device=dev) for _ in range(streams)]
        R = len(wl.requests)
        pls = [pool.place(wl.blocks_per_layer(r)) for r in range(R)]
        opls = [oracle.place(bw, wl.blocks_per_layer(r)) for r in range(R)]
        for pl, opl in zip(pls, opls):
            check_placement(pl, opl)
            check_glt(pl, opl, g.payload)
        tables = [[torch.from_numpy(np.ascontiguousarray(wl.layer_table(r, l))).to(dev) for l in range(g.n_layers)] for r in range(R)]

        def planes(t):
            if interleaved_layout:      # [nphys, 2, elems]: K and V of a block adjacent, stride 2*kvb
                return t.data_ptr(), t.data_ptr() + g.kvb, 2 * g.kvb
            return t[0].data_ptr(), t[1].data_ptr(), g.kvb

        def to_device_layout(a: torch.Tensor) -> torch.Tensor:
            return a.permute(1, 0, 2).contiguous() if interleaved_layout else a

        def from_device_layout(a: torch.Tensor) -> torch.Tensor:
            return a.permute(1, 0, 2).contiguous() if interleaved_layout else a

        n_bytes = 0
        for l in range(g.n_layers):
            src_cpu = W.kv_layer_numpy(wl, l)                                     # [2, nphys, elems] uint16
            src = to_device_layout(W.kv_layer_torch(wl, l, dev))
            torch.cuda.synchronize()
            kb, vb, stride = planes(src)
            for r in range(R):
                pool.offload(pls[r], l, kb, vb, stride, tables[r][l], cuda_streams[r % streams])
            for r in range(R):
                pool.wait_offloads(pls[r], cuda_streams[r % streams])
            torch.cuda.synchronize()
            pool.synchronize()
            ostripes = []
            for r in range(R):
                want = oracle.offload_layer(src_cpu, wl.layer_table(r, l), opls[r][l])
                ostripes.append(want)
                for i in range(pool.n_devices):
                    got = pls[r].stripe(l, i)
                    assert got.nbytes == want[i].nbytes
                    assert np.array_equal(got, want[i]), f"stripe bytes differ: layer {l} request {r} device {i}"
                    n_bytes += got.nbytes
            # retrieve into poison
            dst = to_device_layout(W.poison_torch((2, wl.nphys, elems), dev))
            kb, vb, stride = planes(dst)
            torch.cuda.synchronize()
            for r in range(R):
                pool.retrieve(pls[r], l, kb, vb, stride, tables[r][l], cuda_streams[r % streams])
            torch.cuda.synchronize()
            got = from_device_layout(dst).cpu().numpy().view(np.uint16)
            want = W.poison_numpy((2, wl.nphys, elems))
            for r in range(R):
                oracle.retrieve_layer(want, wl.layer_table(r, l), opls[r][l], ostripes[r])
            assert np.array_equal(got, want), f"retrieved layer {l} differs from the oracle"
            used = np.zeros(wl.nphys, bool)
            for r in range(R):
                used[wl.layer_table(r, l)] = True
            assert np.array_equal(got[:, used], src_cpu[:, used])                 # round trip, bit for bit
            assert np.all(got[:, ~used] == W.POISON_BITS)                         # nothing else written
        k, m = pool.stats()
        prof = {kind: pool.profile_read_clock(kind) for kind in range(4)} if profiling else None
        for pl in pls:
            pl.release()
        assert all(pool.device_info(i)["used"] == 0 for i in range(pool.n_devices))
        return {"bytes_compared": n_bytes, "kernels": k, "memcpys": m, "prof": prof}
    finally:
        pool.destroy()
