"""CPU oracle for the unified-KV-pooling hot path — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes access to `kvpool_oracle.c` (plain C, built with gcc on first use).  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import this
package; the product (`paper_2606_14779_b200/`) never does, and this package never imports the product's
CUDA binding.  See the header of `kvpool_oracle.c` for what each function follows in the paper and for
the list of pins; `oracle/exact.py` is a second, exact-rational statement used on tiny inputs.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import List, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kvpool_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile kvpool_oracle.c -> liboracle.so with gcc (plain -O2, no tuning flags)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.run(["gcc", "-O2", "-shared", "-fPIC", "-pthread", "-o", tmp, _SRC], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64, u32, vp = ctypes.c_uint64, ctypes.c_uint32, ctypes.c_void_p
        lib.orc_kv_bytes.restype = u64
        lib.orc_kv_bytes.argtypes = [u64] * 5
        lib.orc_weights.restype = ctypes.c_int
        lib.orc_weights.argtypes = [vp, u32, vp]
        lib.orc_counts.restype = ctypes.c_int
        lib.orc_counts.argtypes = [vp, u32, u64, vp]
        lib.orc_wrr.restype = ctypes.c_int
        lib.orc_wrr.argtypes = [vp, u32, u64, vp, vp]
        for f in (lib.orc_offload_layer, lib.orc_retrieve_layer):
            f.restype = None
            f.argtypes = [vp, vp, u64, u64, vp, u64, vp, vp, vp]
        lib.orc_retrieve_range.restype = None
        lib.orc_retrieve_range.argtypes = [vp, vp, u64, u64, vp, u64, u64, vp, vp, vp]
        lib.orc_offload_range.restype = None
        lib.orc_offload_range.argtypes = [vp, vp, u64, u64, vp, u64, u64, vp, vp, vp]
        lib.orc_checksum.restype = u64
        lib.orc_checksum.argtypes = [vp, vp, u64, u64, vp, u64]
        lib.orc_layer_parallel.restype = ctypes.c_int
        lib.orc_layer_parallel.argtypes = [ctypes.c_int, vp, vp, u64, u64, vp, u64, vp, vp, vp, u32]
        lib.orc_lba_range_len.restype = u64
        lib.orc_lba_range_len.argtypes = [u64, u64, u64]
        lib.orc_ssd_direct_store.restype = u64
        lib.orc_ssd_direct_store.argtypes = [vp, u64, u64, u64, vp, u64, u64]
        lib.orc_ssd_location.restype = None
        lib.orc_ssd_location.argtypes = [u64, u64, u64, u64, vp, vp]
        lib.orc_ssd_direct_retrieve.restype = None
        lib.orc_ssd_direct_retrieve.argtypes = [vp, u64, u64, u64, vp, u64]
        _lib = lib
    return _lib


def _ptr(a: np.ndarray) -> int:
    return a.ctypes.data


def kv_bytes(n_layers: int, n_kv_heads: int, head_dim: int, elem_bytes: int, tokens: int) -> int:
    return int(_load().orc_kv_bytes(n_layers, n_kv_heads, head_dim, elem_bytes, tokens))


def weights(bandwidth_gbps: Sequence[float]) -> np.ndarray:
    b = np.ascontiguousarray(bandwidth_gbps, dtype=np.float64)
    w = np.zeros(b.shape[0], dtype=np.uint64)
    if _load().orc_weights(_ptr(b), b.shape[0], _ptr(w)) != 0:
        raise ValueError("bandwidth must be positive (weight >= 1 MB/s)")
    return w


def counts(w: Sequence[int], K: int) -> np.ndarray:
    w = np.ascontiguousarray(w, dtype=np.uint64)
    c = np.zeros(w.shape[0], dtype=np.uint32)
    if _load().orc_counts(_ptr(w), w.shape[0], int(K), _ptr(c)) != 0:
        raise ValueError("orc_counts: bad arguments")
    return c


def wrr(c: Sequence[int], K: int) -> Tuple[np.ndarray, np.ndarray]:
    c = np.ascontiguousarray(c, dtype=np.uint32)
    dev = np.zeros(int(K), dtype=np.uint32)
    slot = np.zeros(int(K), dtype=np.uint32)
    if _load().orc_wrr(_ptr(c), c.shape[0], int(K), _ptr(dev), _ptr(slot)) != 0:
        raise ValueError("orc_wrr: counts do not sum to K")
    return dev, slot


@dataclass
class LayerPlacement:
    counts: np.ndarray   # uint32[N]
    dev: np.ndarray      # uint32[K]
    slot: np.ndarray     # uint32[K]


def place(bandwidth_gbps: Sequence[float], blocks_per_layer: Sequence[int]) -> List[LayerPlacement]:
    """Algorithm 1 lines 4-16 applied per layer (R4)."""
    w = weights(bandwidth_gbps)
    out = []
    for K in blocks_per_layer:
        c = counts(w, int(K))
        d, s = wrr(c, int(K))
        out.append(LayerPlacement(c, d, s))
    return out


def _planes(kv_layer: np.ndarray):
    """kv_layer: uint16/uint8 array [2, nphys, block...] C-contiguous -> (K plane ptr, V plane ptr, stride, kvb)."""
    assert kv_layer.flags["C_CONTIGUOUS"] and kv_layer.shape[0] == 2
    plane = kv_layer.nbytes // 2
    kvb = plane // kv_layer.shape[1]
    return _ptr(kv_layer), _ptr(kv_layer) + plane, kvb, kvb


def alloc_stripes(pl: LayerPlacement, payload: int) -> List[np.ndarray]:
    return [np.zeros(int(c) * payload, dtype=np.uint8) for c in pl.counts]


def _stripe_ptrs(stripes: List[np.ndarray]):
    arr = (ctypes.c_void_p * len(stripes))(*[_ptr(s) if s.size else None for s in stripes])
    return arr


def offload_layer(kv_layer: np.ndarray, table: np.ndarray, pl: LayerPlacement, *, parallel: bool = False) -> List[np.ndarray]:
    """MEMSTORE of one layer; returns the N stripes (uint8 arrays of c_i*P bytes)."""
    kp, vp_, stride, kvb = _planes(kv_layer)
    table = np.ascontiguousarray(table, dtype=np.int32)
    assert table.shape[0] == pl.dev.shape[0]
    stripes = alloc_stripes(pl, 2 * kvb)
    ptrs = _stripe_ptrs(stripes)
    lib = _load()
    if parallel:
        rc = lib.orc_layer_parallel(0, kp, vp_, stride, kvb, _ptr(table), table.shape[0], _ptr(pl.dev), _ptr(pl.slot),
                                    ctypes.addressof(ptrs), len(stripes))
        assert rc == 0
    else:
        lib.orc_offload_layer(kp, vp_, stride, kvb, _ptr(table), table.shape[0], _ptr(pl.dev), _ptr(pl.slot),
                              ctypes.addressof(ptrs))
    return stripes


def retrieve_layer(kv_layer_out: np.ndarray, table: np.ndarray, pl: LayerPlacement, stripes: List[np.ndarray], *,
                   parallel: bool = False) -> None:
    """KV retrieval of one layer into kv_layer_out (in place)."""
    kp, vp_, stride, kvb = _planes(kv_layer_out)
    table = np.ascontiguousarray(table, dtype=np.int32)
    ptrs = _stripe_ptrs(stripes)
    lib = _load()
    if parallel:
        rc = lib.orc_layer_parallel(1, kp, vp_, stride, kvb, _ptr(table), table.shape[0], _ptr(pl.dev), _ptr(pl.slot),
                                    ctypes.addressof(ptrs), len(stripes))
        assert rc == 0
    else:
        lib.orc_retrieve_layer(kp, vp_, stride, kvb, _ptr(table), table.shape[0], _ptr(pl.dev), _ptr(pl.slot),
                               ctypes.addressof(ptrs))


def retrieve_range(kv_layer_out: np.ndarray, table: np.ndarray, pl: LayerPlacement, stripes: List[np.ndarray], first: int, n: int) -> None:
    """Partial retrieval of logical blocks [first, first+n) of one layer into kv_layer_out (in place)."""
    kp, vp_, stride, kvb = _planes(kv_layer_out)
    table = np.ascontiguousarray(table, dtype=np.int32)
    assert 0 <= first and first + n <= table.shape[0]
    ptrs = _stripe_ptrs(stripes)
    _load().orc_retrieve_range(kp, vp_, stride, kvb, _ptr(table), int(first), int(n), _ptr(pl.dev), _ptr(pl.slot), ctypes.addressof(ptrs))


def offload_range(kv_layer: np.ndarray, table: np.ndarray, pl: LayerPlacement, stripes: List[np.ndarray], first: int, n: int) -> None:
    """Partial offload: logical blocks [first, first+n) of one layer into the given stripes (in place)."""
    kp, vp_, stride, kvb = _planes(kv_layer)
    table = np.ascontiguousarray(table, dtype=np.int32)
    assert 0 <= first and first + n <= table.shape[0] and table.shape[0] == pl.dev.shape[0]
    ptrs = _stripe_ptrs(stripes)
    _load().orc_offload_range(kp, vp_, stride, kvb, _ptr(table), int(first), int(n), _ptr(pl.dev), _ptr(pl.slot), ctypes.addressof(ptrs))


def checksum(kv_layer: np.ndarray, table: np.ndarray) -> int:
    """Position-weighted 64-bit checksum of the blocks table[0..n) of one layer (see orc_checksum)."""
    kp, vp_, stride, kvb = _planes(kv_layer)
    table = np.ascontiguousarray(table, dtype=np.int32)
    return int(_load().orc_checksum(kp, vp_, stride, kvb, _ptr(table), table.shape[0]))


# ---- KV-passthrough: the SSD as an array of sectors ------------------------------------------------
def lba_range_len(set_size: int, kv_size: int, sector_size: int) -> int:
    """ceil(|offload_set| * KV_size / sector_size) sectors."""
    return int(_load().orc_lba_range_len(int(set_size), int(kv_size), int(sector_size)))


def ssd_direct_store(disk: np.ndarray, sector_size: int, first_lba: int, stripe: np.ndarray, kv_size: int) -> int:
    """SSD_Direct_Store of one offload set (`stripe`: its payloads in slot order) into `disk` (uint8, a whole number of
    sectors) at first_lba; returns the range length in sectors."""
    assert disk.dtype == np.uint8 and disk.flags["C_CONTIGUOUS"] and disk.nbytes % sector_size == 0
    stripe = np.ascontiguousarray(stripe, dtype=np.uint8)
    assert stripe.nbytes % kv_size == 0
    n = int(_load().orc_ssd_direct_store(_ptr(disk), disk.nbytes // sector_size, int(sector_size), int(first_lba),
                                         _ptr(stripe) if stripe.size else None, stripe.nbytes // kv_size, int(kv_size)))
    if n == 2 ** 64 - 1:
        raise ValueError("the LBA range does not fit the disk")
    return n


def ssd_location(first_lba: int, slot: int, kv_size: int, sector_size: int) -> Tuple[int, int]:
    """GLT location of KV cache `slot` of a set stored at first_lba: (LBA, byte inside that sector)."""
    lba, off = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _load().orc_ssd_location(int(first_lba), int(slot), int(kv_size), int(sector_size), ctypes.addressof(lba), ctypes.addressof(off))
    return int(lba.value), int(off.value)


def ssd_direct_retrieve(disk: np.ndarray, sector_size: int, lba: int, byte_in_sector: int, kv_size: int) -> np.ndarray:
    """SSD_Direct_Retrieve of one KV cache by its GLT location."""
    assert disk.dtype == np.uint8 and disk.flags["C_CONTIGUOUS"]
    out = np.empty(int(kv_size), dtype=np.uint8)
    _load().orc_ssd_direct_retrieve(_ptr(disk), int(sector_size), int(lba), int(byte_in_sector), _ptr(out), int(kv_size))
    return out
