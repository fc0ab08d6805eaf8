"""ctypes binding of libkvpool.so — same names as include/kvpool.h (+ include/kvpool_dev.h), argument marshalling only.

Every step of the path runs inside the library's CUDA kernels / stream choreography; nothing here
computes.  There is no fallback: if libkvpool.so is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_int32, c_uint8, c_uint32, c_uint64, c_void_p
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkvpool.so")

MAX_DEVICES = 32
OK, EINVAL, ENOMEM, ECUDA, ENUMA, ESTATE, ENOENT, EIO = 0, -1, -2, -3, -4, -5, -6, -7
DEV_WRITE_COMBINED, DEV_NUMA_STRICT, DEV_HBM, DEV_CUDA_HOSTALLOC, DEV_SSD = 1, 2, 4, 8, 16
TYPE_MEM, TYPE_SSD, TYPE_HBM = 0, 1, 2
NUMA_AUTO = -2
MEASURE_RETRIEVE, MEASURE_OFFLOAD, MEASURE_KERNEL_RETRIEVE, MEASURE_KERNEL_OFFLOAD = 0, 1, 2, 3
PROFILE_OFF, PROFILE_SIDE, PROFILE_INSTREAM = 0, 1, 2
PATH_AUTO, PATH_STAGED, PATH_ZEROCOPY, PATH_HYBRID = 0, 1, 2, 3
KERNEL_VEC16, KERNEL_BULK = 0, 1
_ERRNAMES = {EINVAL: "EINVAL", ENOMEM: "ENOMEM", ECUDA: "ECUDA", ENUMA: "ENUMA", ESTATE: "ESTATE", ENOENT: "ENOENT", EIO: "EIO"}

EXPORTS = [
    "kvpool_plan_weights", "kvpool_plan_layer", "kvpool_plan_lba_range", "kvpool_ssd_range", "kvpool_ssd_location", "kvpool_ssd_info", "kvpool_io_errors", "kvpool_create", "kvpool_destroy", "kvpool_set_bandwidth",
    "kvpool_measure_bandwidth", "kvpool_share_bandwidth", "kvpool_calibrate", "kvpool_bandwidths", "kvpool_set_path", "kvpool_set_tuning", "kvpool_get_tuning", "kvpool_reserve_staging", "kvpool_place", "kvpool_release", "kvpool_set_tables",
    "kvpool_offload", "kvpool_retrieve", "kvpool_retrieve_range", "kvpool_offload_range", "kvpool_offload_layers", "kvpool_retrieve_layers", "kvpool_retrieve_layers_signal", "kvpool_offload_naive", "kvpool_retrieve_naive", "kvpool_wait_offloads", "kvpool_synchronize", "kvpool_pack", "kvpool_unpack", "kvpool_pack_static", "kvpool_checksum", "kvpool_checksum_layers", "kvpool_spin",
    "kvpool_n_devices", "kvpool_weights", "kvpool_device_info", "kvpool_device_type", "kvpool_counts", "kvpool_lookup", "kvpool_stripe", "kvpool_stripe_read",
    "kvpool_glt_bind", "kvpool_glt_find", "kvpool_layer_map", "kvpool_stats", "kvpool_set_profiling", "kvpool_profile_read", "kvpool_profile_read_clock", "kvpool_validate_table", "kvpool_set_table_check", "kvpool_table_errors", "kvpool_last_error", "kvpool_version",
]


class DeviceDesc(ctypes.Structure):
    _fields_ = [("bandwidth_gbps", c_double), ("capacity_bytes", c_uint64), ("numa_node", c_int32), ("flags", c_uint32),
                ("gpu", c_int32), ("link_group", c_uint32), ("path", c_char_p), ("sector_bytes", c_uint32), ("reserved", c_uint32)]


class Geometry(ctypes.Structure):
    _fields_ = [("n_layers", c_uint32), ("block_tokens", c_uint32), ("n_kv_heads", c_uint32), ("head_dim", c_uint32),
                ("elem_bytes", c_uint32)]


class Tuning(ctypes.Structure):
    _fields_ = [("kernel", c_uint32), ("link_kernel", c_uint32), ("hbm_ctas", c_uint32), ("link_ctas", c_uint32), ("bulk_chunk", c_uint32),
                ("bulk_stages", c_uint32), ("bulk_warps", c_uint32), ("stage_slots", c_uint32),
                ("vec_threads", c_uint32), ("vec_unroll", c_uint32), ("auto_threshold_bytes", c_uint64), ("group_bytes", c_uint64),
                ("stage_chunk_bytes", c_uint64), ("pdl", c_uint32), ("ssd_lanes", c_uint32), ("ssd_chunk_bytes", c_uint64)]


class KvPoolError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"kvpool {_ERRNAMES.get(code, code)}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libkvpool.so (loudly: no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing — build it with `python -m paper_2606_14779_b200.build`; "
                              "there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        L.kvpool_last_error.restype = c_char_p
        L.kvpool_version.restype = c_char_p
        vp = c_void_p
        sig = {
            "kvpool_plan_weights": [vp, c_uint32, vp],
            "kvpool_plan_layer": [vp, c_uint32, c_uint64, vp, vp, vp],
            "kvpool_plan_lba_range": [c_uint64, c_uint64, c_uint32, POINTER(c_uint64)],
            "kvpool_ssd_range": [vp, c_uint32, c_uint32, POINTER(c_uint64), POINTER(c_uint64), POINTER(c_uint32)],
            "kvpool_ssd_location": [vp, c_uint32, c_uint32, POINTER(c_uint64), POINTER(c_uint32)],
            "kvpool_ssd_info": [vp, c_uint32, POINTER(c_uint32), POINTER(c_int32), POINTER(c_int32), POINTER(c_uint64), POINTER(c_uint64), POINTER(c_uint32)],
            "kvpool_validate_table": [vp, c_uint64, c_uint64],
            "kvpool_set_table_check": [vp, c_uint64],
            "kvpool_table_errors": [vp, vp],
            "kvpool_create": [vp, c_uint32, vp, c_int, c_uint32, POINTER(vp)],
            "kvpool_destroy": [vp],
            "kvpool_set_bandwidth": [vp, vp],
            "kvpool_measure_bandwidth": [vp, c_uint32, c_int, c_uint64, c_uint32, POINTER(c_double)],
            "kvpool_share_bandwidth": [vp, vp, c_uint32, vp],
            "kvpool_calibrate": [vp, c_int, c_uint64, c_uint32, vp],
            "kvpool_bandwidths": [vp, vp, vp],
            "kvpool_set_path": [vp, c_int],
            "kvpool_set_tuning": [vp, vp],
            "kvpool_reserve_staging": [vp, c_uint64],
            "kvpool_get_tuning": [vp, vp],
            "kvpool_place": [vp, vp, POINTER(vp)],
            "kvpool_release": [vp, vp],
            "kvpool_set_tables": [vp, vp, vp, c_uint64, vp],
            "kvpool_offload": [vp, vp, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_retrieve": [vp, vp, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_retrieve_range": [vp, vp, c_uint32, c_uint32, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_offload_range": [vp, vp, c_uint32, c_uint32, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_offload_layers": [vp, vp, c_uint32, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_retrieve_layers": [vp, vp, c_uint32, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_retrieve_layers_signal": [vp, vp, c_uint32, c_uint32, vp, vp, c_uint64, vp, vp, vp],
            "kvpool_offload_naive": [vp, vp, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_retrieve_naive": [vp, vp, c_uint32, vp, vp, c_uint64, vp, vp],
            "kvpool_wait_offloads": [vp, vp, vp],
            "kvpool_synchronize": [vp],
            "kvpool_pack": [vp, vp, c_uint32, vp, vp, c_uint64, vp, vp, vp],
            "kvpool_unpack": [vp, vp, c_uint32, vp, vp, c_uint64, vp, vp, vp],
            "kvpool_pack_static": [vp, c_uint32, POINTER(Geometry), c_uint32, vp, vp, c_uint64, vp, vp, c_int, vp],
            "kvpool_checksum": [vp, vp, vp, c_uint64, vp, c_uint32, vp, vp],
            "kvpool_checksum_layers": [vp, c_uint32, vp, vp, c_uint64, vp, vp, vp, vp, vp],
            "kvpool_spin": [vp, c_uint64, vp],
            "kvpool_n_devices": [vp, POINTER(c_uint32)],
            "kvpool_weights": [vp, vp],
            "kvpool_device_info": [vp, c_uint32, POINTER(vp), POINTER(c_uint64), POINTER(c_uint64), POINTER(c_int32)],
            "kvpool_io_errors": [vp, POINTER(c_uint64)],
            "kvpool_counts": [vp, c_uint32, vp],
            "kvpool_lookup": [vp, c_uint32, c_uint32, POINTER(c_uint32), POINTER(c_uint32), POINTER(c_uint32), POINTER(vp)],
            "kvpool_stripe": [vp, c_uint32, c_uint32, POINTER(vp), POINTER(c_uint64)],
            "kvpool_stripe_read": [vp, vp, c_uint32, c_uint32, vp, c_uint64],
            "kvpool_device_type": [vp, c_uint32, POINTER(c_uint32), POINTER(c_int32)],
            "kvpool_glt_bind": [vp, vp, c_uint32, vp],
            "kvpool_glt_find": [vp, c_uint64, POINTER(c_uint64), POINTER(c_uint32), POINTER(c_uint32), POINTER(vp), POINTER(vp),
                                POINTER(c_uint32), POINTER(c_uint32)],
            "kvpool_layer_map": [vp, c_uint32, vp, vp],
            "kvpool_stats": [vp, POINTER(c_uint64), POINTER(c_uint64)],
            "kvpool_set_profiling": [vp, c_int],
            "kvpool_profile_read": [vp, c_int, POINTER(c_double), POINTER(c_uint64), POINTER(c_uint64)],
            "kvpool_profile_read_clock": [vp, c_int, POINTER(c_double), POINTER(c_double), POINTER(c_uint64), POINTER(c_uint64), POINTER(c_uint64)],
        }
        for name, argtypes in sig.items():
            f = getattr(L, name)
            f.restype = c_int
            f.argtypes = argtypes
        _lib = L
    return _lib


def _ck(rc: int) -> None:
    if rc != 0:
        raise KvPoolError(rc, lib().kvpool_last_error().decode())


def _addr(x) -> int:
    """Device/host address of a torch tensor, numpy array, int or None."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def _stream(s) -> int:
    if s is None:
        return 0
    if isinstance(s, int):
        return s
    return s.cuda_stream  # torch.cuda.Stream


def _event(e) -> int:
    """cudaEvent_t handle of a torch.cuda.Event (created on first use), an int handle, or None."""
    if e is None:
        return 0
    if isinstance(e, int):
        return e
    if not e.cuda_event:  # torch creates the CUDA event lazily, on its first record
        e.record()
    return e.cuda_event


# ---- pure host arithmetic ----------------------------------------------------------------------------
def kvpool_plan_weights(bandwidth_gbps: Sequence[float]) -> np.ndarray:
    b = np.ascontiguousarray(bandwidth_gbps, dtype=np.float64)
    w = np.zeros(b.shape[0], dtype=np.uint64)
    _ck(lib().kvpool_plan_weights(b.ctypes.data, b.shape[0], w.ctypes.data))
    return w


def kvpool_plan_layer(w: Sequence[int], K: int, with_map: bool = True):
    w = np.ascontiguousarray(w, dtype=np.uint64)
    counts = np.zeros(w.shape[0], dtype=np.uint32)
    dev = np.zeros(int(K), dtype=np.uint8) if with_map else None
    slot = np.zeros(int(K), dtype=np.uint32) if with_map else None
    _ck(lib().kvpool_plan_layer(w.ctypes.data, w.shape[0], int(K), counts.ctypes.data,
                                dev.ctypes.data if with_map else None, slot.ctypes.data if with_map else None))
    return (counts, dev, slot) if with_map else counts


STATIC_MAX_BLOCKS = 32768


def kvpool_pack_static(w: Sequence[int], K: int, k_base, v_base, block_stride_bytes: int, block_table_dev, stage_dev, *,
                       n_kv_heads: int, head_dim: int, block_tokens: int = 16, elem_bytes: int = 2, cuda_device: int = 0, stream=None) -> None:
    """kvpool_pack without a pool and without any GPU allocation by the library (for code that runs inside an engine which
    owns all of HBM and cannot stall on cudaMalloc): places the K blocks of one layer over the devices of integer weights
    `w` and gathers them into `stage_dev` in stripe order.  The maps live in a fixed array inside the library, shared by
    every call on the GPU: K <= STATIC_MAX_BLOCKS, and calls that could overlap on the GPU must be ordered by the caller."""
    wa = np.ascontiguousarray(w, dtype=np.uint64)
    geom = Geometry(1, block_tokens, n_kv_heads, head_dim, elem_bytes)
    _ck(lib().kvpool_pack_static(wa.ctypes.data, wa.shape[0], byref(geom), int(K), _addr(k_base), _addr(v_base), int(block_stride_bytes),
                                 _addr(block_table_dev), _addr(stage_dev), int(cuda_device), _stream(stream)))


def kvpool_plan_lba_range(set_size: int, kv_size: int, sector_bytes: int) -> int:
    n = c_uint64()
    _ck(lib().kvpool_plan_lba_range(int(set_size), int(kv_size), int(sector_bytes), byref(n)))
    return n.value


def kvpool_share_bandwidth(alone_gbps: Sequence[float], link_group: Sequence[int]) -> np.ndarray:
    a = np.ascontiguousarray(alone_gbps, dtype=np.float64)
    g = np.ascontiguousarray(link_group, dtype=np.uint32)
    assert a.shape == g.shape
    out = np.zeros(a.shape[0], dtype=np.float64)
    _ck(lib().kvpool_share_bandwidth(a.ctypes.data, g.ctypes.data, a.shape[0], out.ctypes.data))
    return out


def kvpool_validate_table(table: np.ndarray, nphys: int) -> None:
    """Raises KvPoolError(EINVAL) unless `table` (host int32) names distinct physical blocks in [0, nphys)."""
    t = np.ascontiguousarray(table, dtype=np.int32)
    _ck(lib().kvpool_validate_table(t.ctypes.data, t.shape[0], int(nphys)))


# ---- pool ---------------------------------------------------------------------------------------------
class Placement:
    def __init__(self, pool: "KvPool", handle: int, blocks_per_layer: np.ndarray):
        self.pool, self.handle, self.blocks_per_layer = pool, handle, blocks_per_layer

    def counts(self, layer: int) -> np.ndarray:
        c = np.zeros(self.pool.n_devices, dtype=np.uint32)
        _ck(lib().kvpool_counts(self.handle, layer, c.ctypes.data))
        return c

    def layer_map(self, layer: int) -> Tuple[np.ndarray, np.ndarray]:
        K = int(self.blocks_per_layer[layer])
        dev, slot = np.zeros(K, dtype=np.uint8), np.zeros(K, dtype=np.uint32)
        _ck(lib().kvpool_layer_map(self.handle, layer, dev.ctypes.data, slot.ctypes.data))
        return dev, slot

    def lookup(self, layer: int, block: int) -> Tuple[int, int, int, int]:
        d, t, s, p = c_uint32(), c_uint32(), c_uint32(), c_void_p()
        _ck(lib().kvpool_lookup(self.handle, layer, block, byref(d), byref(t), byref(s), byref(p)))
        return d.value, t.value, s.value, p.value or 0

    def stripe_location(self, layer: int, dev: int) -> Tuple[int, int]:
        """(location, nbytes) of the stripe: a host address for a MEM device, a device address for an HBM device."""
        p, n = c_void_p(), c_uint64()
        _ck(lib().kvpool_stripe(self.handle, layer, dev, byref(p), byref(n)))
        return p.value or 0, n.value

    def stripe(self, layer: int, dev: int) -> np.ndarray:
        """The stripe's bytes as uint8: a numpy VIEW of the pinned pool buffer for a MEM device (no copy), a host
        copy made by kvpool_stripe_read for an HBM or SSD device."""
        loc, n = self.stripe_location(layer, dev)
        if n == 0:
            return np.zeros(0, dtype=np.uint8)
        if self.pool.device_type(dev)[0] != TYPE_MEM:
            out = np.empty(n, dtype=np.uint8)
            _ck(lib().kvpool_stripe_read(self.pool.handle, self.handle, layer, dev, out.ctypes.data, n))
            return out
        return np.ctypeslib.as_array(ctypes.cast(loc, POINTER(c_uint8)), shape=(n,))

    def ssd_range(self, layer: int, dev: int) -> Tuple[int, int, int]:
        """(first LBA, sectors, sector bytes) of the stripe's LBA range on an SSD-type device."""
        a, n, sec = c_uint64(), c_uint64(), c_uint32()
        _ck(lib().kvpool_ssd_range(self.handle, layer, dev, byref(a), byref(n), byref(sec)))
        return a.value, n.value, sec.value

    def ssd_location(self, layer: int, block: int) -> Tuple[int, int]:
        """(LBA, byte inside that sector) of a KV cache that lives on an SSD-type device."""
        a, b = c_uint64(), c_uint32()
        _ck(lib().kvpool_ssd_location(self.handle, layer, block, byref(a), byref(b)))
        return a.value, b.value

    def release(self) -> None:
        if self.handle:
            _ck(lib().kvpool_release(self.pool.handle, self.handle))
            self.handle = 0


class KvPool:
    """kvpool_create / kvpool_destroy and the per-layer calls, one method per ABI entry point."""

    def __init__(self, bandwidth_gbps: Sequence[float], capacity_bytes: Sequence[int], *, n_layers: int, n_kv_heads: int,
                 head_dim: int, block_tokens: int = 16, elem_bytes: int = 2, cuda_device: int = 0,
                 numa_nodes: Optional[Sequence[int]] = None, dev_flags: Optional[Sequence[int]] = None,
                 gpus: Optional[Sequence[int]] = None, link_groups: Optional[Sequence[int]] = None,
                 paths: Optional[Sequence[Optional[str]]] = None, sector_bytes: Optional[Sequence[int]] = None):
        n = len(bandwidth_gbps)
        descs = (DeviceDesc * n)()
        for i in range(n):
            descs[i] = DeviceDesc(float(bandwidth_gbps[i]), int(capacity_bytes[i]), int(numa_nodes[i]) if numa_nodes else -1,
                                  int(dev_flags[i]) if dev_flags else 0, int(gpus[i]) if gpus else -1,
                                  int(link_groups[i]) if link_groups else 0,
                                  os.fsencode(paths[i]) if paths and paths[i] else None, int(sector_bytes[i]) if sector_bytes else 0, 0)
        self.geometry = Geometry(n_layers, block_tokens, n_kv_heads, head_dim, elem_bytes)
        self.kvb = block_tokens * n_kv_heads * head_dim * elem_bytes
        self.payload = 2 * self.kvb
        h = c_void_p()
        _ck(lib().kvpool_create(ctypes.addressof(descs), n, ctypes.addressof(self.geometry), cuda_device, 0, byref(h)))
        self.handle = h.value
        self.n_devices = n

    def destroy(self) -> None:
        if getattr(self, "handle", 0):
            _ck(lib().kvpool_destroy(self.handle))
            self.handle = 0

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def set_bandwidth(self, bandwidth_gbps: Sequence[float]) -> None:
        b = np.ascontiguousarray(bandwidth_gbps, dtype=np.float64)
        assert b.shape[0] == self.n_devices
        _ck(lib().kvpool_set_bandwidth(self.handle, b.ctypes.data))

    def measure_bandwidth(self, dev: int, direction: int = 0, nbytes: int = 256 << 20, iters: int = 5) -> float:
        g = c_double()
        _ck(lib().kvpool_measure_bandwidth(self.handle, dev, direction, nbytes, iters, byref(g)))
        return g.value

    def calibrate(self, direction: int = 0, nbytes: int = 256 << 20, iters: int = 5) -> np.ndarray:
        """Measure every device, divide what link groups share, install the result as the pool's bandwidths; returns them."""
        out = np.zeros(self.n_devices, dtype=np.float64)
        _ck(lib().kvpool_calibrate(self.handle, direction, int(nbytes), iters, out.ctypes.data))
        return out

    def bandwidths(self) -> Tuple[np.ndarray, np.ndarray]:
        """(b_i the pool places by, link group of each device)."""
        b, g = np.zeros(self.n_devices, dtype=np.float64), np.zeros(self.n_devices, dtype=np.uint32)
        _ck(lib().kvpool_bandwidths(self.handle, b.ctypes.data, g.ctypes.data))
        return b, g

    def set_path(self, path: int) -> None:
        _ck(lib().kvpool_set_path(self.handle, path))

    def set_tuning(self, **kw) -> None:
        cur = self.get_tuning()
        t = Tuning()
        t.kernel = kw.pop("kernel", cur.kernel)
        t.link_kernel = kw.pop("link_kernel", cur.link_kernel)
        for k, v in kw.items():
            setattr(t, k, v)
        _ck(lib().kvpool_set_tuning(self.handle, ctypes.addressof(t)))

    def get_tuning(self) -> Tuning:
        t = Tuning()
        _ck(lib().kvpool_get_tuning(self.handle, ctypes.addressof(t)))
        return t

    def reserve_staging(self, nbytes: int) -> None:
        _ck(lib().kvpool_reserve_staging(self.handle, int(nbytes)))

    def place(self, blocks_per_layer: Sequence[int]) -> Placement:
        b = np.ascontiguousarray(blocks_per_layer, dtype=np.uint32)
        assert b.shape[0] == self.geometry.n_layers
        h = c_void_p()
        _ck(lib().kvpool_place(self.handle, b.ctypes.data, byref(h)))
        return Placement(self, h.value, b)

    def set_tables(self, pl: Placement, tables_host, stream=None) -> None:
        """tables_host: int32 numpy array / pinned torch tensor / address holding every layer's table back to back."""
        n = int(np.sum(pl.blocks_per_layer))
        if isinstance(tables_host, np.ndarray):
            assert tables_host.dtype == np.int32 and tables_host.flags["C_CONTIGUOUS"] and tables_host.size == n
        _ck(lib().kvpool_set_tables(self.handle, pl.handle, _addr(tables_host), n, _stream(stream)))

    def offload(self, pl: Placement, layer: int, k_base, v_base, block_stride_bytes: int, block_table_dev, stream=None) -> None:
        _ck(lib().kvpool_offload(self.handle, pl.handle, layer, _addr(k_base), _addr(v_base), block_stride_bytes,
                                 _addr(block_table_dev), _stream(stream)))

    def retrieve(self, pl: Placement, layer: int, k_base, v_base, block_stride_bytes: int, block_table_dev, stream=None) -> None:
        _ck(lib().kvpool_retrieve(self.handle, pl.handle, layer, _addr(k_base), _addr(v_base), block_stride_bytes,
                                  _addr(block_table_dev), _stream(stream)))

    def retrieve_range(self, pl: Placement, layer: int, first_block: int, n_blocks: int, k_base, v_base, block_stride_bytes: int,
                       block_table_dev, stream=None) -> None:
        _ck(lib().kvpool_retrieve_range(self.handle, pl.handle, layer, first_block, n_blocks, _addr(k_base), _addr(v_base),
                                        block_stride_bytes, _addr(block_table_dev), _stream(stream)))

    def offload_range(self, pl: Placement, layer: int, first_block: int, n_blocks: int, k_base, v_base, block_stride_bytes: int,
                      block_table_dev, stream=None) -> None:
        _ck(lib().kvpool_offload_range(self.handle, pl.handle, layer, first_block, n_blocks, _addr(k_base), _addr(v_base),
                                       block_stride_bytes, _addr(block_table_dev), _stream(stream)))

    @staticmethod
    def _ptr_array(items) -> "Optional[ctypes.Array]":
        if items is None:               # block_tables=None: the tables uploaded with set_tables
            return None
        return (c_void_p * len(items))(*[_addr(x) or None for x in items])

    def offload_layers(self, pl: Placement, first_layer: int, k_bases, v_bases, block_stride_bytes: int, block_tables, stream=None) -> None:
        n = len(k_bases)
        ka, va, ta = self._ptr_array(k_bases), self._ptr_array(v_bases), self._ptr_array(block_tables)
        _ck(lib().kvpool_offload_layers(self.handle, pl.handle, first_layer, n, ctypes.addressof(ka), ctypes.addressof(va),
                                        block_stride_bytes, ctypes.addressof(ta) if ta is not None else None, _stream(stream)))

    def retrieve_layers(self, pl: Placement, first_layer: int, k_bases, v_bases, block_stride_bytes: int, block_tables, stream=None) -> None:
        n = len(k_bases)
        ka, va, ta = self._ptr_array(k_bases), self._ptr_array(v_bases), self._ptr_array(block_tables)
        _ck(lib().kvpool_retrieve_layers(self.handle, pl.handle, first_layer, n, ctypes.addressof(ka), ctypes.addressof(va),
                                         block_stride_bytes, ctypes.addressof(ta) if ta is not None else None, _stream(stream)))

    def retrieve_layers_signal(self, pl: Placement, first_layer: int, k_bases, v_bases, block_stride_bytes: int, block_tables, layer_ready,
                               stream=None) -> None:
        """layer_ready: one torch.cuda.Event (or raw cudaEvent_t handle, or None) per layer, recorded when that layer is complete."""
        n = len(k_bases)
        ka, va, ta = self._ptr_array(k_bases), self._ptr_array(v_bases), self._ptr_array(block_tables)
        ea = (c_void_p * n)(*[_event(e) for e in layer_ready])
        _ck(lib().kvpool_retrieve_layers_signal(self.handle, pl.handle, first_layer, n, ctypes.addressof(ka), ctypes.addressof(va),
                                                block_stride_bytes, ctypes.addressof(ta) if ta is not None else None, ctypes.addressof(ea), _stream(stream)))

    def offload_naive(self, pl: Placement, layer: int, k_base, v_base, block_stride_bytes: int, block_table_host: np.ndarray, stream=None) -> None:
        t = np.ascontiguousarray(block_table_host, dtype=np.int32)
        _ck(lib().kvpool_offload_naive(self.handle, pl.handle, layer, _addr(k_base), _addr(v_base), block_stride_bytes, t.ctypes.data, _stream(stream)))

    def retrieve_naive(self, pl: Placement, layer: int, k_base, v_base, block_stride_bytes: int, block_table_host: np.ndarray, stream=None) -> None:
        t = np.ascontiguousarray(block_table_host, dtype=np.int32)
        _ck(lib().kvpool_retrieve_naive(self.handle, pl.handle, layer, _addr(k_base), _addr(v_base), block_stride_bytes, t.ctypes.data, _stream(stream)))

    def pack(self, pl: Placement, layer: int, k_base, v_base, block_stride_bytes: int, block_table_dev, stage_dev, stream=None) -> None:
        _ck(lib().kvpool_pack(self.handle, pl.handle, layer, _addr(k_base), _addr(v_base), block_stride_bytes,
                              _addr(block_table_dev), _addr(stage_dev), _stream(stream)))

    def unpack(self, pl: Placement, layer: int, k_base, v_base, block_stride_bytes: int, block_table_dev, stage_dev, stream=None) -> None:
        _ck(lib().kvpool_unpack(self.handle, pl.handle, layer, _addr(k_base), _addr(v_base), block_stride_bytes,
                                _addr(block_table_dev), _addr(stage_dev), _stream(stream)))

    def checksum(self, k_base, v_base, block_stride_bytes: int, block_table_dev, n_blocks: int, sum_dev, stream=None) -> None:
        _ck(lib().kvpool_checksum(self.handle, _addr(k_base), _addr(v_base), block_stride_bytes, _addr(block_table_dev), n_blocks,
                                  _addr(sum_dev), _stream(stream)))

    def checksum_layers(self, k_bases, v_bases, block_stride_bytes: int, block_tables, n_blocks, layer_ready, sums_dev, stream=None) -> None:
        """For every layer q: `stream` waits for layer_ready[q] (torch event / handle / None), then checksums the layer into sums_dev[q]."""
        n = len(k_bases)
        ka, va, ta = self._ptr_array(k_bases), self._ptr_array(v_bases), self._ptr_array(block_tables)
        nb = (c_uint32 * n)(*[int(x) for x in n_blocks])
        ea = (c_void_p * n)(*[_event(e) for e in layer_ready]) if layer_ready is not None else None
        _ck(lib().kvpool_checksum_layers(self.handle, n, ctypes.addressof(ka), ctypes.addressof(va), block_stride_bytes, ctypes.addressof(ta),
                                         ctypes.addressof(nb), ctypes.addressof(ea) if ea is not None else None, _addr(sums_dev), _stream(stream)))

    def spin(self, nanoseconds: int, stream=None) -> None:
        _ck(lib().kvpool_spin(self.handle, int(nanoseconds), _stream(stream)))

    def wait_offloads(self, pl: Placement, stream=None) -> None:
        _ck(lib().kvpool_wait_offloads(self.handle, pl.handle, _stream(stream)))

    def synchronize(self) -> None:
        _ck(lib().kvpool_synchronize(self.handle))

    def glt_bind(self, pl: Placement, layer: int, ids) -> None:
        a = np.ascontiguousarray(ids, dtype=np.uint64)
        assert a.shape[0] == int(pl.blocks_per_layer[layer])
        _ck(lib().kvpool_glt_bind(self.handle, pl.handle, layer, a.ctypes.data))

    def glt_find(self, ident: int) -> dict:
        key, d, t, loc, ph, layer, block = c_uint64(), c_uint32(), c_uint32(), c_void_p(), c_void_p(), c_uint32(), c_uint32()
        _ck(lib().kvpool_glt_find(self.handle, int(ident), byref(key), byref(d), byref(t), byref(loc), byref(ph), byref(layer), byref(block)))
        return {"key": key.value, "device_id": d.value, "type": t.value, "location": loc.value or 0, "placement": ph.value,
                "layer": layer.value, "block": block.value}

    def io_errors(self) -> int:
        """Failed store / retrieve commands of the pool's SSD-type devices since create (non-blocking)."""
        n = c_uint64()
        _ck(lib().kvpool_io_errors(self.handle, byref(n)))
        return n.value

    def weights(self) -> np.ndarray:
        w = np.zeros(self.n_devices, dtype=np.uint64)
        _ck(lib().kvpool_weights(self.handle, w.ctypes.data))
        return w

    def device_info(self, dev: int) -> dict:
        base, cap, used, node = c_void_p(), c_uint64(), c_uint64(), c_int32()
        _ck(lib().kvpool_device_info(self.handle, dev, byref(base), byref(cap), byref(used), byref(node)))
        return {"host_base": base.value, "capacity": cap.value, "used": used.value, "numa_node": node.value}

    def device_type(self, dev: int) -> Tuple[int, int]:
        """(TYPE_MEM | TYPE_SSD | TYPE_HBM, CUDA ordinal holding an HBM device or -1)."""
        t, g = c_uint32(), c_int32()
        _ck(lib().kvpool_device_type(self.handle, dev, byref(t), byref(g)))
        return t.value, g.value

    def ssd_info(self, dev: int) -> dict:
        sec, direct, blk, st, rt, qd = c_uint32(), c_int32(), c_int32(), c_uint64(), c_uint64(), c_uint32()
        _ck(lib().kvpool_ssd_info(self.handle, dev, byref(sec), byref(direct), byref(blk), byref(st), byref(rt), byref(qd)))
        return {"sector_bytes": sec.value, "direct_io": bool(direct.value), "block_device": bool(blk.value), "stores": st.value, "retrieves": rt.value,
                "queue_depth": qd.value}

    def set_table_check(self, nphys: int) -> None:
        _ck(lib().kvpool_set_table_check(self.handle, int(nphys)))

    def table_errors(self) -> int:
        n = c_uint64()
        _ck(lib().kvpool_table_errors(self.handle, byref(n)))
        return n.value

    def stats(self) -> Tuple[int, int]:
        k, m = c_uint64(), c_uint64()
        _ck(lib().kvpool_stats(self.handle, byref(k), byref(m)))
        return k.value, m.value


    PROF_PACK, PROF_UNPACK, PROF_ZC_OFFLOAD, PROF_ZC_RETRIEVE = 0, 1, 2, 3

    def set_profiling(self, enabled) -> None:
        """False / True (= PROFILE_SIDE: timing events on side streams behind non-timing markers) / PROFILE_INSTREAM."""
        _ck(lib().kvpool_set_profiling(self.handle, int(enabled)))

    def profile_read(self, kind: int) -> Tuple[float, int, int]:
        """(total ms, launches, algorithmic bytes) of the profiled kernels of `kind` since the last read."""
        ms, n, b = c_double(), c_uint64(), c_uint64()
        _ck(lib().kvpool_profile_read(self.handle, kind, byref(ms), byref(n), byref(b)))
        return ms.value, n.value, b.value

    def profile_read_clock(self, kind: int) -> Tuple[float, float, int, int, int]:
        """(event ms, in-kernel %globaltimer ms, launches, launches with a device span, algorithmic bytes) since the last read."""
        ms, dms, n, nd, b = c_double(), c_double(), c_uint64(), c_uint64(), c_uint64()
        _ck(lib().kvpool_profile_read_clock(self.handle, kind, byref(ms), byref(dms), byref(n), byref(nd), byref(b)))
        return ms.value, dms.value, n.value, nd.value, b.value


def version() -> str:
    return lib().kvpool_version().decode()
