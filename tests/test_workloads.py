"""The seeded input generators: structure of the five configurations and CPU-side bit-identity of the KV stream."""
import numpy as np
import pytest
import torch

from paper_2606_14779_b200 import workloads as W


def test_config_shapes_match_baseline_json():
    GiB = 2 ** 30
    wl = W.make_workload(1)
    assert (wl.geom.kvb, wl.geom.payload, wl.nphys, wl.requests[0].n_blocks) == (32768, 65536, 64, 64)
    assert wl.moved_bytes() == 128 * 2 ** 20 and wl.weights == (2.0, 1.0)
    assert sorted(wl.requests[0].table.tolist()) == list(range(64))              # a permutation of 64 blocks
    wl = W.make_workload(2)
    assert wl.moved_bytes() == 4 * GiB and wl.nphys == 4096 and wl.n_pool_devices == 4
    t = wl.requests[0].table
    assert len(set(t.tolist())) == 2048 and t.max() < 4096 and np.any(np.diff(t) < 0)   # fragmented, non-monotone
    wl = W.make_workload(3)
    bpl = wl.blocks_per_layer(0)
    assert list(bpl[:4]) == [8, 8192, 8, 8192] and wl.geom.payload == 32768
    assert np.array_equal(wl.layer_table(0, 0), wl.requests[0].table[-8:])       # sliding window: the LAST 8 blocks
    assert wl.moved_bytes() == 12 * (8192 + 8) * 32768
    wl = W.make_workload(4)
    assert wl.moved_bytes() == 12 * GiB and wl.nphys == 12288 and wl.weights == (4.0, 4.0, 2.0, 2.0, 1.0, 1.0)
    wl = W.make_workload(5)
    assert [r.n_blocks for r in wl.requests] == [2048, 4096, 6144, 8192] and wl.nphys == 24576
    assert [int(wl.blocks_per_layer(r)[0]) for r in range(4)] == [1536, 3072, 4608, 6144]
    allb = np.concatenate([r.table for r in wl.requests])
    assert len(set(allb.tolist())) == 20480                                      # requests share one pool, disjointly
    assert wl.moved_bytes() == 30 * GiB and wl.n_streams == 4
    # interleaved dealing: the first four physical blocks dealt go to the four requests in turn
    assert len({int(r.table[0]) for r in wl.requests}) == 4


def test_scaled_config_keeps_structure():
    wl = W.make_workload(5, scale=1 / 64, n_layers=3)
    assert [r.n_blocks for r in wl.requests] == [32, 64, 96, 128] and wl.geom.n_layers == 3
    assert [r.retained_prefix for r in wl.requests] == [8, 16, 24, 32]


def test_kv_stream_numpy_equals_torch_cpu_and_is_block_addressable():
    wl = W.make_workload(1, n_layers=2)
    a = W.kv_layer_numpy(wl, 1)
    b = W.kv_layer_torch(wl, 1, "cpu").numpy().view(np.uint16)
    assert a.shape == (2, 64, 16384) and np.array_equal(a, b)
    for plane, phys in ((0, 0), (1, 63), (0, 17)):
        assert np.array_equal(W.kv_block_numpy(wl, 1, plane, phys), a[plane, phys])
    assert not np.array_equal(W.kv_layer_numpy(wl, 0), a)                         # layers differ


def test_kv_values_are_standard_normal_bf16():
    wl = W.make_workload(1, n_layers=1)
    bits = W.kv_layer_numpy(wl, 0).reshape(-1)
    x = (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    assert np.all(np.isfinite(x))
    assert abs(x.mean()) < 5e-3 and abs(x.std() - 1.0) < 5e-3
    assert abs(np.mean(np.abs(x) < 1.0) - 0.6827) < 5e-3
    assert W.POISON_BITS not in set(W.normal_quantile_table().tolist())           # poison never occurs as a value
