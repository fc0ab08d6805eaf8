"""GPU parity: the CUDA path, called through the C ABI, against the CPU oracle on the same seeded inputs.
Bit-exact on placement (counts, dev[], slot[]), on every stripe byte after offload and on the whole paged
tensor after retrieve into a poison-filled pool (tolerance: none — integer and byte work only)."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
from paper_2606_14779_b200 import binding as kv
from paper_2606_14779_b200 import build as kvbuild
from paper_2606_14779_b200 import workloads as W

from parity_util import check_placement, make_pool, run_parity

pytestmark = pytest.mark.gpu

PATHS = {"staged": kv.PATH_STAGED, "zerocopy": kv.PATH_ZEROCOPY, "auto": kv.PATH_AUTO, "hybrid": kv.PATH_HYBRID}
KERNELS = {"vec16": kv.KERNEL_VEC16, "bulk": kv.KERNEL_BULK}


@pytest.fixture(scope="module", autouse=True)
def _built():
    kvbuild.build()
    assert torch.cuda.is_available()
    kv.lib()                                    # raises if libkvpool.so is missing: no fallback


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("path", ["staged", "zerocopy"])
def test_config1_llama_1k_all_paths(path, kernel):
    wl = W.make_workload(1)                     # the full config: 32 layers x 64 blocks, 2 buffers 2:1
    out = run_parity(wl, path=PATHS[path], kernel=KERNELS[kernel])
    assert out["bytes_compared"] == 128 << 20
    assert out["kernels"] == 64 and out["memcpys"] == (128 if path == "staged" else 0)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_config2_llama_32k_measured_weights(kernel):
    wl = W.make_workload(2, n_layers=3)         # full 32K context (2048 of 4096 blocks), 4 buffers
    probe = make_pool(wl)
    try:                                        # weights = measured per-buffer H2D bandwidth (R10)
        bw = [probe.measure_bandwidth(i, 0, 64 << 20, 3) for i in range(4)]
    finally:
        probe.destroy()
    assert all(b > 1.0 for b in bw)
    run_parity(wl, path=kv.PATH_STAGED, kernel=KERNELS[kernel], bandwidth=bw)
    run_parity(wl, path=kv.PATH_ZEROCOPY, kernel=KERNELS[kernel], bandwidth=bw)


@pytest.mark.parametrize("path", ["staged", "zerocopy", "auto"])
def test_config3_gptoss_sliding_window_layers(path):
    wl = W.make_workload(3, scale=1 / 8, n_layers=6)     # 1024 blocks; even layers move only the last 8
    assert list(wl.blocks_per_layer(0)) == [8, 1024, 8, 1024, 8, 1024]
    run_parity(wl, path=PATHS[path], kernel=kv.KERNEL_VEC16)
    run_parity(wl, path=PATHS[path], kernel=kv.KERNEL_BULK)


@pytest.mark.parametrize("path", ["staged", "zerocopy", "hybrid"])
def test_config4_qwen3_heterogeneous_weights(path):
    wl = W.make_workload(4, scale=1 / 8, n_layers=4)     # 1024 of 1536 blocks, 6 buffers 4:4:2:2:1:1
    out = run_parity(wl, path=PATHS[path], kernel=kv.KERNEL_VEC16)
    # 32 MiB layers: the hybrid path offloads with the kernel's own stores (no copy) and retrieves through the copy engines
    assert out["kernels"] == 8 and out["memcpys"] == {"staged": 48, "zerocopy": 0, "hybrid": 24}[path]
    run_parity(wl, path=PATHS[path], kernel=kv.KERNEL_BULK)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_hybrid_path_offload_by_kernel_retrieve_by_copy_engine(kernel):
    """KVPOOL_PATH_HYBRID (both directions of the link at once): same stripes and same retrieved tensors
    as every other path, on the batched calls, with ranges, with link groups and with a mixed host / HBM pool."""
    k = KERNELS[kernel]
    _run_batched(W.make_workload(1), kv.PATH_HYBRID, k, expect_kernels=4, expect_memcpys=4)          # 2 groups: 2 zero-copy packs; 2 unpacks + 2 x 2 copies
    run_parity(W.make_workload(3, scale=1 / 8, n_layers=4), path=kv.PATH_HYBRID, kernel=k, link_groups=[1, 1, 1, 1])
    run_parity(W.make_workload(5, scale=1 / 16, n_layers=2), path=kv.PATH_HYBRID, kernel=k, streams=4, tuning={"stage_chunk_bytes": 2 << 20})
    run_parity(W.make_workload(4, scale=1 / 16, n_layers=2), path=kv.PATH_HYBRID, kernel=k, dev_flags=[0, HBM, 0, 0, HBM, 0])
    _retrieve_ranges("hybrid", kernel, {"stage_chunk_bytes": 2 << 20}, None)


@pytest.mark.parametrize("path", ["staged", "zerocopy"])
def test_config5_four_requests_four_streams_retained_prefix(path):
    wl = W.make_workload(5, scale=1 / 16, n_layers=3)    # 128..512 blocks, 25% prefix kept, 8 buffers
    run_parity(wl, path=PATHS[path], kernel=kv.KERNEL_VEC16, streams=4)
    run_parity(wl, path=PATHS[path], kernel=kv.KERNEL_BULK, streams=4, tuning={"stage_slots": 2})


def _custom(geom, nphys, tables, n_dev, weights, cfg=77):
    return W.Workload(cfg, "custom", geom, (0,), nphys, [W.Request(np.asarray(t, dtype=np.int32)) for t in tables], n_dev, weights)


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("path", ["staged", "zerocopy"])
def test_edge_cases_ragged_blocks_small_k_and_layouts(path, kernel):
    rng = np.random.default_rng(5)
    # ragged block size: 16 tokens x 1 head x 80 dims x 2 B = 2560 B (not a multiple of the 4 KiB warp piece)
    g = W.Geometry(n_layers=2, n_kv_heads=1, head_dim=80)
    run_parity(_custom(g, 301, [rng.permutation(301)[:257]], 3, (3.0, 2.0, 1.0)), path=PATHS[path], kernel=KERNELS[kernel])
    # 12 KiB + ragged tail: 16 x 3 x 136 x 2 = 13056 B
    g = W.Geometry(n_layers=1, n_kv_heads=3, head_dim=136)
    run_parity(_custom(g, 97, [rng.permutation(97)[:61]], 5, (5.0, 1.0, 1.0, 3.0, 2.0)), path=PATHS[path], kernel=KERNELS[kernel])
    # smallest legal block (16 B), K < N, one device left empty
    g = W.Geometry(n_layers=1, n_kv_heads=1, head_dim=8, block_tokens=1)
    run_parity(_custom(g, 9, [[7, 2, 5]], 6, (4.0, 4.0, 2.0, 2.0, 1.0, 1.0)), path=PATHS[path], kernel=KERNELS[kernel])
    # one block, one device; identity table over the whole pool; [nphys, 2, ...] layout
    g = W.Geometry(n_layers=1, n_kv_heads=2, head_dim=64)
    run_parity(_custom(g, 4, [[3]], 1, (1.0,)), path=PATHS[path], kernel=KERNELS[kernel])
    run_parity(_custom(g, 128, [np.arange(128)], 2, (1.0, 1.0)), path=PATHS[path], kernel=KERNELS[kernel])
    run_parity(_custom(g, 200, [rng.permutation(200)[:150]], 4, (9.0, 1.0, 1.0, 1.0)), path=PATHS[path], kernel=KERNELS[kernel],
               interleaved_layout=True)
    # the maximum number of pool devices
    run_parity(_custom(g, 700, [rng.permutation(700)[:555]], 32, tuple(float(1 + (i * 7) % 5) for i in range(32))),
               path=PATHS[path], kernel=KERNELS[kernel])


def test_empty_layers_and_state_errors():
    g = W.Geometry(n_layers=3, n_kv_heads=2, head_dim=64)
    wl = _custom(g, 16, [np.arange(16)], 2, (2.0, 1.0))
    pool = make_pool(wl)
    try:
        pl = pool.place([0, 5, 0])
        opl = oracle.place([2.0, 1.0], [0, 5, 0])
        check_placement(pl, opl)
        kvt = W.kv_layer_torch(wl, 1, "cuda:0")
        table = torch.arange(5, dtype=torch.int32, device="cuda:0")
        pool.offload(pl, 0, None, None, g.kvb, None)                        # K_l = 0: no-op, null pointers fine
        pool.retrieve(pl, 0, None, None, g.kvb, None)
        with pytest.raises(kv.KvPoolError) as e:                            # never offloaded
            pool.retrieve(pl, 1, kvt[0], kvt[1], g.kvb, table)
        assert e.value.code == kv.ESTATE
        with pytest.raises(kv.KvPoolError) as e:                            # misaligned base
            pool.offload(pl, 1, kvt[0].data_ptr() + 2, kvt[1], g.kvb, table)
        assert e.value.code == kv.EINVAL
        with pytest.raises(kv.KvPoolError) as e:                            # stride not a multiple of 16
            pool.offload(pl, 1, kvt[0], kvt[1], g.kvb + 8, table)
        assert e.value.code == kv.EINVAL
        with pytest.raises(kv.KvPoolError) as e:                            # layer out of range
            pool.offload(pl, 3, kvt[0], kvt[1], g.kvb, table)
        assert e.value.code == kv.EINVAL
        with pytest.raises(kv.KvPoolError) as e:                            # weights are frozen while placements live
            pool.set_bandwidth([1.0, 1.0])
        assert e.value.code == kv.ESTATE
        pl.release()
        pool.set_bandwidth([1.0, 1.0])
        assert list(pool.weights()) == [1000, 1000]
    finally:
        pool.destroy()


def test_place_does_not_wait_for_work_on_the_legacy_default_stream():
    """kvpool_place uploads its tables on the library's own stream: with the staging ring reserved up front it returns in
    host time while a long kernel still occupies the legacy default stream (a synchronous cudaMemcpy would wait for it)."""
    import time
    g = W.Geometry(n_layers=4, n_kv_heads=2, head_dim=64)
    wl = _custom(g, 600, [np.random.default_rng(41).permutation(600)[:512]], 2, (2.0, 1.0))
    pool = make_pool(wl)
    try:
        pool.set_path(kv.PATH_STAGED)
        pool.reserve_staging(64 << 20)                    # >= max(largest layer, group_bytes): no placement below grows the ring
        torch.cuda.synchronize()
        pool.spin(400_000_000, None)                      # 0.4 s on the legacy default stream
        t0 = time.perf_counter()
        pl = pool.place(wl.blocks_per_layer(0))
        dt = time.perf_counter() - t0
        busy = not torch.cuda.default_stream().query()    # the spin kernel must still be running for the timing to mean anything
        torch.cuda.synchronize()
        assert busy and dt < 0.1, (busy, dt)
        check_placement(pl, oracle.place([2.0, 1.0], wl.blocks_per_layer(0)))
        pl.release()
    finally:
        pool.destroy()
    run_parity(wl, path=kv.PATH_STAGED, kernel=kv.KERNEL_VEC16)


def test_pool_full_is_enomem_with_no_partial_reservation():
    g = W.Geometry(n_layers=4, n_kv_heads=2, head_dim=64)
    pool = kv.KvPool([1.0, 1.0], [64 * g.payload, 64 * g.payload], n_layers=4, n_kv_heads=2, head_dim=64)
    try:
        a = pool.place([32, 32, 32, 32])                                    # 16 blocks per layer per device: fits exactly
        assert [pool.device_info(i)["used"] for i in range(2)] == [64 * g.payload] * 2
        with pytest.raises(kv.KvPoolError) as e:
            pool.place([2, 0, 0, 0])
        assert e.value.code == kv.ENOMEM
        assert [pool.device_info(i)["used"] for i in range(2)] == [64 * g.payload] * 2
        a.release()
        with pytest.raises(kv.KvPoolError) as e:                            # layer 3 does not fit: layers 0-2 rolled back
            pool.place([40, 40, 40, 40])
        assert e.value.code == kv.ENOMEM
        assert [pool.device_info(i)["used"] for i in range(2)] == [0, 0]
        b = pool.place([128, 0, 0, 0])                                      # freed space coalesced back into one range
        b.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_pack_unpack_in_device_stripe_order(kernel):
    """a5 / a8 alone: the staging buffer is the N stripes concatenated in device order."""
    wl = W.make_workload(4, scale=1 / 16, n_layers=2)
    g = wl.geom
    bw = list(wl.default_weights())
    pool = make_pool(wl)
    try:
        pool.set_tuning(kernel=KERNELS[kernel])
        pl = pool.place(wl.blocks_per_layer(0))
        opl = oracle.place(bw, wl.blocks_per_layer(0))
        for l in range(g.n_layers):
            table_np = wl.layer_table(0, l)
            table = torch.from_numpy(np.ascontiguousarray(table_np)).cuda()
            src = W.kv_layer_torch(wl, l, "cuda:0")
            stage = torch.zeros(len(table_np) * g.payload, dtype=torch.uint8, device="cuda:0")
            pool.pack(pl, l, src[0], src[1], g.kvb, table, stage)
            torch.cuda.synchronize()
            want = np.concatenate(oracle.offload_layer(W.kv_layer_numpy(wl, l), table_np, opl[l]))
            assert np.array_equal(stage.cpu().numpy(), want)
            dst = W.poison_torch((2, wl.nphys, g.kvb // 2), "cuda:0")
            pool.unpack(pl, l, dst[0], dst[1], g.kvb, table, stage)
            torch.cuda.synchronize()
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_layer(ref, table_np, opl[l], oracle.offload_layer(W.kv_layer_numpy(wl, l), table_np, opl[l]))
            assert np.array_equal(dst.cpu().numpy().view(np.uint16), ref)
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_profiling_keeps_parity_and_reports_event_and_kernel_clock_spans(kernel):
    """With profiling on the kernels also fold their start/end (%globaltimer) into a per-launch span: results must stay
    bit-exact on both paths, every launch gets a span, and a launch's own span cannot exceed the event pair around it
    by more than the clocks' granularity."""
    wl = W.make_workload(4, scale=1 / 8, n_layers=4)
    for path in (kv.PATH_STAGED, kv.PATH_ZEROCOPY):
        out = run_parity(wl, path=path, kernel=KERNELS[kernel], profiling=True)
        prof = out["prof"]
        pack_kind, unpack_kind = (kv.KvPool.PROF_PACK, kv.KvPool.PROF_UNPACK) if path == kv.PATH_STAGED else (kv.KvPool.PROF_ZC_OFFLOAD, kv.KvPool.PROF_ZC_RETRIEVE)
        for kind in range(4):
            ms, dms, n, nd, b = prof[kind]
            if kind in (pack_kind, unpack_kind):
                assert n == nd == wl.geom.n_layers and b == sum(int(k) for k in wl.blocks_per_layer(0)) * wl.geom.payload
                assert 0.0 < dms <= ms + 0.02 * n, (ms, dms)          # events bracket the kernel; 20 us per launch of clock slack
            else:
                assert (ms, dms, n, nd, b) == (0.0, 0.0, 0, 0, 0)


def test_kv_stream_is_identical_on_cpu_and_gpu():
    wl = W.make_workload(2, n_layers=1)
    a = W.kv_layer_torch(wl, 0, "cuda:0").cpu().numpy().view(np.uint16)
    rng = np.random.default_rng(3)
    for plane, phys in [(0, 0), (1, wl.nphys - 1)] + [(int(rng.integers(0, 2)), int(rng.integers(0, wl.nphys))) for _ in range(32)]:
        assert np.array_equal(a[plane, phys], W.kv_block_numpy(wl, 0, plane, phys))


# (cfg, path, kernel): every BASELINE.json configuration at its FULL size on the default path and kernel — what bench.py
# times — plus the hand-written link path with the cp.async.bulk kernel on the two largest per-layer launches (config 4,
# the headline, and config 6, 512 MiB per layer), the two remaining path x kernel combinations on the headline config, and the
# hybrid path on config 6 (whose 512 MiB layers retrieve through DEVICE-MAJOR chunks, as on the default path: the ring's
# slots hold 256 MiB).
FULL_SIZE_CASES = [(2, "auto", "vec16"), (3, "auto", "vec16"), (4, "auto", "vec16"), (5, "auto", "vec16"), (6, "auto", "vec16"),
                   (4, "zerocopy", "bulk"), (6, "zerocopy", "bulk"), (4, "auto", "bulk"), (4, "zerocopy", "vec16"), (3, "zerocopy", "bulk"),
                   (6, "hybrid", "bulk")]


@pytest.mark.parametrize("cfg,path,kernel", FULL_SIZE_CASES)
def test_full_size_configs_every_byte_against_oracle(cfg, path, kernel):
    """BASELINE.json's full sizes in bench.py's launch configuration (batched calls over all layers, one stream per
    request, every layer resident in HBM), compared with the oracle BYTE FOR BYTE, streamed layer by layer so that host
    memory holds one layer and its stripes at a time: the full placement; every byte of every stripe
    against orc_offload_layer of the same seeded layer; the whole retrieved tensor (request blocks, retained prefixes,
    free blocks) against orc_retrieve_layer into poison.  PAPER.md:240-245: every KV cache is stored and read back
    through its GLT entry.  The oracle's input is the seeded generator's layer (workloads.kv_layer_torch, spot-checked
    here against its numpy form block by block); nothing the library wrote is ever an expected value."""
    wl = W.make_workload(cfg)
    g, dev, R, L = wl.geom, torch.device("cuda:0"), len(wl.requests), wl.geom.n_layers
    bw = list(wl.default_weights())
    pool = make_pool(wl)
    try:
        pool.set_path(PATHS[path])
        pool.set_tuning(kernel=KERNELS[kernel], link_kernel=KERNELS[kernel])
        bpl = [wl.blocks_per_layer(r) for r in range(R)]
        pls = [pool.place(bpl[r]) for r in range(R)]
        opls = [oracle.place(bw, bpl[r]) for r in range(R)]
        for r in range(R):
            check_placement(pls[r], opls[r])
        table_np = [[np.ascontiguousarray(wl.layer_table(r, l)) for l in range(L)] for r in range(R)]
        tables = [[torch.from_numpy(t).to(dev) for t in row] for row in table_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for l in range(L)]
        torch.cuda.synchronize()                                                  # inputs were generated on the default stream
        streams = [torch.cuda.Stream() for _ in range(R)]
        for r in range(R):
            pool.offload_layers(pls[r], 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables[r], streams[r])
        for r in range(R):
            pool.wait_offloads(pls[r], streams[r])
        torch.cuda.synchronize()
        pool.synchronize()
        for r in range(R):
            pool.retrieve_layers(pls[r], 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables[r], streams[r])
        torch.cuda.synchronize()

        rng = np.random.default_rng(cfg)
        shape = (2, wl.nphys, g.kvb // 2)
        pin_src, pin_got = torch.empty(shape, dtype=torch.int16).pin_memory(), torch.empty(shape, dtype=torch.int16).pin_memory()
        ref = np.empty(shape, dtype=np.uint16)
        stripe_bytes = retrieved_bytes = 0
        for l in range(L):
            pin_src.copy_(src[l], non_blocking=True)
            pin_got.copy_(dst[l], non_blocking=True)
            torch.cuda.synchronize()
            src_cpu, got = pin_src.numpy().view(np.uint16), pin_got.numpy().view(np.uint16)
            for plane, phys in [(0, 0), (1, wl.nphys - 1)] + [(int(rng.integers(0, 2)), int(rng.integers(0, wl.nphys))) for _ in range(2)]:
                assert np.array_equal(src_cpu[plane, phys], W.kv_block_numpy(wl, l, plane, phys)), "the seeded layer differs between numpy and torch"
            ref[...] = W.POISON_BITS
            for r in range(R):
                K = len(table_np[r][l])
                want = oracle.offload_layer(src_cpu, table_np[r][l], opls[r][l], parallel=True)
                for i in range(pool.n_devices):
                    have = pls[r].stripe(l, i)
                    assert have.nbytes == want[i].nbytes == int(opls[r][l].counts[i]) * g.payload
                    assert np.array_equal(have, want[i]), f"stripe bytes differ: request {r} layer {l} device {i}"
                    stripe_bytes += have.nbytes
                    # byte share of every device within one block of its bandwidth share (north star invariant)
                    assert abs(have.nbytes - bw[i] / sum(bw) * K * g.payload) < g.payload
                oracle.retrieve_layer(ref, table_np[r][l], opls[r][l], want, parallel=True)
                retrieved_bytes += K * g.payload
                del want
            assert np.array_equal(got, ref), f"retrieved layer {l} differs from the oracle's (request blocks, retained prefixes or free blocks)"
        assert stripe_bytes == wl.moved_bytes() and retrieved_bytes == wl.moved_bytes()      # every byte of both legs was compared
        for pl in pls:
            pl.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("path", ["staged", "zerocopy"])
def test_retrieve_range_partial_and_prefix(path, kernel):
    """kvpool_retrieve_range against the oracle's partial retrieval: prefix, middle, tail, empty and whole ranges."""
    _retrieve_ranges(path, kernel, {}, None)


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_retrieve_range_larger_than_a_staging_slot_in_device_major_chunks(kernel):
    """The same ranges under a 2 MiB chunk cap (64 blocks per slot; ranges of 128, 256 and 512 blocks travel device-major),
    with the pool devices in link groups (shared I/O streams)."""
    _retrieve_ranges("staged", kernel, {"stage_chunk_bytes": 2 << 20}, [1, 1, 1, 2, 2, 0])


def _retrieve_ranges(path, kernel, tuning, link_groups):
    wl = W.make_workload(4, scale=1 / 16, n_layers=2)          # 512 of 768 blocks, 6 buffers 4:4:2:2:1:1
    g, dev = wl.geom, torch.device("cuda:0")
    bw = list(wl.default_weights())
    pool = make_pool(wl, link_groups=link_groups)
    try:
        pool.set_path(PATHS[path])
        pool.set_tuning(kernel=KERNELS[kernel], link_kernel=KERNELS[kernel], **tuning)
        pl = pool.place(wl.blocks_per_layer(0))
        opl = oracle.place(bw, wl.blocks_per_layer(0))
        rng = np.random.default_rng(13)
        for l in range(g.n_layers):
            table_np = np.ascontiguousarray(wl.layer_table(0, l))
            K = len(table_np)
            table = torch.from_numpy(table_np).to(dev)
            src = W.kv_layer_torch(wl, l, dev)
            src_cpu = W.kv_layer_numpy(wl, l)
            with pytest.raises(kv.KvPoolError) as e:                               # not offloaded yet
                pool.retrieve_range(pl, l, 0, 4, src[0], src[1], g.kvb, table)
            assert e.value.code == kv.ESTATE
            pool.offload(pl, l, src[0], src[1], g.kvb, table)
            pool.wait_offloads(pl)
            torch.cuda.synchronize()
            stripes = oracle.offload_layer(src_cpu, table_np, opl[l])
            ranges = [(0, K // 4), (K // 4, K // 2), (K - 1, 1), (0, K), (7, 0), (K, 0), (0, 1)]
            ranges += [(int(a), int(b)) for a, b in ((rng.integers(0, K), rng.integers(0, 64)) for _ in range(6)) if a + b <= K]
            for first, n in ranges:
                dst = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
                pool.retrieve_range(pl, l, first, n, dst[0], dst[1], g.kvb, table)
                torch.cuda.synchronize()
                want = W.poison_numpy((2, wl.nphys, g.kvb // 2))
                oracle.retrieve_range(want, table_np, opl[l], stripes, first, n)
                assert np.array_equal(dst.cpu().numpy().view(np.uint16), want), (l, first, n)
            with pytest.raises(kv.KvPoolError) as e:                               # range past the end
                pool.retrieve_range(pl, l, K - 2, 3, src[0], src[1], g.kvb, table)
            assert e.value.code == kv.EINVAL
        pl.release()
    finally:
        pool.destroy()


def test_checksum_consumer_matches_oracle_and_detects_round_trip():
    """kvpool_checksum (the consumer stand-in) is bit-exact against the oracle's definition, including ragged block
    sizes, and the checksum of a retrieved layer equals the checksum of the source."""
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(17)
    for g, nphys, n in ((W.Geometry(1, 1, 80), 67, 41), (W.Geometry(1, 3, 136), 33, 33), (W.Geometry(1, 1, 8, block_tokens=1), 9, 5),
                        (W.QWEN3_30B, 1536, 1024)):
        wl = _custom(W.Geometry(2, g.n_kv_heads, g.head_dim, g.block_tokens), nphys, [rng.permutation(nphys)[:n]], 3, (3.0, 2.0, 1.0))
        pool = make_pool(wl)
        try:
            table_np = np.ascontiguousarray(wl.layer_table(0, 0))
            table = torch.from_numpy(table_np).to(dev)
            src = W.kv_layer_torch(wl, 0, dev)
            out = torch.zeros(3, dtype=torch.int64, device=dev)
            pool.checksum(src[0], src[1], wl.geom.kvb, table, n, out[0:1])
            pool.checksum(src[0], src[1], wl.geom.kvb, table, n // 2, out[1:2])
            both = torch.zeros(2, dtype=torch.int64, device=dev)                 # the same two through the one-call layer loop
            pool.checksum_layers([src[0], src[0]], [src[1], src[1]], wl.geom.kvb, [table, table], [n, n // 2], None, both)
            torch.cuda.synchronize()
            assert torch.equal(both, out[0:2])
            want = oracle.checksum(W.kv_layer_numpy(wl, 0), table_np)
            want_half = oracle.checksum(W.kv_layer_numpy(wl, 0), table_np[:n // 2])
            pl = pool.place(wl.blocks_per_layer(0))
            pool.offload(pl, 0, src[0], src[1], wl.geom.kvb, table)
            dst = W.poison_torch((2, nphys, wl.geom.kvb // 2), dev)
            pool.retrieve(pl, 0, dst[0], dst[1], wl.geom.kvb, table)
            pool.checksum(dst[0], dst[1], wl.geom.kvb, table, n, out[2:3])
            torch.cuda.synchronize()
            got = [int(x) % 2 ** 64 for x in out.cpu().tolist()]
            assert got == [want, want_half, want]
            pl.release()
        finally:
            pool.destroy()


def _run_batched(wl, path, kernel, expect_kernels=None, expect_memcpys=None, tuning=None, dev_flags=None, own_tables=False):
    """Offload and retrieve ALL layers with one kvpool_offload_layers / kvpool_retrieve_layers call each and compare
    every stripe and every retrieved layer with the oracle.  own_tables: the block tables reach the GPU through ONE
    kvpool_set_tables upload of the packed host tables and the calls pass block_tables = NULL."""
    dev = torch.device("cuda:0")
    g, L = wl.geom, wl.geom.n_layers
    bw = list(wl.default_weights())
    pool = make_pool(wl, dev_flags=dev_flags)
    try:
        pool.set_path(path)
        pool.set_tuning(kernel=kernel, link_kernel=kernel, **(tuning or {}))
        bpl = wl.blocks_per_layer(0)
        pl = pool.place(bpl)
        opl = oracle.place(bw, bpl)
        check_placement(pl, opl)
        tables_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(L)]
        tables = [torch.from_numpy(t).to(dev) if len(t) else None for t in tables_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for l in range(L)]
        torch.cuda.synchronize()                                                  # inputs were generated on the default stream
        s = torch.cuda.Stream()
        with pytest.raises(kv.KvPoolError) as e:                                  # nothing offloaded yet: ESTATE, nothing enqueued
            pool.retrieve_layers(pl, 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, s)
        assert e.value.code == kv.ESTATE
        k0, m0 = pool.stats()
        if own_tables:
            with pytest.raises(kv.KvPoolError) as e:                              # no tables given and none uploaded
                pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, None, s)
            assert e.value.code == kv.EINVAL
            packed = np.concatenate(tables_np).astype(np.int32)
            with pytest.raises(kv.KvPoolError) as e:                              # wrong entry count
                lib_rc = kv.lib().kvpool_set_tables(pool.handle, pl.handle, packed.ctypes.data, len(packed) + 1, s.cuda_stream)
                kv._ck(lib_rc)
            assert e.value.code == kv.EINVAL
            pool.set_tables(pl, packed, s)
            packed[:] = -1                                                        # the caller's buffer is free again
            tables = None
        pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, s)
        pool.wait_offloads(pl, s)
        pool.retrieve_layers(pl, 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, s)
        s.synchronize()
        k1, m1 = pool.stats()
        if expect_kernels is not None:
            assert k1 - k0 == expect_kernels
        if expect_memcpys is not None:
            assert m1 - m0 == expect_memcpys
        for l in range(L):
            src_cpu = W.kv_layer_numpy(wl, l)
            want = oracle.offload_layer(src_cpu, tables_np[l], opl[l])
            for i in range(pool.n_devices):
                assert np.array_equal(pl.stripe(l, i), want[i]), f"stripe differs: layer {l} device {i}"
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_layer(ref, tables_np[l], opl[l], want)
            assert np.array_equal(dst[l].cpu().numpy().view(np.uint16), ref), f"retrieved layer {l} differs"
            if own_tables and l in (0, L - 1):                                    # the per-layer calls take NULL tables too
                again = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
                torch.cuda.synchronize()
                pool.retrieve(pl, l, again[0], again[1], g.kvb, None, s)
                pool.retrieve_range(pl, l, 0, len(tables_np[l]), again[0], again[1], g.kvb, None, s)
                s.synchronize()
                assert np.array_equal(again.cpu().numpy().view(np.uint16), ref)
        pl.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_batched_layers_grouped_launches(kernel):
    k = KERNELS[kernel]
    # config 1, whole request (32 layers x 4 MiB): two 64 MiB groups, each ONE pack/unpack launch + one copy per device
    _run_batched(W.make_workload(1), kv.PATH_AUTO, k, expect_kernels=4, expect_memcpys=8)
    _run_batched(W.make_workload(1), kv.PATH_ZEROCOPY, k, expect_kernels=4, expect_memcpys=0)     # groups are capped at group_bytes on every path
    _run_batched(W.make_workload(1), kv.PATH_ZEROCOPY, k, expect_kernels=2, expect_memcpys=1, tuning={"group_bytes": 1 << 30}, own_tables=True)
    _run_batched(W.make_workload(1), kv.PATH_AUTO, k, expect_kernels=2, expect_memcpys=0, tuning={"group_bytes": 1 << 30, "auto_threshold_bytes": 1 << 30})   # one group, below the staged threshold
    # sliding-window + full layers (config 3 scaled: 256 KiB and 32 MiB layers alternate): groups {0,1,2} {3,4} {5}
    wl = W.make_workload(3, scale=1 / 8, n_layers=6)
    _run_batched(wl, kv.PATH_AUTO, k, expect_kernels=6, expect_memcpys=24)
    _run_batched(wl, kv.PATH_STAGED, k, expect_kernels=6, expect_memcpys=24)
    _run_batched(wl, kv.PATH_ZEROCOPY, k, expect_kernels=6, expect_memcpys=0)
    _run_batched(wl, kv.PATH_AUTO, k, expect_kernels=6, expect_memcpys=25, own_tables=True)
    _run_batched(wl, kv.PATH_STAGED, k, expect_kernels=12, expect_memcpys=48, tuning={"group_bytes": 1})      # every layer alone
    # more layers than one launch holds (64), 160-byte payloads (stripes need alignment padding inside a group)
    g = W.Geometry(n_layers=150, n_kv_heads=1, head_dim=40, block_tokens=1)
    rng = np.random.default_rng(23)
    wl = W.Workload(78, "many-tiny-layers", g, (0,), 40, [W.Request(rng.permutation(40)[:29].astype(np.int32))], 3, (3.0, 2.0, 1.0),
                    sliding_layers=tuple(range(0, 150, 7)))
    _run_batched(wl, kv.PATH_ZEROCOPY, k, expect_kernels=2 * 3)
    _run_batched(wl, kv.PATH_STAGED, k, expect_kernels=2 * 3, expect_memcpys=2 * 3 * 3)


@pytest.mark.parametrize("path", ["staged", "zerocopy", "auto"])
def test_retrieve_layers_signal_feeds_a_consumer_on_another_stream(path):
    """Layerwise pipelining through ONE batched call: the retrieve stream records a caller-owned event per
    layer; a consumer stream waits on each and checksums that layer straight away.  Every checksum must equal the oracle's
    for the source layer (a consumer that ran before its layer was complete would read poison), and the retrieved tensors
    must equal the oracle's retrieve."""
    dev = torch.device("cuda:0")
    wl = W.make_workload(3, scale=1 / 8, n_layers=6)       # 256 KiB and 32 MiB layers alternate: groups and single layers
    g, L = wl.geom, wl.geom.n_layers
    bw = list(wl.default_weights())
    pool = make_pool(wl)
    try:
        pool.set_path(PATHS[path])
        bpl = list(wl.blocks_per_layer(0))
        bpl[4] = 0                                         # an empty layer in the middle: ready at once, nothing moved
        pl, opl = pool.place(bpl), oracle.place(bw, bpl)
        tables_np = [np.ascontiguousarray(wl.layer_table(0, l))[:bpl[l]] for l in range(L)]
        tables = [torch.from_numpy(t).to(dev) if len(t) else None for t in tables_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for l in range(L)]
        sums = torch.zeros(L, dtype=torch.int64, device=dev)
        torch.cuda.synchronize()
        io, consumer = torch.cuda.Stream(), torch.cuda.Stream()
        pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, io)
        pool.wait_offloads(pl, io)
        ready = [torch.cuda.Event() for _ in range(L)]
        with pytest.raises(kv.KvPoolError) as e:           # validated before anything is enqueued
            pool.retrieve_layers_signal(pl, 0, [d[0] for d in dst], [None] + [d[1] for d in dst][1:], g.kvb, tables, ready, io)
        assert e.value.code == kv.EINVAL
        pool.retrieve_layers_signal(pl, 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, ready, io)
        for l in range(L):                                 # the consumer never synchronises with `io` except through the events
            consumer.wait_event(ready[l])
            if bpl[l]:
                pool.checksum(dst[l][0], dst[l][1], g.kvb, tables[l], bpl[l], sums[l:l + 1], consumer)
        consumer.synchronize()
        got = [int(x) % 2 ** 64 for x in sums.cpu().tolist()]
        want = [oracle.checksum(W.kv_layer_numpy(wl, l), tables_np[l]) if bpl[l] else 0 for l in range(L)]
        assert got == want
        io.synchronize()
        for l in range(L):
            stripes = oracle.offload_layer(W.kv_layer_numpy(wl, l), tables_np[l], opl[l])
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_layer(ref, tables_np[l], opl[l], stripes)
            assert np.array_equal(dst[l].cpu().numpy().view(np.uint16), ref), f"retrieved layer {l} differs"
        pl.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("path", ["staged", "zerocopy", "auto"])
def test_layer_ready_events_fire_layer_by_layer_not_at_the_end_of_the_request(path):
    """Layerwise pipelining is only worth its name if the consumer of layer 0 does not wait for the whole
    request: on every path groups are capped at `group_bytes`, so with eight 32 MiB layers (0.6 ms each over the link)
    ready[0] must fire several layer times before the call's last layer has moved."""
    dev = torch.device("cuda:0")
    wl = W.make_workload(4, scale=1 / 8, n_layers=8)       # 1024 blocks x 32 KiB = 32 MiB per layer
    g, L = wl.geom, wl.geom.n_layers
    pool = make_pool(wl)
    try:
        pool.set_path(PATHS[path])
        pool.set_tuning(group_bytes=16 << 20)              # a 32 MiB layer is a group of its own
        bpl = wl.blocks_per_layer(0)
        pl = pool.place(bpl)
        tables = [torch.from_numpy(np.ascontiguousarray(wl.layer_table(0, l))).to(dev) for l in range(L)]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for l in range(L)]
        torch.cuda.synchronize()
        io, consumer = torch.cuda.Stream(), torch.cuda.Stream()
        pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, io)
        pool.wait_offloads(pl, io)
        io.synchronize()
        pool.synchronize()
        for attempt in range(2):                           # the second pass is the measured one (first-use costs gone)
            ready = [torch.cuda.Event() for _ in range(L)]
            first, last = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            pool.retrieve_layers_signal(pl, 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, ready, io)
            consumer.wait_event(ready[0])
            first.record(consumer)
            consumer.wait_event(ready[L - 1])
            last.record(consumer)
            consumer.synchronize()
            io.synchronize()
        lead_ms = first.elapsed_time(last)
        per_layer_ms = int(bpl[0]) * g.payload / 58e9 * 1e3            # a layer cannot move faster than the link
        assert lead_ms > 4 * per_layer_ms, f"ready[0] fired only {lead_ms:.3f} ms before ready[{L - 1}]: layers were fused into one unit"
        for l in range(L):
            assert torch.equal(dst[l][:, tables[l].long()], src[l][:, tables[l].long()])
        pl.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_one_signalled_launch_hands_small_layers_over_one_by_one(kernel):
    """Zero-copy path, a request of 32 layers x 2 MiB (less than two groups' worth): kvpool_retrieve_layers_signal moves it
    with ONE kernel launch whose kernel raises a flag per layer; the per-layer events, recorded behind stream wait-values on
    those flags, fire in layer order and spread over the launch (ready[0] long before ready[31]); a consumer that waits on
    nothing but the events reads the oracle's bytes."""
    dev = torch.device("cuda:0")
    wl = W.make_workload(4, scale=1 / 128, n_layers=32)    # 64 blocks x 32 KiB = 2 MiB per layer, 6 buffers 4:4:2:2:1:1
    g, L = wl.geom, wl.geom.n_layers
    bw = list(wl.default_weights())
    pool = make_pool(wl)
    try:
        pool.set_path(kv.PATH_ZEROCOPY)
        pool.set_tuning(kernel=KERNELS[kernel], link_kernel=KERNELS[kernel])
        bpl = wl.blocks_per_layer(0)
        pl, opl = pool.place(bpl), oracle.place(bw, bpl)
        tables_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(L)]
        tables = [torch.from_numpy(t).to(dev) for t in tables_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        torch.cuda.synchronize()
        io, consumer = torch.cuda.Stream(), torch.cuda.Stream()
        pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, io)
        pool.wait_offloads(pl, io)
        io.synchronize()
        pool.synchronize()
        for attempt in range(3):                           # the flag sets are reused round-robin; the last pass is the measured one
            dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for l in range(L)]
            sums = torch.zeros(L, dtype=torch.int64, device=dev)
            torch.cuda.synchronize()
            ready = [torch.cuda.Event() for _ in range(L)]
            stamps = [torch.cuda.Event(enable_timing=True) for _ in range(L)]
            k0, m0 = pool.stats()
            pool.retrieve_layers_signal(pl, 0, [d[0] for d in dst], [d[1] for d in dst], g.kvb, tables, ready, io)
            k1, m1 = pool.stats()
            assert (k1 - k0, m1 - m0) == (1, 0)             # one launch, no copy
            for l in range(L):                             # the consumer never synchronises with `io` except through the events
                consumer.wait_event(ready[l])
                stamps[l].record(consumer)
                pool.checksum(dst[l][0], dst[l][1], g.kvb, tables[l], int(bpl[l]), sums[l:l + 1], consumer)
            consumer.synchronize()
            got = [int(x) % 2 ** 64 for x in sums.cpu().tolist()]
            assert got == [oracle.checksum(W.kv_layer_numpy(wl, l), tables_np[l]) for l in range(L)]
            io.synchronize()
        at = [stamps[0].elapsed_time(stamps[l]) for l in range(L)]
        assert all(b >= a - 0.01 for a, b in zip(at, at[1:])), at          # in layer order
        assert at[L - 1] > 0.6 and at[L // 2] > 0.25 * at[L - 1], at        # 62 MiB behind layer 0 take > 1 ms on the link: spread over the launch
        for l in range(L):
            stripes = oracle.offload_layer(W.kv_layer_numpy(wl, l), tables_np[l], opl[l])
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_layer(ref, tables_np[l], opl[l], stripes)
            assert np.array_equal(dst[l].cpu().numpy().view(np.uint16), ref), f"retrieved layer {l} differs"
        pl.release()
    finally:
        pool.destroy()


def test_release_waits_for_work_still_queued_on_the_callers_stream():
    """kvpool_release must not hand stripes back to the allocator while a kernel on a caller's stream still uses them: a
    zero-copy retrieve queued behind 80 ms of other work is still pending when release is called; release returns only
    after it has run, and the retrieved bytes are right although the next placement reuses (and overwrites) the region."""
    import time
    dev = torch.device("cuda:0")
    wl = W.make_workload(1, n_layers=2)
    g = wl.geom
    pool = make_pool(wl)
    try:
        pool.set_path(kv.PATH_ZEROCOPY)
        bpl = wl.blocks_per_layer(0)
        tables = [torch.from_numpy(np.ascontiguousarray(wl.layer_table(0, l))).to(dev) for l in range(2)]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(2)]
        other = [W.kv_layer_torch(wl, l + 7, dev) for l in range(2)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for l in range(2)]
        s = torch.cuda.Stream()
        torch.cuda.synchronize()
        pl = pool.place(bpl)
        for l in range(2):
            pool.offload(pl, l, src[l][0], src[l][1], g.kvb, tables[l], s)
        s.synchronize()
        pool.spin(80_000_000, s)
        for l in range(2):
            pool.retrieve(pl, l, dst[l][0], dst[l][1], g.kvb, tables[l], s)
        t0 = time.perf_counter()
        pl.release()
        waited = time.perf_counter() - t0
        assert s.query(), "release returned while the retrieve was still queued on the caller's stream"
        assert waited > 0.04
        pl2 = pool.place(bpl)                               # same region (first fit): overwritten with other bytes right away
        for l in range(2):
            pool.offload(pl2, l, other[l][0], other[l][1], g.kvb, tables[l], s)
        s.synchronize()
        for l in range(2):
            assert torch.equal(dst[l][:, tables[l].long()], src[l][:, tables[l].long()])
        pl2.release()
    finally:
        pool.destroy()


def test_numa_bound_registered_and_write_combined_pool_buffers():
    """Pool-device flavours: mmap + mbind(node 0) + cudaHostRegister, a node that does not exist (falls back unless
    KVPOOL_DEV_NUMA_STRICT, then ENUMA), write-combined buffers, and cudaHostAlloc buffers next to the default ones
    (2 MiB-aligned mapping faulted in in parallel, then cudaHostRegister) — all bit-exact through both paths."""
    g = W.Geometry(n_layers=2, n_kv_heads=2, head_dim=64)
    rng = np.random.default_rng(29)
    wl = _custom(g, 300, [rng.permutation(300)[:256]], 3, (2.0, 1.0, 1.0))
    cap = [8 << 20] * 3
    with pytest.raises(kv.KvPoolError) as e:
        kv.KvPool([2.0, 1.0, 1.0], cap, n_layers=2, n_kv_heads=2, head_dim=64, numa_nodes=[0, 977, 0], dev_flags=[0, kv.DEV_NUMA_STRICT, 0])
    assert e.value.code == kv.ENUMA
    with pytest.raises(kv.KvPoolError) as e:
        kv.KvPool([2.0, 1.0, 1.0], cap, n_layers=2, n_kv_heads=2, head_dim=64, numa_nodes=[0, -3, 0])
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:   # more than the host has: refused before a page is touched, not left to the OOM killer
        kv.KvPool([2.0, 1.0, 1.0], [8 << 20, 1 << 46, 8 << 20], n_layers=2, n_kv_heads=2, head_dim=64)
    assert e.value.code == kv.ENOMEM and "available" in str(e.value)
    auto = [kv.NUMA_AUTO] * 3               # the node the GPU hangs off, read from sysfs; no preference where sysfs does not say
    for numa, flags in (([0, 0, -1], [kv.DEV_NUMA_STRICT, 0, 0]), ([0, 977, -1], [0, 0, 0]), (None, [kv.DEV_WRITE_COMBINED] * 3), (auto, [0, 0, 0]),
                        (None, [kv.DEV_CUDA_HOSTALLOC, 0, kv.DEV_CUDA_HOSTALLOC])):   # cudaHostAlloc next to the default (huge pages + register)
        pool = kv.KvPool([2.0, 1.0, 1.0], cap, n_layers=2, n_kv_heads=2, head_dim=64, numa_nodes=numa, dev_flags=flags)
        try:
            if numa is not None and numa is not auto:
                assert pool.device_info(0)["numa_node"] == 0                         # pages really sit on the bound node
            if numa is auto:
                assert pool.device_info(0)["numa_node"] in (-1, 0)                   # this box has one node
            opl = oracle.place([2.0, 1.0, 1.0], wl.blocks_per_layer(0))
            for path in (kv.PATH_STAGED, kv.PATH_ZEROCOPY):
                pool.set_path(path)
                pl = pool.place(wl.blocks_per_layer(0))
                for l in range(2):
                    table_np = np.ascontiguousarray(wl.layer_table(0, l))
                    table = torch.from_numpy(table_np).cuda()
                    src = W.kv_layer_torch(wl, l, "cuda:0")
                    pool.offload(pl, l, src[0], src[1], g.kvb, table)
                    pool.wait_offloads(pl)
                    torch.cuda.synchronize()
                    want = oracle.offload_layer(W.kv_layer_numpy(wl, l), table_np, opl[l])
                    for i in range(3):
                        assert np.array_equal(np.array(pl.stripe(l, i)), want[i])
                    dst = W.poison_torch((2, wl.nphys, g.kvb // 2), "cuda:0")
                    pool.retrieve(pl, l, dst[0], dst[1], g.kvb, table)
                    torch.cuda.synchronize()
                    ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
                    oracle.retrieve_layer(ref, table_np, opl[l], want)
                    assert np.array_equal(dst.cpu().numpy().view(np.uint16), ref)
                pl.release()
        finally:
            pool.destroy()


def test_naive_per_block_memcpy_baseline_matches_oracle():
    """The comparison baseline (one cudaMemcpyAsync per K/V block) produces the same stripes and the same retrieve."""
    wl = W.make_workload(4, scale=1 / 32, n_layers=2)
    g, dev = wl.geom, torch.device("cuda:0")
    bw = list(wl.default_weights())
    pool = make_pool(wl)
    try:
        pl = pool.place(wl.blocks_per_layer(0))
        opl = oracle.place(bw, wl.blocks_per_layer(0))
        for l in range(g.n_layers):
            table_np = np.ascontiguousarray(wl.layer_table(0, l))
            src = W.kv_layer_torch(wl, l, dev)
            pool.offload_naive(pl, l, src[0], src[1], g.kvb, table_np)
            torch.cuda.synchronize()
            want = oracle.offload_layer(W.kv_layer_numpy(wl, l), table_np, opl[l])
            for i in range(pool.n_devices):
                assert np.array_equal(pl.stripe(l, i), want[i])
            dst = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
            pool.retrieve_naive(pl, l, dst[0], dst[1], g.kvb, table_np)
            torch.cuda.synchronize()
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_layer(ref, table_np, opl[l], want)
            assert np.array_equal(dst.cpu().numpy().view(np.uint16), ref)
        pl.release()
    finally:
        pool.destroy()


def test_plain_c_client_creates_a_pool_on_the_gpu(tmp_path):
    """tests/c_abi_client.c gpu: a C99 program with no Python and no oracle in it offloads a paged layer it filled itself,
    finds every payload through kvpool_lookup on a pinned host device and on an HBM-type device, retrieves into a poisoned
    copy and compares (round trip bit for bit, nothing else written).  Its placement is checked against the oracle here."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    exe, lib_dir = str(tmp_path / "c_abi_client"), os.path.dirname(kv.LIB_PATH)
    cuda_lib = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "lib64")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(root, "include"), os.path.join(root, "tests", "c_abi_client.c"),
                    "-o", exe, "-L", lib_dir, "-lkvpool", "-L", cuda_lib, "-lcudart", f"-Wl,-rpath,{lib_dir}"], check=True)
    run = subprocess.run([exe, "gpu"], capture_output=True, text=True)
    assert run.returncode == 0, run.stderr
    out = run.stdout.splitlines()
    c = oracle.counts([2000, 1000], 64)
    d, s = oracle.wrr(c, 64)
    # pool device 1 of the client is an HBM-type device (KVPOOL_TYPE_HBM = 2), device 0 pinned host memory (MEM = 0)
    assert f"glt block 63: device {int(d[63])} type {2 * int(d[63])} slot {int(s[63])} ptr set" in out
    assert f"glt block 2: device {int(d[2])} type {2 * int(d[2])} slot {int(s[2])} ptr set" in out
    assert f"payloads ok: {int(c[0])} on the host device, {int(c[1])} on the HBM device" in out
    assert out[-1] == "round trip ok: 64 blocks of 8192 bytes, 32 other blocks untouched"
    # the same program with a third, SSD-type device backed by a file: payloads found by LBA and read with plain pread
    run = subprocess.run([exe, "gpu", str(tmp_path / "ssd.img")], capture_output=True, text=True, timeout=120)
    assert run.returncode == 0, run.stderr
    out = run.stdout.splitlines()
    c = oracle.counts([2000, 1000, 1000], 64)
    assert f"payloads ok: {int(c[0])} on the host device, {int(c[1])} on the HBM device" in out
    assert f"payloads ok: {int(c[2])} on the SSD device (512-byte sectors)" in out
    assert out[-1] == "round trip ok: 64 blocks of 8192 bytes, 32 other blocks untouched" and not (tmp_path / "ssd.img").exists()


def test_keyed_glt_finds_blocks_across_placements_and_forgets_them_on_release():
    """Table I with its `key` column: identifiers bound to the blocks of two requests are found by identifier alone
    and give the same (device_id, type, location) as the dense lookup; a found run retrieves through
    kvpool_retrieve_range; release forgets the identifiers.  (Semantics only: parity unpinned, R15.)"""
    g = W.Geometry(n_layers=2, n_kv_heads=2, head_dim=64)
    rng = np.random.default_rng(31)
    wl = _custom(g, 200, [rng.permutation(200)[:96]], 3, (3.0, 2.0, 1.0))
    pool = make_pool(wl, slack=4.0)
    try:
        a, b = pool.place([96, 96]), pool.place([40, 0])
        ids_a = [rng.integers(0, 2 ** 63, size=96, dtype=np.uint64) for _ in range(2)]
        ids_b = rng.integers(0, 2 ** 63, size=40, dtype=np.uint64)
        for l in range(2):
            pool.glt_bind(a, l, ids_a[l])
        pool.glt_bind(b, 0, ids_b)
        pool.glt_bind(b, 1, [])                                                       # K_l = 0
        for pl, l, ids in ((a, 0, ids_a[0]), (a, 1, ids_a[1]), (b, 0, ids_b)):
            for j in (0, len(ids) - 1, 17):
                f = pool.glt_find(int(ids[j]))
                d, t, s, ptr = pl.lookup(l, j)
                assert (f["placement"], f["layer"], f["block"], f["device_id"], f["type"], f["location"]) == (pl.handle, l, j, d, t, ptr)
        assert len({pool.glt_find(int(i))["key"] for i in ids_b}) == 40                # distinct hash keys
        for bad in ([int(ids_b[3])] + [1, 2, 3] * 13, [5] * 40):                     # already bound / repeating: nothing bound
            with pytest.raises(kv.KvPoolError) as e:
                pool.glt_bind(b, 0, bad[:40])
            assert e.value.code == kv.EINVAL
        with pytest.raises(kv.KvPoolError) as e:
            pool.glt_find(1)
        assert e.value.code == kv.ENOENT
        # prefix reuse: find a run of request a's layer-0 blocks by identifier, then fetch exactly that run
        table_np = np.ascontiguousarray(wl.layer_table(0, 0))
        table = torch.from_numpy(table_np).cuda()
        src = W.kv_layer_torch(wl, 0, "cuda:0")
        pool.offload(a, 0, src[0], src[1], g.kvb, table)
        first = pool.glt_find(int(ids_a[0][8]))
        assert (first["layer"], first["block"]) == (0, 8)
        dst = W.poison_torch((2, wl.nphys, g.kvb // 2), "cuda:0")
        pool.retrieve_range(a, 0, first["block"], 24, dst[0], dst[1], g.kvb, table)
        torch.cuda.synchronize()
        opl = oracle.place([3.0, 2.0, 1.0], [96])[0]
        ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
        oracle.retrieve_range(ref, table_np, opl, oracle.offload_layer(W.kv_layer_numpy(wl, 0), table_np, opl), 8, 24)
        assert np.array_equal(dst.cpu().numpy().view(np.uint16), ref)
        b.release()
        with pytest.raises(kv.KvPoolError) as e:
            pool.glt_find(int(ids_b[0]))
        assert e.value.code == kv.ENOENT
        assert pool.glt_find(int(ids_a[1][95]))["block"] == 95
        a.release()
    finally:
        pool.destroy()


HBM = kv.DEV_HBM


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("path", ["staged", "zerocopy", "auto"])
def test_hbm_type_pool_devices_alone_and_mixed_with_host_devices(path, kernel):
    """KVPOOL_DEV_HBM: pool devices that are GPU memory — here the pool's own GPU, standing in for an
    NVLink peer — next to pinned host devices.  Same placement, same stripe bytes, same retrieved tensors as the oracle;
    GLT type = KVPOOL_TYPE_HBM and location = a device pointer for their blocks (checked in run_parity / check_glt)."""
    p, k = PATHS[path], KERNELS[kernel]
    # config 1 whole (2 devices 2:1), the slower one in HBM: staged path = 1 pack launch + ONE copy (device 0) per layer
    out = run_parity(W.make_workload(1), path=p, kernel=k, dev_flags=[0, HBM])
    assert out["kernels"] == 64 and out["memcpys"] == (64 if path == "staged" else 0)
    # config 4 cut (6 devices 4:4:2:2:1:1, 16 MiB layers), devices 0 and 3 in HBM
    out = run_parity(W.make_workload(4, scale=1 / 16, n_layers=3), path=p, kernel=k, dev_flags=[HBM, 0, 0, HBM, 0, 0])
    assert out["memcpys"] == (0 if path == "zerocopy" else 2 * 3 * 4)
    # every device in HBM: no copy engine at all, whatever the path
    out = run_parity(W.make_workload(4, scale=1 / 16, n_layers=2), path=p, kernel=k, dev_flags=[HBM] * 6)
    assert out["memcpys"] == 0
    # ragged block size, K < N, sliding-window layers (config 3 scaled: 8-block and 1024-block layers alternate)
    rng = np.random.default_rng(31)
    g = W.Geometry(n_layers=2, n_kv_heads=1, head_dim=80)
    run_parity(_custom(g, 301, [rng.permutation(301)[:257]], 3, (3.0, 2.0, 1.0)), path=p, kernel=k, dev_flags=[HBM, 0, HBM])
    g = W.Geometry(n_layers=1, n_kv_heads=1, head_dim=8, block_tokens=1)
    run_parity(_custom(g, 9, [[7, 2, 5]], 6, (4.0, 4.0, 2.0, 2.0, 1.0, 1.0)), path=p, kernel=k, dev_flags=[0, HBM, 0, HBM, 0, HBM])
    run_parity(W.make_workload(3, scale=1 / 8, n_layers=4), path=p, kernel=k, dev_flags=[0, HBM, HBM, 0])
    # a slow host device next to a fast HBM one, few blocks: counts (0, 8) — nothing to stage, so no copy and no staging
    # slot is taken whatever the path (a slot recycled without waits could be overwritten under an earlier offload's copy)
    g = W.Geometry(n_layers=2, n_kv_heads=1, head_dim=64)
    out = run_parity(_custom(g, 16, [rng.permutation(16)[:8]], 2, (1.0, 50.0)), path=p, kernel=k, dev_flags=[0, HBM])
    assert out["memcpys"] == 0


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_hbm_type_pool_devices_batched_groups_and_ranges(kernel):
    k = KERNELS[kernel]
    # batched calls: a group's host stripes travel by one copy per HOST device, its HBM stripes inside the kernel
    _run_batched(W.make_workload(1), kv.PATH_AUTO, k, expect_kernels=4, expect_memcpys=4, dev_flags=[0, HBM])
    _run_batched(W.make_workload(1), kv.PATH_STAGED, k, expect_kernels=4, expect_memcpys=0, dev_flags=[HBM, HBM])
    _run_batched(W.make_workload(1), kv.PATH_ZEROCOPY, k, expect_kernels=4, expect_memcpys=0, dev_flags=[HBM, 0])   # two 64 MiB groups per leg
    wl = W.make_workload(3, scale=1 / 8, n_layers=6)                      # groups {0,1,2} {3,4} {5}; 4 devices, 2 of them host
    _run_batched(wl, kv.PATH_STAGED, k, expect_kernels=6, expect_memcpys=12, dev_flags=[HBM, 0, 0, HBM])
    # partial retrieval over a mixed pool
    wl = W.make_workload(4, scale=1 / 16, n_layers=1)
    g, dev = wl.geom, torch.device("cuda:0")
    bw = list(wl.default_weights())
    for path in (kv.PATH_STAGED, kv.PATH_ZEROCOPY):
        pool = make_pool(wl, dev_flags=[0, HBM, 0, HBM, HBM, 0])
        try:
            pool.set_path(path)
            pool.set_tuning(kernel=k, link_kernel=k)
            pl = pool.place(wl.blocks_per_layer(0))
            opl = oracle.place(bw, wl.blocks_per_layer(0))
            table_np = np.ascontiguousarray(wl.layer_table(0, 0))
            K, table = len(table_np), torch.from_numpy(table_np).to(dev)
            src, src_cpu = W.kv_layer_torch(wl, 0, dev), W.kv_layer_numpy(wl, 0)
            pool.offload(pl, 0, src[0], src[1], g.kvb, table)
            pool.wait_offloads(pl)
            torch.cuda.synchronize()
            stripes = oracle.offload_layer(src_cpu, table_np, opl[0])
            for first, n in ((0, K // 4), (K // 3, K // 2), (K - 1, 1), (0, K), (5, 0), (17, 3)):
                dst = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
                pool.retrieve_range(pl, 0, first, n, dst[0], dst[1], g.kvb, table)
                torch.cuda.synchronize()
                want = W.poison_numpy((2, wl.nphys, g.kvb // 2))
                oracle.retrieve_range(want, table_np, opl[0], stripes, first, n)
                assert np.array_equal(dst.cpu().numpy().view(np.uint16), want), (path, first, n)
            pl.release()
        finally:
            pool.destroy()


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs a second GPU: the peer (NVLink / NVSwitch) branch of HBM-type pool devices")
@pytest.mark.parametrize("path", ["staged", "zerocopy", "auto"])
def test_hbm_type_pool_device_on_a_peer_gpu(path):
    """SURVEY.md 8(f) row 2 on real hardware, the day a box with two GPUs runs this suite: pool devices in the HBM of GPU 1
    (cudaDeviceEnablePeerAccess from GPU 0; the kernels reach the stripes by peer loads / stores), alone and mixed with a host
    buffer — same oracle parity as every other pool, and the GLT says where each stripe lives."""
    wl = W.make_workload(4, scale=1 / 16, n_layers=3)
    g = wl.geom
    caps = [wl.moved_bytes() + (64 << 20)] * 3
    with kv.KvPool([1.0, 8.0, 8.0], caps, n_layers=g.n_layers, n_kv_heads=g.n_kv_heads, head_dim=g.head_dim, dev_flags=[0, HBM, HBM],
                   gpus=[-1, 1, 1], link_groups=[0, 1, 1]) as pool:
        assert pool.device_type(1) == (kv.TYPE_HBM, 1) and pool.device_type(2) == (kv.TYPE_HBM, 1)
        peer = pool.measure_bandwidth(1, kv.MEASURE_KERNEL_RETRIEVE, 64 << 20, 3)
        host = pool.measure_bandwidth(0, kv.MEASURE_RETRIEVE, 64 << 20, 3)
        assert peer > 2 * host                                                     # NVLink, not the host link
    for flags, gpus in (([HBM, HBM], [1, 1]), ([0, HBM], [-1, 1]), ([HBM, 0, HBM], [1, -1, 0])):
        n = len(flags)
        wl_n = _custom(g, wl.nphys, [wl.layer_table(0, 0)], n, tuple(float(1 + (i % 2) * 3) for i in range(n)))
        out = run_parity(wl_n, path=PATHS[path], kernel=kv.KERNEL_VEC16, dev_flags=flags, gpus=gpus)
        assert out["bytes_compared"] == wl_n.moved_bytes()


def test_hbm_type_pool_device_introspection_bandwidth_and_errors():
    g = dict(n_layers=1, n_kv_heads=2, head_dim=64)
    with pytest.raises(kv.KvPoolError) as e:                                       # HBM excludes the host-memory flags
        kv.KvPool([1.0], [1 << 20], dev_flags=[HBM | kv.DEV_WRITE_COMBINED], **g)
    assert e.value.code == kv.EINVAL
    with pytest.raises(kv.KvPoolError) as e:                                       # a GPU that does not exist
        kv.KvPool([1.0], [1 << 20], dev_flags=[HBM], gpus=[torch.cuda.device_count() + 3], **g)
    assert e.value.code == kv.EINVAL
    pool = kv.KvPool([50.0, 1500.0], [64 << 20, 64 << 20], dev_flags=[0, HBM], gpus=[-1, 0], **g)
    try:
        assert pool.device_type(0) == (kv.TYPE_MEM, -1) and pool.device_type(1) == (kv.TYPE_HBM, 0)
        assert pool.device_info(0)["host_base"] and not pool.device_info(1)["host_base"]
        host = pool.measure_bandwidth(0, 0, 32 << 20, 3)
        hbm_r, hbm_w = pool.measure_bandwidth(1, 0, 64 << 20, 3), pool.measure_bandwidth(1, 1, 64 << 20, 3)
        assert hbm_r > 5 * host and hbm_w > 5 * host                               # a device-to-device copy, not the host link
        # the same devices measured with the library's own gather / scatter kernel (what reaches the stripes of such a pool)
        k_host = [pool.measure_bandwidth(0, d, 32 << 20, 3) for d in (kv.MEASURE_KERNEL_RETRIEVE, kv.MEASURE_KERNEL_OFFLOAD)]
        k_hbm = [pool.measure_bandwidth(1, d, 64 << 20, 3) for d in (kv.MEASURE_KERNEL_RETRIEVE, kv.MEASURE_KERNEL_OFFLOAD)]
        assert all(0.5 * host < x < 1.2 * host for x in k_host) and all(x > 5 * host for x in k_hbm)
        with pytest.raises(kv.KvPoolError) as e:
            pool.measure_bandwidth(0, 4, 32 << 20, 3)
        assert e.value.code == kv.EINVAL
        # kvpool_calibrate: measure, divide what link groups share (none here), install; Eq. 1's weights follow
        b = pool.calibrate(kv.MEASURE_KERNEL_RETRIEVE, 32 << 20, 3)
        assert np.array_equal(pool.bandwidths()[0], b) and list(pool.bandwidths()[1]) == [0, 0]
        assert np.array_equal(pool.weights(), oracle.weights(list(b)))
        pool.set_bandwidth([50.0, 1500.0])
        pl = pool.place([31])
        c = pl.counts(0)
        assert list(c) == [1, 30]                                                   # 50 : 1500 of 31 blocks
        assert pl.stripe_location(0, 1)[1] == 30 * pool.payload
        pl.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_zero_copy_retrieve_is_capturable_into_a_cuda_graph(kernel):
    """Once the offloads have landed (caller's stream synchronised + kvpool_synchronize), a zero-copy retrieve enqueues one
    kernel and nothing else, so a serving engine can capture it into its decode graph: capture per-layer, range and
    batched retrieves, replay twice into re-poisoned destinations, compare with the oracle."""
    wl = W.make_workload(3, scale=1 / 16, n_layers=6)          # sliding-window (8-block) and full (512-block) layers alternate
    g, L, dev = wl.geom, wl.geom.n_layers, torch.device("cuda:0")
    bw, bpl = list(wl.default_weights()), wl.blocks_per_layer(0)
    pool = make_pool(wl)
    try:
        pool.set_path(kv.PATH_ZEROCOPY)
        pool.set_tuning(kernel=KERNELS[kernel], link_kernel=KERNELS[kernel])
        pl, opl = pool.place(bpl), oracle.place(bw, bpl)
        tables_np = [np.ascontiguousarray(wl.layer_table(0, l)) for l in range(L)]
        tables = [torch.from_numpy(t).to(dev) for t in tables_np]
        src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
        dst = [W.poison_torch((2, wl.nphys, g.kvb // 2), dev) for l in range(L)]
        torch.cuda.synchronize()
        s = torch.cuda.Stream()
        pool.offload_layers(pl, 0, [x[0] for x in src], [x[1] for x in src], g.kvb, tables, s)
        pool.wait_offloads(pl, s)
        s.synchronize()
        pool.synchronize()
        k0, m0 = pool.stats()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s, capture_error_mode="relaxed"):
            pool.retrieve_layers(pl, 0, [d[0] for d in dst[:3]], [d[1] for d in dst[:3]], g.kvb, tables[:3], s)    # one fused launch
            pool.retrieve(pl, 3, dst[3][0], dst[3][1], g.kvb, tables[3], s)
            pool.retrieve_range(pl, 4, 0, 5, dst[4][0], dst[4][1], g.kvb, tables[4], s)
            pool.retrieve_range(pl, 5, 100, 300, dst[5][0], dst[5][1], g.kvb, tables[5], s)
        assert pool.stats() == (k0 + 4, m0)
        want = []
        for l in range(L):
            stripes = oracle.offload_layer(W.kv_layer_numpy(wl, l), tables_np[l], opl[l])
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            first, n = {4: (0, 5), 5: (100, 300)}.get(l, (0, len(tables_np[l])))
            oracle.retrieve_range(ref, tables_np[l], opl[l], stripes, first, n)
            want.append(ref)
        for _ in range(2):
            for d in dst:
                d.copy_(W.poison_torch(d.shape, dev))
            torch.cuda.synchronize()
            graph.replay()
            torch.cuda.synchronize()
            for l in range(L):
                assert np.array_equal(dst[l].cpu().numpy().view(np.uint16), want[l]), f"graph replay: layer {l} differs"
        del graph
        pl.release()
    finally:
        pool.destroy()


def test_host_threads_share_one_pool():
    """Four host threads, one request each (config 5 scaled: interleaved block tables over one shared paged pool), drive one
    pool handle concurrently — place, offload every layer, retrieve every layer, release, three times over, each on its
    own stream.  ctypes drops the GIL inside the library, so the calls really interleave; staging slots, events, the table
    arena and the allocators are shared.  Every request's stripes and retrieved blocks must equal the oracle's."""
    import threading
    wl = W.make_workload(5, scale=1 / 16, n_layers=4)
    g, dev = wl.geom, torch.device("cuda:0")
    R, L, elems = len(wl.requests), wl.geom.n_layers, wl.geom.kvb // 2
    bw = list(wl.default_weights())
    pool = make_pool(wl, bw)
    src = [W.kv_layer_torch(wl, l, dev) for l in range(L)]
    src_cpu = [W.kv_layer_numpy(wl, l) for l in range(L)]
    dst = [W.poison_torch((2, wl.nphys, elems), dev) for l in range(L)]      # requests own disjoint physical blocks
    torch.cuda.synchronize()
    errors, stripes_ok = [], [0] * R
    barrier = threading.Barrier(R)

    def worker(r: int) -> None:
        try:
            torch.cuda.set_device(dev)
            s = torch.cuda.Stream(device=dev)
            bpl = wl.blocks_per_layer(r)
            opl = oracle.place(bw, bpl)
            tables_np = [np.ascontiguousarray(wl.layer_table(r, l)) for l in range(L)]
            with torch.cuda.stream(s):
                tables = [torch.from_numpy(t).to(dev) for t in tables_np]
            s.synchronize()
            barrier.wait()
            for rep in range(3):
                pool.set_path((kv.PATH_STAGED, kv.PATH_AUTO, kv.PATH_STAGED)[rep] if r % 2 == 0 else kv.PATH_STAGED)
                pl = pool.place(bpl)
                check_placement(pl, opl)
                for l in range(L):
                    pool.offload(pl, l, src[l][0], src[l][1], g.kvb, tables[l], s)
                pool.wait_offloads(pl, s)
                s.synchronize()
                for l in range(L):
                    want = oracle.offload_layer(src_cpu[l], tables_np[l], opl[l])
                    for i in range(pool.n_devices):
                        assert np.array_equal(pl.stripe(l, i), want[i]), (r, rep, l, i)
                        stripes_ok[r] += 1
                for l in range(L):
                    pool.retrieve(pl, l, dst[l][0], dst[l][1], g.kvb, tables[l], s)
                s.synchronize()
                pl.release()
        except BaseException as e:        # noqa: BLE001 - reported by the main thread
            errors.append((r, repr(e)))
            barrier.abort()

    threads = [threading.Thread(target=worker, args=(r,)) for r in range(R)]
    try:
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        assert not errors, errors
        assert all(n == 3 * L * pool.n_devices for n in stripes_ok)
        torch.cuda.synchronize()
        for l in range(L):                # every request's blocks came back; everything else is still poison
            want = W.poison_numpy((2, wl.nphys, elems))
            for r in range(R):
                t = wl.layer_table(r, l)
                want[:, t] = src_cpu[l][:, t]
            assert np.array_equal(dst[l].cpu().numpy().view(np.uint16), want), l
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_chunked_staging_caps_the_ring_and_keeps_parity(kernel):
    """tune.stage_chunk_bytes: a layer larger than a staging slot travels in DEVICE-MAJOR chunks — runs of consecutive slots
    of one pool device's stripe, one copy and one launch each (the launch finds its logical blocks through the device's
    inverse map) — same stripes, same retrieved tensors, a ring that no longer grows with the layer."""
    k = KERNELS[kernel]
    wl = W.make_workload(4, scale=1 / 8, n_layers=3)                      # 1024 blocks x 32 KiB = 32 MiB per layer, 6 devices
    base = run_parity(wl, path=kv.PATH_STAGED, kernel=k)
    # 5 MiB chunks = 160 slots: stripes of 293, 293, 146, 146, 73, 73 blocks travel as 2 + 2 + 1 + 1 + 1 + 1 chunks
    counts = oracle.place(list(wl.default_weights()), wl.blocks_per_layer(0))[0].counts
    chunks = sum(-(-int(c) // 160) for c in counts)
    assert chunks == 8
    out = run_parity(wl, path=kv.PATH_STAGED, kernel=k, tuning={"stage_chunk_bytes": 5 << 20})
    assert out["bytes_compared"] == base["bytes_compared"]
    assert out["kernels"] == chunks * base["kernels"] and out["memcpys"] * 6 == chunks * base["memcpys"]
    # the same with the devices in link groups (shared I/O streams: {0,1,2} on one, {3,4} on another, 5 alone) and 3 slots
    out = run_parity(wl, path=kv.PATH_STAGED, kernel=k, tuning={"stage_chunk_bytes": 5 << 20, "stage_slots": 3}, link_groups=[7, 7, 7, 2, 2, 0])
    assert out["kernels"] == chunks * base["kernels"] and out["memcpys"] * 6 == chunks * base["memcpys"]
    # a chunk smaller than one block still moves one block at a time; 2 slots; mixed host / HBM pool; ragged block size
    g = W.Geometry(n_layers=2, n_kv_heads=1, head_dim=80)
    rng = np.random.default_rng(53)
    run_parity(_custom(g, 301, [rng.permutation(301)[:257]], 3, (3.0, 2.0, 1.0)), path=kv.PATH_STAGED, kernel=k,
               tuning={"stage_chunk_bytes": 1000, "stage_slots": 2}, dev_flags=[0, HBM, 0])
    # auto path, sliding-window layers (tiny layers go zero-copy, big ones chunked), several requests on several streams
    run_parity(W.make_workload(3, scale=1 / 8, n_layers=4), path=kv.PATH_AUTO, kernel=k, tuning={"stage_chunk_bytes": 3 << 20})
    run_parity(W.make_workload(5, scale=1 / 16, n_layers=2), path=kv.PATH_STAGED, kernel=k, streams=4, tuning={"stage_chunk_bytes": 2 << 20})
    # batched calls and partial retrieval under a chunk cap
    _run_batched(W.make_workload(3, scale=1 / 8, n_layers=6), kv.PATH_STAGED, k, expect_kernels=None, expect_memcpys=None,
                 tuning={"stage_chunk_bytes": 3 << 20})
    # the ring really is capped: 4 slots of ~5 MiB instead of 4 x 32 MiB
    pool = make_pool(wl)
    try:
        pool.set_path(kv.PATH_STAGED)
        free0 = torch.cuda.mem_get_info()[0]
        pool.set_tuning(stage_chunk_bytes=5 << 20, stage_slots=4)
        pl = pool.place(wl.blocks_per_layer(0))
        assert free0 - torch.cuda.mem_get_info()[0] < 4 * (8 << 20)
        pl.release()
    finally:
        pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("path", ["staged", "zerocopy", "auto"])
def test_offload_range_fills_a_layer_in_instalments(path, kernel):
    """kvpool_offload_range: a layer placed once and offloaded in instalments, in any order, ends with the
    oracle's stripes; after each instalment exactly its slots have changed (the rest of the stripes still hold the fill
    written before), a retrieve of blocks not yet offloaded is ESTATE, and what has arrived can be retrieved at once."""
    p, k = PATHS[path], KERNELS[kernel]
    wl = W.make_workload(4, scale=1 / 16, n_layers=1)                    # 512 blocks x 32 KiB, 6 devices 4:4:2:2:1:1
    g, dev = wl.geom, torch.device("cuda:0")
    bw = list(wl.default_weights())
    for flags, tuning in (([0] * 6, {}), ([0, HBM, 0, 0, HBM, 0], {"stage_chunk_bytes": 3 << 20, "stage_slots": 2})):
        pool = make_pool(wl, dev_flags=flags)
        try:
            pool.set_path(p)
            pool.set_tuning(kernel=k, link_kernel=k, **tuning)
            bpl = wl.blocks_per_layer(0)
            K = int(bpl[0])
            pl = pool.place(bpl)
            opl = oracle.place(bw, bpl)
            table_np = np.ascontiguousarray(wl.layer_table(0, 0))
            table = torch.from_numpy(table_np).to(dev)
            src, src_cpu = W.kv_layer_torch(wl, 0, dev), W.kv_layer_numpy(wl, 0)
            fill = torch.full_like(src, 0x1111)                           # a first whole-layer offload of a constant: the stripes' fill
            fill_cpu = np.full_like(src_cpu, 0x1111)
            torch.cuda.synchronize()
            s = torch.cuda.Stream()
            with pytest.raises(kv.KvPoolError) as e:
                pool.offload_range(pl, 0, K - 3, 4, src[0], src[1], g.kvb, table, s)
            assert e.value.code == kv.EINVAL
            pool.offload_range(pl, 0, 0, 40, fill[0], fill[1], g.kvb, table, s)
            dst = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
            with pytest.raises(kv.KvPoolError) as e:                      # blocks 40.. are not in the pool yet
                pool.retrieve(pl, 0, dst[0], dst[1], g.kvb, table, s)
            assert e.value.code == kv.ESTATE
            with pytest.raises(kv.KvPoolError) as e:
                pool.retrieve_range(pl, 0, 30, 20, dst[0], dst[1], g.kvb, table, s)
            assert e.value.code == kv.ESTATE
            pool.retrieve_range(pl, 0, 5, 30, dst[0], dst[1], g.kvb, table, s)       # these are
            pool.offload(pl, 0, fill[0], fill[1], g.kvb, table, s)                   # now the whole layer holds the fill
            want = oracle.offload_layer(fill_cpu, table_np, opl[0])
            cuts = [0, 1, 130, 130, 131, 400, K]
            order = [4, 0, 5, 2, 1, 3]
            for q in order:
                lo, hi = cuts[q], cuts[q + 1]
                pool.offload_range(pl, 0, lo, hi - lo, src[0], src[1], g.kvb, table, s)
                oracle.offload_range(src_cpu, table_np, opl[0], want, lo, hi - lo)
                if q in (0, 2):                                           # check the intermediate state twice, else keep enqueueing
                    pool.wait_offloads(pl, s)
                    s.synchronize()
                    for i in range(pool.n_devices):
                        assert np.array_equal(pl.stripe(0, i), want[i]), (path, q, i)
            pool.wait_offloads(pl, s)
            dst2 = W.poison_torch((2, wl.nphys, g.kvb // 2), dev)
            pool.retrieve(pl, 0, dst2[0], dst2[1], g.kvb, table, s)
            s.synchronize()
            full = oracle.offload_layer(src_cpu, table_np, opl[0])
            for i in range(pool.n_devices):
                assert np.array_equal(pl.stripe(0, i), full[i]) and np.array_equal(want[i], full[i])
            ref = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_layer(ref, table_np, opl[0], full)
            assert np.array_equal(dst2.cpu().numpy().view(np.uint16), ref)
            ref1 = W.poison_numpy((2, wl.nphys, g.kvb // 2))
            oracle.retrieve_range(ref1, table_np, opl[0], oracle.offload_layer(fill_cpu, table_np, opl[0]), 5, 30)
            assert np.array_equal(dst.cpu().numpy().view(np.uint16), ref1)
            pl.release()
        finally:
            pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
def test_red_zones_around_planes_stripes_and_staging_stay_intact(kernel):
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are hunted with red zones: the K and V planes
    and a caller staging buffer sit inside larger poison-filled allocations, the table names the first and the last
    physical block, block sizes are ragged (not a multiple of the kernels' 4 KiB / 16 KiB pieces) — after pack, unpack,
    offload and retrieve on every path the guards on both sides of each buffer still hold the poison, and so does every
    pool-buffer byte outside the placement's stripes."""
    k = KERNELS[kernel]
    rng = np.random.default_rng(61)
    dev = torch.device("cuda:0")
    GUARD = 0x5AA5
    for g, nphys, n_dev, w in ((W.Geometry(n_layers=1, n_kv_heads=1, head_dim=80), 67, 3, (3.0, 2.0, 1.0)),
                               (W.Geometry(n_layers=1, n_kv_heads=3, head_dim=136), 41, 2, (2.0, 1.0)),
                               (W.Geometry(n_layers=1, n_kv_heads=4, head_dim=128), 33, 4, (4.0, 2.0, 1.0, 1.0))):
        table_np = np.ascontiguousarray(rng.permutation(nphys).astype(np.int32))          # every block, the first and the last included
        wl = _custom(g, nphys, [table_np], n_dev, w)
        elems, pad = g.kvb // 2, 3
        src_cpu = W.kv_layer_numpy(wl, 0)
        table = torch.from_numpy(table_np).to(dev)
        opl = oracle.place(list(w), [nphys])
        want = oracle.offload_layer(src_cpu, table_np, opl[0])

        def guarded(fill_from=None):
            """Two planes of (pad + nphys + pad) blocks each; returns (buffers, views of the nphys blocks in the middle)."""
            bufs = [torch.full((nphys + 2 * pad, elems), GUARD, dtype=torch.int16, device=dev) for _ in range(2)]
            mids = [b[pad:pad + nphys] for b in bufs]
            for h in range(2):
                mids[h].copy_(torch.from_numpy(fill_from[h].view(np.int16)).to(dev) if fill_from is not None
                              else torch.full((nphys, elems), np.int16(np.uint16(W.POISON_BITS).view(np.int16)).item(), dtype=torch.int16, device=dev))
            return bufs, mids

        def guards_intact(bufs):
            return all(bool((b[:pad] == GUARD).all()) and bool((b[pad + nphys:] == GUARD).all()) for b in bufs)

        sbufs, smid = guarded(src_cpu)
        for path in (kv.PATH_STAGED, kv.PATH_ZEROCOPY):
            pool = make_pool(wl)
            try:
                pool.set_path(path)
                pool.set_tuning(kernel=k, link_kernel=k)
                caps = [pool.device_info(i)["capacity"] for i in range(n_dev)]
                hosts = [np.ctypeslib.as_array(ctypes.cast(pool.device_info(i)["host_base"], ctypes.POINTER(ctypes.c_uint8)), shape=(caps[i],))
                         for i in range(n_dev)]
                for h in hosts:
                    h[:] = 0xC3                                                        # every pool byte; the stripes are then the only change
                pl = pool.place([nphys])
                # caller staging with red zones: exactly K*P bytes in the middle
                stage_all = torch.full((nphys * g.payload + 2 * 4096,), 0x77, dtype=torch.uint8, device=dev)
                stage = stage_all[4096:4096 + nphys * g.payload]
                pool.pack(pl, 0, smid[0], smid[1], g.kvb, table, stage)
                dbufs, dmid = guarded()
                pool.unpack(pl, 0, dmid[0], dmid[1], g.kvb, table, stage)
                torch.cuda.synchronize()
                assert bool((stage_all[:4096] == 0x77).all()) and bool((stage_all[4096 + nphys * g.payload:] == 0x77).all())
                assert np.array_equal(stage.cpu().numpy(), np.concatenate(want))
                assert guards_intact(dbufs) and guards_intact(sbufs)
                for h in range(2):
                    assert np.array_equal(dmid[h].cpu().numpy().view(np.uint16), src_cpu[h])
                # through the pool
                pool.offload(pl, 0, smid[0], smid[1], g.kvb, table)
                pool.wait_offloads(pl)
                dbufs, dmid = guarded()
                pool.retrieve(pl, 0, dmid[0], dmid[1], g.kvb, table)
                torch.cuda.synchronize()
                assert guards_intact(dbufs) and guards_intact(sbufs)
                for h in range(2):
                    assert np.array_equal(dmid[h].cpu().numpy().view(np.uint16), src_cpu[h])
                for i in range(n_dev):
                    loc, nb = pl.stripe_location(0, i)
                    off = loc - pool.device_info(i)["host_base"]
                    assert np.array_equal(hosts[i][off:off + nb], want[i])
                    assert bool((hosts[i][:off] == 0xC3).all()) and bool((hosts[i][off + nb:] == 0xC3).all()), (path, i)
                pl.release()
            finally:
                del hosts
                pool.destroy()


@pytest.mark.parametrize("kernel", list(KERNELS))
@pytest.mark.parametrize("path", ["staged", "zerocopy", "staged-chunked"])
def test_device_side_table_check_skips_and_counts_bad_entries(path, kernel):
    """kvpool_set_table_check (R12, opt-in): table entries outside [0, nphys) are skipped — nothing outside the
    planes is read or written (red zones intact), the other blocks move exactly as the oracle says — and counted; with
    a clean table the check changes nothing."""
    # staged-chunked: a slot holds 5 blocks, so the layer travels in device-major chunks (launches that walk the inverse map)
    p, k, chunked = PATHS[path.split("-")[0]], KERNELS[kernel], path.endswith("chunked")
    rng = np.random.default_rng(71)
    dev = torch.device("cuda:0")
    g = W.Geometry(n_layers=1, n_kv_heads=2, head_dim=80)                 # kvb = 5120 B, ragged against the 4 KiB piece
    nphys, K, elems, pad, GUARD = 90, 64, g.kvb // 2, 4, 0x5AA5
    good = np.ascontiguousarray(rng.permutation(nphys)[:K].astype(np.int32))
    bad = good.copy()
    bad_at = [3, 17, 40, 63]
    bad[bad_at] = [nphys, -1, nphys + 2, 2 ** 31 - 1]                     # one past the end, negative, inside the guard, huge
    wl = _custom(g, nphys, [good], 3, (3.0, 2.0, 1.0))
    src_cpu = W.kv_layer_numpy(wl, 0)
    opl = oracle.place([3.0, 2.0, 1.0], [K])
    pool = make_pool(wl)
    try:
        pool.set_path(p)
        pool.set_tuning(kernel=k, link_kernel=k, **({"stage_chunk_bytes": 5 * 2 * g.kvb} if chunked else {}))
        pool.set_table_check(nphys)
        pl = pool.place([K])

        def guarded(fill):
            bufs = [torch.full((nphys + 2 * pad, elems), GUARD, dtype=torch.int16, device=dev) for _ in range(2)]
            for h in range(2):
                bufs[h][pad:pad + nphys].copy_(torch.from_numpy(fill[h].view(np.int16)).to(dev))
            return bufs, [b[pad:pad + nphys] for b in bufs]

        sbufs, smid = guarded(src_cpu)
        # clean table: identical to the unchecked path, zero errors
        pool.offload(pl, 0, smid[0], smid[1], g.kvb, torch.from_numpy(good).to(dev))
        pool.wait_offloads(pl)
        torch.cuda.synchronize()
        want = oracle.offload_layer(src_cpu, good, opl[0])
        assert all(np.array_equal(pl.stripe(0, i), want[i]) for i in range(3)) and pool.table_errors() == 0
        # bad table at retrieve: the four entries are skipped, everything else lands, guards intact
        dbufs, dmid = guarded(W.poison_numpy((2, nphys, elems)))
        pool.retrieve(pl, 0, dmid[0], dmid[1], g.kvb, torch.from_numpy(bad).to(dev))
        torch.cuda.synchronize()
        assert pool.table_errors() == len(bad_at) and pool.table_errors() == 0        # read and reset
        ref = W.poison_numpy((2, nphys, elems))
        ok = np.ones(K, bool); ok[bad_at] = False
        ref[:, good[ok]] = src_cpu[:, good[ok]]
        for h in range(2):
            assert np.array_equal(dmid[h].cpu().numpy().view(np.uint16), ref[h])
            assert bool((dbufs[h][:pad] == GUARD).all()) and bool((dbufs[h][pad + nphys:] == GUARD).all())
        # bad table at offload: every other block lands; on the zero-copy path the skipped entries' slots keep what they held
        fill = np.full_like(src_cpu, 0x2222)
        fbufs, fmid = guarded(fill)
        pool.offload(pl, 0, fmid[0], fmid[1], g.kvb, torch.from_numpy(good).to(dev))        # whole layer = 0x2222
        pool.offload(pl, 0, smid[0], smid[1], g.kvb, torch.from_numpy(bad).to(dev))
        pool.wait_offloads(pl)
        torch.cuda.synchronize()
        assert pool.table_errors() == len(bad_at)
        want2 = oracle.offload_layer(fill, good, opl[0])
        for j in np.flatnonzero(ok):
            oracle.offload_range(src_cpu, good, opl[0], want2, int(j), 1)
        got = [np.array(pl.stripe(0, i)) for i in range(3)]
        P = g.payload
        for j in range(K):                                                             # the pool slot of a rejected entry is unspecified on
            d, sl = int(opl[0].dev[j]), int(opl[0].slot[j])                             # the staged path (its staging bytes were never written)
            if ok[j] or path == "zerocopy":
                assert np.array_equal(got[d][sl * P:(sl + 1) * P], want2[d][sl * P:(sl + 1) * P]), j
        # check off again: trusted tables, counter stays at zero
        pool.set_table_check(0)
        pool.offload(pl, 0, smid[0], smid[1], g.kvb, torch.from_numpy(good).to(dev))
        pool.wait_offloads(pl)
        torch.cuda.synchronize()
        assert all(np.array_equal(pl.stripe(0, i), want[i]) for i in range(3)) and pool.table_errors() == 0
        pl.release()
    finally:
        pool.destroy()
